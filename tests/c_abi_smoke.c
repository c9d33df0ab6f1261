/* c_abi_smoke.c -- the C ABI of include/lgf.h driven from plain C (no Python, no torch, no CUDA headers):
 * lgf_create_simple, lgf_load / lgf_store with HOST buffers, lgf_measure, lgf_iterate, lgf_fix, error codes.
 * Expected values are closed forms (SURVEY.md §8(c) pins P3, P6): for an x-independent field U_mu(x) = V_mu
 * Delta = 0, so theta = 0 and F = (1/12) sum_mu Re Tr V_mu, and the field is a fixed point of the iteration.
 * On the same field the temporal Wilson line is V_t^Lt at every site, so the singlet correlator (eq. (1))
 * is 1 for every r.  lgf_create_batch needs a caller-allocated DEVICE workspace, which this CUDA-free program cannot
 * make: the batch entry points are exercised through lgf_batch_size and lgf_workspace_bytes_batch only (the batched
 * iteration itself: tests/test_gpu_parity.py).
 * Built and run by tests/test_c_abi.py; exit code 0 = all checks passed. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "lgf.h"

#define CHECK(cond)                                                                      \
    do {                                                                                 \
        if (!(cond)) {                                                                   \
            fprintf(stderr, "FAILED line %d: %s (%s)\n", __LINE__, #cond, lgf_last_error()); \
            return 1;                                                                    \
        }                                                                                \
    } while (0)

/* diag(e^{ia}, e^{ib}, e^{-i(a+b)}) at every site for direction mu, angles depending on mu only */
static void fill_constant(double* links, long long V, const double a[4], const double b[4]) {
    memset(links, 0, sizeof(double) * (size_t)V * 72);
    for (long long s = 0; s < V; ++s)
        for (int mu = 0; mu < 4; ++mu) {
            double* m = links + ((size_t)s * 4 + mu) * 18;
            const double ph[3] = {a[mu], b[mu], -(a[mu] + b[mu])};
            for (int i = 0; i < 3; ++i) {
                m[(3 * i + i) * 2] = cos(ph[i]);
                m[(3 * i + i) * 2 + 1] = sin(ph[i]);
            }
        }
}

static int run(int precision, int storage) {
    const int32_t L[4] = {8, 6, 4, 12};
    const long long V = 8LL * 6 * 4 * 12;
    const double a[4] = {0.3, -0.7, 1.1, 0.05}, b[4] = {-0.2, 0.4, 0.9, -1.3};
    double Fexp = 0.0;
    for (int mu = 0; mu < 4; ++mu) Fexp += cos(a[mu]) + cos(b[mu]) + cos(a[mu] + b[mu]);
    Fexp /= 12.0;
    const double tol = precision == LGF_F64 ? 1e-13 : 2e-6;

    lgf_ctx* ctx = NULL;
    lgf_result r;
    CHECK(lgf_workspace_bytes(L, precision, storage) > 0);
    CHECK(lgf_create_simple(L, precision, storage, &ctx) == LGF_OK && ctx);
    CHECK(lgf_measure(ctx, &r) == LGF_ESTATE);                 /* nothing loaded yet */

    double* h = (double*)malloc(sizeof(double) * (size_t)V * 72);
    CHECK(h);
    fill_constant(h, V, a, b);
    void* in = h;
    float* hf = NULL;
    if (precision == LGF_F32) {
        hf = (float*)malloc(sizeof(float) * (size_t)V * 72);
        CHECK(hf);
        for (size_t i = 0; i < (size_t)V * 72; ++i) hf[i] = (float)h[i];
        in = hf;
    }
    CHECK(lgf_load(ctx, in, LGF_HOST) == LGF_OK);
    CHECK(lgf_measure(ctx, &r) == LGF_OK);
    CHECK(r.iterations == 0 && fabs(r.F - Fexp) <= tol && r.theta <= tol * tol);

    /* already gauge fixed: lgf_fix applies no update */
    CHECK(lgf_fix(ctx, 0.08, 1e-10, 100, &r) == LGF_OK);
    CHECK(r.iterations == 0 && r.converged == 1 && fabs(r.F - Fexp) <= tol);

    /* a fixed point of the iteration: three updates leave F and every link where they were */
    CHECK(lgf_iterate(ctx, 3, 0.08, &r) == LGF_OK);
    CHECK(r.iterations == 3 && fabs(r.F - Fexp) <= tol && r.theta <= tol * tol);
    if (precision == LGF_F64) {
        double* o = (double*)malloc(sizeof(double) * (size_t)V * 72);
        CHECK(o && lgf_store(ctx, o, LGF_HOST) == LGF_OK);
        double md = 0.0;
        for (size_t i = 0; i < (size_t)V * 72; ++i) md = fmax(md, fabs(o[i] - h[i]));
        CHECK(md <= 1e-13);
        free(o);
    } else {
        float* o = (float*)malloc(sizeof(float) * (size_t)V * 72);
        CHECK(o && lgf_store(ctx, o, LGF_HOST) == LGF_OK);
        double md = 0.0;
        for (size_t i = 0; i < (size_t)V * 72; ++i) md = fmax(md, fabs((double)o[i] - (double)hf[i]));
        CHECK(md <= 2e-6);
        free(o);
    }
    /* the step after the path: W(x) = V_t^Lt = diag(e^{i Lt a_t}, e^{i Lt b_t}, e^{-i Lt (a_t+b_t)}), C(r) = 1 */
    {
        const long long Vs = V / L[3];
        const double wtol = precision == LGF_F64 ? 1e-12 : 2e-5;
        const double ph[3] = {L[3] * a[3], L[3] * b[3], -L[3] * (a[3] + b[3])};
        if (precision == LGF_F64) {
            double* w = (double*)malloc(sizeof(double) * (size_t)Vs * 18);
            double* cr = (double*)malloc(sizeof(double) * (size_t)Vs * 2);
            CHECK(w && cr && lgf_wilson_lines(ctx, w, LGF_HOST) == LGF_OK && lgf_singlet_correlator(ctx, cr, LGF_HOST) == LGF_OK);
            double md = 0.0;
            for (long long x = 0; x < Vs; ++x)
                for (int i = 0; i < 3; ++i)
                    for (int j = 0; j < 3; ++j) {
                        const double re = i == j ? cos(ph[i]) : 0.0, im = i == j ? sin(ph[i]) : 0.0;
                        md = fmax(md, fmax(fabs(w[(x * 9 + 3 * i + j) * 2] - re), fabs(w[(x * 9 + 3 * i + j) * 2 + 1] - im)));
                    }
            for (long long x = 0; x < Vs; ++x) md = fmax(md, fmax(fabs(cr[2 * x] - 1.0), fabs(cr[2 * x + 1])));
            CHECK(md <= wtol);
            free(w);
            free(cr);
        } else {
            float* cr = (float*)malloc(sizeof(float) * (size_t)Vs * 2);
            CHECK(cr && lgf_singlet_correlator(ctx, cr, LGF_HOST) == LGF_OK);
            double md = 0.0;
            for (long long x = 0; x < Vs; ++x) md = fmax(md, fmax(fabs((double)cr[2 * x] - 1.0), fabs((double)cr[2 * x + 1])));
            CHECK(md <= wtol);
            free(cr);
        }
        CHECK(lgf_iterate(ctx, 1, 0.08, &r) == LGF_OK && r.iterations == 1 && fabs(r.F - Fexp) <= tol);   /* scratch use is harmless */
        CHECK(lgf_batch_size(ctx) == 1);
        CHECK(lgf_workspace_bytes_batch(L, precision, storage, 3) > lgf_workspace_bytes(L, precision, storage));
        CHECK(lgf_workspace_bytes_batch(L, precision, storage, 0) == 0);
    }
    /* argument errors leave *out untouched */
    r.iterations = -7;
    CHECK(lgf_iterate(ctx, 1, -1.0, &r) == LGF_EINVAL && r.iterations == -7);
    CHECK(lgf_load(ctx, NULL, LGF_HOST) == LGF_EINVAL);
    CHECK(lgf_launch_count(ctx) > 0);
    CHECK(lgf_destroy(ctx) == LGF_OK);
    free(h);
    free(hf);
    return 0;
}

int main(void) {
    const int32_t bad[4] = {8, 8, 8, 10};                      /* 10 = 2 * 5 */
    lgf_ctx* c = NULL;
    if (lgf_create_simple(bad, LGF_F64, LGF_REAL18, &c) != LGF_EUNSUPPORTED) { fprintf(stderr, "expected LGF_EUNSUPPORTED\n"); return 1; }
    if (strcmp(lgf_strerror(LGF_OK), "ok") != 0) return 1;
    if (run(LGF_F64, LGF_REAL18) || run(LGF_F64, LGF_REAL12) || run(LGF_F32, LGF_REAL18) || run(LGF_F32, LGF_REAL12)) return 1;
    printf("c_abi_smoke: ok (lgf %s)\n", lgf_version());
    return 0;
}
