// lgf_oracle.cpp -- ORACLE (test infrastructure, NOT the product).
//
// A plain, slow, obviously-correct CPU implementation of Landau gauge fixing of a 4D SU(3)
// lattice gauge field by steepest descent with Fourier acceleration (arXiv 1208.1186;
// PAPER.md:11, 35 name the method; PAPER.md prints none of its formulas, so the binding
// definition is the five steps of BASELINE.json `north_star`, restated in SURVEY.md §8(c)).
// Everything is fp64, full 3x3 matrices, all 9 matrix elements of Delta are Fourier
// transformed separately ("The FFT is applied for all elements of Delta(x) matrix
// separately"), sites are lexicographic with x fastest ("lexicographic layout").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this library.  It shares no code, header, table or constant with the CUDA path in
// paper_1208_1186_b200/csrc/.
//
// Pins (tests/test_oracle_*.py): FFT vs O(N^2) DFT and numpy.fft; p^2
// table closed forms; Delta anti-Hermitian/traceless/sum-zero; unitarity; plaquette and
// Polyakov-loop invariance; F monotone, F -> 1 on a pure-gauge field; the closed form
// theta1/theta0 = (1 - alpha p2max)^2 for an infinitesimal gauge copy of the unit field;
// E[theta] = 128/9 on Haar links; position-space convolution brute force.
// "parity unpinned": the final links of a rough configuration have no external truth; they
// are validated only through the pins above.
// The step after the path (eq. (1)): temporal Wilson lines and the singlet
// correlator of ONE configuration, written out as the definition (ordered product along t; direct double sum over
// the spatial lattice).  Pins (tests/test_oracle_correlator.py): W = 1 and C = 1 on the unit field; C(0) = 1;
// C(-r) = conj C(r); sum_r C(r) = |sum_x W(x)|_F^2 / (3 Vs); Tr W against a torch restatement of the Polyakov loop;
// covariance W -> g(x,0) W g(x,0)^+ under a gauge transform, invariance of C under x-independent transforms.
//
// Loops carry `#pragma omp parallel for` over sites / FFT lines only; every reduction is a
// serial compensated sum over a per-site array, so results are bit-identical for any thread
// count.
//
// Layouts (all double, complex interleaved re,im):
//   links  U[s][mu][row][col]   72 doubles per site
//   Delta  D[s][row][col]       18 doubles per site
//   g      g[s][row][col]       18 doubles per site
//   scalar complex field f[s]   2 doubles per site
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
typedef long double ldbl;

namespace {

struct Lat {
    int L[4];
    int64_t V;
    explicit Lat(const int32_t* l) {
        V = 1;
        for (int i = 0; i < 4; ++i) { L[i] = l[i]; V *= l[i]; }
    }
    void coords(int64_t s, int x[4]) const {
        for (int i = 0; i < 4; ++i) { x[i] = int(s % L[i]); s /= L[i]; }
    }
    int64_t index(const int x[4]) const {
        return x[0] + (int64_t)L[0] * (x[1] + (int64_t)L[1] * (x[2] + (int64_t)L[2] * x[3]));
    }
    // site x + dir * mu_hat with periodic wrap, dir = +1 or -1
    int64_t neighbour(int64_t s, int mu, int dir) const {
        int x[4];
        coords(s, x);
        x[mu] = (x[mu] + dir + L[mu]) % L[mu];
        return index(x);
    }
};

struct Mat3 {
    cplx a[3][3];
};

Mat3 load(const double* p) {
    Mat3 m;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) m.a[i][j] = cplx(p[2 * (3 * i + j)], p[2 * (3 * i + j) + 1]);
    return m;
}
void store(double* p, const Mat3& m) {
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            p[2 * (3 * i + j)] = m.a[i][j].real();
            p[2 * (3 * i + j) + 1] = m.a[i][j].imag();
        }
}
Mat3 mul(const Mat3& x, const Mat3& y) {
    Mat3 r;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            cplx acc = 0;
            for (int k = 0; k < 3; ++k) acc += x.a[i][k] * y.a[k][j];
            r.a[i][j] = acc;
        }
    return r;
}
Mat3 dagger(const Mat3& x) {
    Mat3 r;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) r.a[i][j] = std::conj(x.a[j][i]);
    return r;
}

// Neumaier compensated sum, serial, index order: the value is independent of how the per-site
// terms were produced (SURVEY.md §8(c) "theta and F are summed with compensated summation").
double compensated_sum(const std::vector<double>& v) {
    double sum = 0.0, c = 0.0;
    for (double x : v) {
        double t = sum + x;
        if (std::fabs(sum) >= std::fabs(x)) c += (sum - t) + x;
        else c += (x - t) + sum;
        sum = t;
    }
    return sum + c;
}

// exp(sign * 2 pi i k / n), argument reduced exactly in integers, evaluated in long double.
cplx root_of_unity(int64_t k, int64_t n, int sign) {
    k %= n;
    if (k < 0) k += n;
    const ldbl two_pi = 6.283185307179586476925286766559005768L;
    ldbl ang = two_pi * (ldbl)k / (ldbl)n;
    return cplx((double)cosl(ang), (double)(sign * sinl(ang)));
}

// Direct O(n^2) DFT of one line: out[k] = sum_x in[x] exp(sign 2 pi i k x / n).  No scaling.
void dft_direct(int n, const cplx* in, cplx* out, int sign) {
    for (int k = 0; k < n; ++k) {
        cplx acc = 0;
        for (int x = 0; x < n; ++x) acc += in[x] * root_of_unity((int64_t)k * x, n, sign);
        out[k] = acc;
    }
}

// Table w[j] = exp(sign 2 pi i j / n), j = 0..n-1, each entry from the long double routine.
std::vector<cplx> root_table(int n, int sign) {
    std::vector<cplx> w(n);
    for (int j = 0; j < n; ++j) w[j] = root_of_unity(j, n, sign);
    return w;
}

// Recursive mixed-radix decimation-in-time FFT (radix = smallest prime factor; a prime length
// falls back to the direct DFT).  out[k], k = 0..n-1, from in[0], in[stride], ...  No scaling.
// w is the root table of the TOP-level length ntop (n divides ntop): exp(sign 2 pi i j/n) =
// w[j * (ntop/n)].
void fft_rec(int n, const cplx* in, int stride, cplx* out, const cplx* w, int ntop) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = 0;
    for (int q = 2; q * q <= n; ++q)
        if (n % q == 0) { p = q; break; }
    const int step = ntop / n;
    if (p == 0) {  // n prime: direct sum
        for (int k = 0; k < n; ++k) {
            cplx acc = 0;
            for (int x = 0; x < n; ++x) acc += in[(int64_t)x * stride] * w[(int64_t)(((int64_t)k * x) % n) * step];
            out[k] = acc;
        }
        return;
    }
    const int m = n / p;
    // sub[r][k1] = DFT_m of the subsequence x = p*x1 + r
    std::vector<cplx> sub((size_t)n);
    for (int r = 0; r < p; ++r) fft_rec(m, in + (int64_t)r * stride, stride * p, sub.data() + (size_t)r * m, w, ntop);
    // out[k] = sum_r w_n^{r k} sub[r][k mod m]
    for (int k = 0; k < n; ++k) {
        cplx acc = 0;
        for (int r = 0; r < p; ++r) acc += w[(int64_t)(((int64_t)r * k) % n) * step] * sub[(size_t)r * m + (k % m)];
        out[k] = acc;
    }
}

// Apply a 1D transform along every axis of a complex scalar field f[s].
// sign = -1: forward, unnormalised.  sign = +1: inverse, multiplied by 1/V at the end
// (SURVEY.md §8(c) reading #5).  direct != 0 uses the O(n^2) DFT per line.
void transform4d(const Lat& lat, cplx* f, int sign, int direct) {
    int64_t stride = 1;
    for (int mu = 0; mu < 4; ++mu) {
        const int n = lat.L[mu];
        const int64_t nlines = lat.V / n;
        const std::vector<cplx> w = root_table(n, sign);
#pragma omp parallel
        {
            std::vector<cplx> line(n), res(n);
#pragma omp for schedule(static)
            for (int64_t l = 0; l < nlines; ++l) {
                // line l: inner index (below axis mu) and outer index (above it)
                const int64_t inner = l % stride, outer = l / stride;
                cplx* base = f + inner + outer * stride * n;
                for (int x = 0; x < n; ++x) line[x] = base[(int64_t)x * stride];
                if (direct) dft_direct(n, line.data(), res.data(), sign);
                else fft_rec(n, line.data(), 1, res.data(), w.data(), n);
                for (int x = 0; x < n; ++x) base[(int64_t)x * stride] = res[x];
            }
        }
        stride *= n;
    }
    if (sign > 0) {
        const double inv = 1.0 / (double)lat.V;
        for (int64_t s = 0; s < lat.V; ++s) f[s] *= inv;
    }
}

// p^2(k) = sum_mu 4 sin^2(pi k_mu / L_mu)   (north_star step 3)
double psq_of(const Lat& lat, const int k[4]) {
    const ldbl pi = 3.141592653589793238462643383279502884L;
    ldbl acc = 0;
    for (int mu = 0; mu < 4; ++mu) {
        ldbl s = sinl(pi * (ldbl)k[mu] / (ldbl)lat.L[mu]);
        acc += 4 * s * s;
    }
    return (double)acc;
}
// p^2_max = max over the lattice's own momenta (SURVEY.md §8(c) reading #7).
double psq_max_of(const Lat& lat) {
    int k[4];
    for (int mu = 0; mu < 4; ++mu) k[mu] = lat.L[mu] / 2;
    return psq_of(lat, k);
}

// Row Gram-Schmidt: rows 0, 1 orthonormalised in order, row 2 = conj(row0 x row1)
// (SURVEY.md §8(c) reading #9; "first two rows ... reconstruct the third row").
Mat3 reunitarise(const Mat3& m) {
    Mat3 r;
    double n0 = 0;
    for (int j = 0; j < 3; ++j) n0 += std::norm(m.a[0][j]);
    n0 = std::sqrt(n0);
    for (int j = 0; j < 3; ++j) r.a[0][j] = m.a[0][j] / n0;
    cplx dot = 0;  // r0^* . m1
    for (int j = 0; j < 3; ++j) dot += std::conj(r.a[0][j]) * m.a[1][j];
    double n1 = 0;
    for (int j = 0; j < 3; ++j) {
        r.a[1][j] = m.a[1][j] - dot * r.a[0][j];
        n1 += std::norm(r.a[1][j]);
    }
    n1 = std::sqrt(n1);
    for (int j = 0; j < 3; ++j) r.a[1][j] /= n1;
    r.a[2][0] = std::conj(r.a[0][1] * r.a[1][2] - r.a[0][2] * r.a[1][1]);
    r.a[2][1] = std::conj(r.a[0][2] * r.a[1][0] - r.a[0][0] * r.a[1][2]);
    r.a[2][2] = std::conj(r.a[0][0] * r.a[1][1] - r.a[0][1] * r.a[1][0]);
    return r;
}

// Step 1 (north_star): Delta(x) = sum_mu [U_mu(x - mu) - U_mu(x) - h.c.]_traceless,
// theta = (1/(3V)) sum_x Tr Delta Delta^+,  F = (1/(12V)) sum_x sum_mu Re Tr U_mu(x).
void measure(const Lat& lat, const double* U, double* Delta, double* theta, double* F) {
    std::vector<double> th((size_t)lat.V), fn((size_t)lat.V);
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < lat.V; ++s) {
        Mat3 M;
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) M.a[i][j] = 0;
        double retr = 0;
        for (int mu = 0; mu < 4; ++mu) {
            const Mat3 here = load(U + (s * 4 + mu) * 18);
            const Mat3 back = load(U + (lat.neighbour(s, mu, -1) * 4 + mu) * 18);
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) M.a[i][j] += back.a[i][j] - here.a[i][j];
            retr += here.a[0][0].real() + here.a[1][1].real() + here.a[2][2].real();
        }
        const Mat3 Md = dagger(M);
        Mat3 A;
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) A.a[i][j] = M.a[i][j] - Md.a[i][j];
        const cplx tr3 = (A.a[0][0] + A.a[1][1] + A.a[2][2]) / 3.0;
        for (int i = 0; i < 3; ++i) A.a[i][i] -= tr3;
        double t = 0;
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) t += std::norm(A.a[i][j]);
        th[s] = t;
        fn[s] = retr;
        if (Delta) store(Delta + s * 18, A);
    }
    *theta = compensated_sum(th) / (3.0 * (double)lat.V);
    *F = compensated_sum(fn) / (12.0 * (double)lat.V);
}

// Steps 2-3 (north_star): every one of the 9 matrix elements e of Delta separately:
//   Dhat_e(k) = sum_x Delta_e(x) exp(-2 pi i k.x/L);  Dhat_e(k) *= p2max / p2(k), Dhat_e(0) = 0;
//   Dtilde_e(x) = (1/V) sum_k Dhat_e(k) exp(+2 pi i k.x/L).
void fourier_accelerate(const Lat& lat, const double* Delta, double* Dtilde, int direct) {
    std::vector<cplx> f((size_t)lat.V);
    const double pmax = psq_max_of(lat);
    for (int e = 0; e < 9; ++e) {
        for (int64_t s = 0; s < lat.V; ++s) f[s] = cplx(Delta[s * 18 + 2 * e], Delta[s * 18 + 2 * e + 1]);
        transform4d(lat, f.data(), -1, direct);
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < lat.V; ++s) {
            int k[4];
            lat.coords(s, k);
            if (s == 0) f[s] = 0;
            else f[s] *= pmax / psq_of(lat, k);
        }
        transform4d(lat, f.data(), +1, direct);
        for (int64_t s = 0; s < lat.V; ++s) {
            Dtilde[s * 18 + 2 * e] = f[s].real();
            Dtilde[s * 18 + 2 * e + 1] = f[s].imag();
        }
    }
}

// Step 4 (north_star): g(x) = reunitarise(1 + (alpha/2) Dtilde(x)).
void build_g(const Lat& lat, const double* Dtilde, double alpha, double* g) {
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < lat.V; ++s) {
        Mat3 m = load(Dtilde + s * 18);
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) m.a[i][j] = (alpha / 2.0) * m.a[i][j] + (i == j ? 1.0 : 0.0);
        store(g + s * 18, reunitarise(m));
    }
}

// Step 5 (north_star): U'_mu(x) = g(x) U_mu(x) g(x + mu)^+, all from the old field (Jacobi).
void update_links(const Lat& lat, const double* U, const double* g, double* Unew) {
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < lat.V; ++s) {
        const Mat3 gx = load(g + s * 18);
        for (int mu = 0; mu < 4; ++mu) {
            const Mat3 gf = load(g + lat.neighbour(s, mu, +1) * 18);
            store(Unew + (s * 4 + mu) * 18, mul(mul(gx, load(U + (s * 4 + mu) * 18)), dagger(gf)));
        }
    }
}

// Temporal Wilson line ("W(.) is the temporal Wilson line"): W(x) = U_t(x,0) U_t(x,1) ... U_t(x,Lt-1),
// the ordered product of the t-links at spatial site x = (x,y,z); xs = x + Lx (y + Ly z).
void wilson_lines(const Lat& lat, const double* U, double* W) {
    const int64_t Vs = lat.V / lat.L[3];
#pragma omp parallel for schedule(static)
    for (int64_t xs = 0; xs < Vs; ++xs) {
        Mat3 w = load(U + ((xs + 0 * Vs) * 4 + 3) * 18);
        for (int t = 1; t < lat.L[3]; ++t) w = mul(w, load(U + ((xs + (int64_t)t * Vs) * 4 + 3) * 18));
        store(W + xs * 18, w);
    }
}

// Singlet correlator of one configuration, eq. (1) of PAPER.md:33 with the ensemble average replaced by the average
// over the spatial lattice:  C(r) = (1/(3 Vs)) sum_x Tr[ W(x + r) W(x)^+ ],  r on the periodic spatial lattice.
// Direct O(Vs^2) double sum, compensated per r.
void singlet_correlator(const Lat& lat, const double* U, double* C) {
    const int64_t Vs = lat.V / lat.L[3];
    std::vector<double> W((size_t)Vs * 18);
    wilson_lines(lat, U, W.data());
    const int Lx = lat.L[0], Ly = lat.L[1], Lz = lat.L[2];
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < Vs; ++r) {
        const int rx = int(r % Lx), ry = int((r / Lx) % Ly), rz = int(r / ((int64_t)Lx * Ly));
        std::vector<double> re((size_t)Vs), im((size_t)Vs);
        for (int64_t xs = 0; xs < Vs; ++xs) {
            const int x = int(xs % Lx), y = int((xs / Lx) % Ly), z = int(xs / ((int64_t)Lx * Ly));
            const int64_t xr = (x + rx) % Lx + (int64_t)Lx * ((y + ry) % Ly + (int64_t)Ly * ((z + rz) % Lz));
            const Mat3 a = load(W.data() + xr * 18), b = load(W.data() + xs * 18);
            cplx tr = 0;                       // Tr[a b^+] = sum_ij a_ij conj(b_ij)
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) tr += a.a[i][j] * std::conj(b.a[i][j]);
            re[xs] = tr.real();
            im[xs] = tr.imag();
        }
        C[2 * r] = compensated_sum(re) / (3.0 * (double)Vs);
        C[2 * r + 1] = compensated_sum(im) / (3.0 * (double)Vs);
    }
}

}  // namespace

extern "C" {

int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

void orc_dft1d(int n, const double* in, double* out, int sign) {
    dft_direct(n, reinterpret_cast<const cplx*>(in), reinterpret_cast<cplx*>(out), sign);
}
void orc_fft1d(int n, const double* in, double* out, int sign) {
    const std::vector<cplx> w = root_table(n, sign);
    fft_rec(n, reinterpret_cast<const cplx*>(in), 1, reinterpret_cast<cplx*>(out), w.data(), n);
}
// In-place 4D transform of a complex scalar field; sign=-1 forward (no scaling), +1 inverse (1/V).
void orc_transform4d(const int32_t* L, double* f, int sign, int direct) {
    transform4d(Lat(L), reinterpret_cast<cplx*>(f), sign, direct);
}
void orc_psq(const int32_t* L, double* p2, double* p2max) {
    Lat lat(L);
    for (int64_t s = 0; s < lat.V; ++s) {
        int k[4];
        lat.coords(s, k);
        p2[s] = psq_of(lat, k);
    }
    *p2max = psq_max_of(lat);
}
void orc_measure(const int32_t* L, const double* U, double* Delta, double* theta, double* F) {
    measure(Lat(L), U, Delta, theta, F);
}
void orc_fourier_accelerate(const int32_t* L, const double* Delta, double* Dtilde, int direct) {
    fourier_accelerate(Lat(L), Delta, Dtilde, direct);
}
void orc_build_g(const int32_t* L, const double* Dtilde, double alpha, double* g) {
    build_g(Lat(L), Dtilde, alpha, g);
}
void orc_reunitarise(const double* m, double* out) { store(out, reunitarise(load(m))); }
void orc_update_links(const int32_t* L, const double* U, const double* g, double* Unew) {
    update_links(Lat(L), U, g, Unew);
}
// 12-real storage: keep rows 0,1 of every link, rebuild row 2 = conj(row0 x row1).
void orc_two_row_roundtrip(int64_t nlinks, const double* U, double* out) {
    for (int64_t l = 0; l < nlinks; ++l) {
        Mat3 m = load(U + l * 18);
        m.a[2][0] = std::conj(m.a[0][1] * m.a[1][2] - m.a[0][2] * m.a[1][1]);
        m.a[2][1] = std::conj(m.a[0][2] * m.a[1][0] - m.a[0][0] * m.a[1][2]);
        m.a[2][2] = std::conj(m.a[0][0] * m.a[1][1] - m.a[0][1] * m.a[1][0]);
        store(out + l * 18, m);
    }
}

// n updates in place (steps 2-5 then step 1 each).  theta_hist/F_hist (nullable) get n+1
// entries: the measurement before the first update and after each update.
void orc_iterate(const int32_t* L, double* U, int64_t n, double alpha, double* theta_hist, double* F_hist) {
    Lat lat(L);
    std::vector<double> D((size_t)lat.V * 18), Dt((size_t)lat.V * 18), g((size_t)lat.V * 18), Un((size_t)lat.V * 72);
    double theta, F;
    measure(lat, U, D.data(), &theta, &F);
    if (theta_hist) theta_hist[0] = theta;
    if (F_hist) F_hist[0] = F;
    for (int64_t it = 1; it <= n; ++it) {
        fourier_accelerate(lat, D.data(), Dt.data(), 0);
        build_g(lat, Dt.data(), alpha, g.data());
        update_links(lat, U, g.data(), Un.data());
        std::memcpy(U, Un.data(), sizeof(double) * (size_t)lat.V * 72);
        measure(lat, U, D.data(), &theta, &F);
        if (theta_hist) theta_hist[it] = theta;
        if (F_hist) F_hist[it] = F;
    }
}

// fix(U, alpha, tol, max_iter): measure; while theta >= tol and n < max_iter: update, measure.
// Returns the number of updates applied (SURVEY.md §8(c) readings #11, #12).  hist arrays
// (nullable) must hold max_iter+1 entries.
int64_t orc_fix(const int32_t* L, double* U, double alpha, double theta_tol, int64_t max_iter,
                double* theta_out, double* F_out, double* theta_hist, double* F_hist) {
    Lat lat(L);
    std::vector<double> D((size_t)lat.V * 18), Dt((size_t)lat.V * 18), g((size_t)lat.V * 18), Un((size_t)lat.V * 72);
    double theta, F;
    measure(lat, U, D.data(), &theta, &F);
    int64_t n = 0;
    if (theta_hist) theta_hist[0] = theta;
    if (F_hist) F_hist[0] = F;
    while (theta >= theta_tol && n < max_iter) {
        fourier_accelerate(lat, D.data(), Dt.data(), 0);
        build_g(lat, Dt.data(), alpha, g.data());
        update_links(lat, U, g.data(), Un.data());
        std::memcpy(U, Un.data(), sizeof(double) * (size_t)lat.V * 72);
        measure(lat, U, D.data(), &theta, &F);
        ++n;
        if (theta_hist) theta_hist[n] = theta;
        if (F_hist) F_hist[n] = F;
    }
    *theta_out = theta;
    *F_out = F;
    return n;
}


void orc_wilson_lines(const int32_t* L, const double* U, double* W) { wilson_lines(Lat(L), U, W); }
void orc_singlet_correlator(const int32_t* L, const double* U, double* C) { singlet_correlator(Lat(L), U, C); }

}  // extern "C"
