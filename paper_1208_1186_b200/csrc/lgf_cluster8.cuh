// lgf_cluster8.cuh -- the WHOLE iteration loop of an 8^4 lattice in ONE kernel on ONE 16-CTA thread-block cluster
// (a batched context launches one cluster per lattice)
// (SURVEY.md §8(f) rank 1 "persistent single-kernel iteration for 8^4"; north_star steps 1-5 and the convergence loop).
//
// One lattice of 8^4 is launch-latency-bound on the five-kernel graph (22 us per iteration for 6.8 MB of traffic).
// Here the links never leave the chip: CTA r of the cluster owns the 256 sites of time slice t = r/2, z-half zh = r%2
// (x, y in 0..7, z = 4 zh + zl), one thread per site, and keeps their four links in its shared memory for the whole call
// (fp64 18-real: 147 KB).  Steps of one iteration, separated by four cluster barriers (barrier.cluster, ~0.25 us each):
//   A  forward DFT along x, y of the packed Delta (4 complex per site) in the CTA's own shared memory
//      -- barrier 1 --   (also publishes the per-CTA theta / F partials of the previous step: every warp of every CTA
//      sums the 16 partials with the same butterfly, so all CTAs take the same stopping decision)
//   B  every CTA PULLS its 16 (z,t) planes -- the 8 kx of row ky = r/2 for two of the four components -- from the 16
//      CTAs through distributed shared memory (128-byte rows), C transforms them along z, t, scales by
//      p2max/(V p2(k)) (the 8 quotients of a thread are loop-invariant: registers) and transforms back
//      -- barrier 2 --
//   D  every CTA pulls the Delta~ spectrum of its own sites back, inverse DFT along y, x
//   E  g = reunitarise(1 + (alpha/2) Delta~) per site; rows 0, 1 of g go to shared memory for the neighbours
//      -- barrier 3 (arrive here, wait after the x and y directions of F: their g are in this CTA) --
//   F  U'_mu = g U_mu g(x+mu)^+ (g of the z / t neighbours read from the neighbouring CTA), and -- since
//      Delta is linear in the links -- the projected link P(U'_mu(x)) (the packed anti-Hermitian traceless part,
//      8 reals) is PUSHED to site x+mu: by warp shuffle along x, into shared-memory inboxes along y, z, t (remote
//      stores for the z / t faces).  Nobody ever reads another site's links.
//      -- barrier 4 --
//   G  Delta(x) = sum_mu [P(U_mu(x-mu)) - P(U_mu(x))] from the inboxes, theta and F partials per CTA.
// Links are read from and written back to the context's global buffers at the start and the end of the call, Delta
// too, so every other entry point (lgf_store, lgf_measure, the per-kernel hooks) sees the same state as after the
// five-kernel path.  Rounding differs from K1 in one place: the trace is removed per link before the sum over mu.
// -DLGF_CL8_PROF (developer builds only) prints per-step cycle counts of the last iteration.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cooperative_groups.h>

#include "lgf_async.cuh"
#include "lgf_regfft.cuh"
#include "lgf_site.cuh"

namespace lgf {

namespace cg = cooperative_groups;

#ifdef LGF_CL8_PROF
#define CL8_STAMP(i) do { if (tid == 0) prof[i] = clock64(); } while (0)
#else
#define CL8_STAMP(i) do {} while (0)
#endif

struct Cluster8Args {
    const void* psq;        // p^2 table of one axis of 8 points (all four axes are equal), element type T
    double scale_num;       // p2max / V
    double half_alpha;
};

template <typename T, int NC>
struct Cl8 {
    static constexpr int kCtas = 16, kThreads = 256, kSites = 256;
    static constexpr int kPad = 288;                       // 256 sites at row pitch 9: index l + (l >> 3)
    static constexpr int kLinks = 4 * NC * kSites;         // [mu][c][l]
    static constexpr int kG = 6 * kSites;                  // rows 0, 1 of g: [k][l]
    static constexpr int kField = 4 * kPad;                // a packed field in the padded site order (>= the 1024 plane elements)
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)(kLinks + kG + 3 * kField) + 64;
    static_assert(kSmem <= 227 * 1024, "cluster path: shared memory");
};

__device__ __forceinline__ int cl8_pad(int l) { return l + (l >> 3); }

// distributed shared memory: the shared::cluster address of `p` (an address in THIS CTA's window) in CTA `rank`
__device__ __forceinline__ uint32_t cl8_map(const void* p, unsigned rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
__device__ __forceinline__ Cx<double> cl8_ld(uint32_t a, double) {
    double x, y;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(x), "=d"(y) : "r"(a) : "memory");
    return Cx<double>(x, y);
}
__device__ __forceinline__ Cx<float> cl8_ld(uint32_t a, float) {
    float x, y;
    asm volatile("ld.shared::cluster.v2.f32 {%0, %1}, [%2];" : "=f"(x), "=f"(y) : "r"(a) : "memory");
    return Cx<float>(x, y);
}
__device__ __forceinline__ void cl8_st(uint32_t a, Cx<double> v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(a), "d"(v.re), "d"(v.im) : "memory");
}
__device__ __forceinline__ void cl8_st(uint32_t a, Cx<float> v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.re), "f"(v.im) : "memory");
}
__device__ __forceinline__ double cl8_ld_f64(uint32_t a) {
    double x;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(x) : "r"(a) : "memory");
    return x;
}

// 8-point DFT of the line f[0], f[stride], ..., f[7 stride] in place
template <int SIGN, typename T>
__device__ __forceinline__ void cl8_line(Cx<T>* f, int stride) {
    Cx<T> v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = f[j * stride];
    RegFft<8, SIGN, T>::run(v);
#pragma unroll
    for (int j = 0; j < 8; ++j) f[j * stride] = v[j];
}

template <typename T> __device__ __forceinline__ T cl8_shfl(T v, int src) { return __shfl_sync(0xffffffffu, v, src); }

// Cluster barriers.  cg::cluster_group::sync() costs two block barriers around the fence + hardware barrier;
// barrier.cluster counts every thread of every CTA, so the block barriers are redundant and the kernel issues the
// PTX itself.  Every arrive keeps its RELEASE semantics (MEMBAR.ALL.GPU in SASS): a relaxed arrive behind a CTA-scope
// fence, for the barriers that only publish a CTA's own shared memory, was 0.45 us per iteration faster and WRONG --
// 18 of 3300 batched fp32 runs (two CTAs per SM, several clusters in flight) read stale data.
__device__ __forceinline__ void cl8_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl8_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cl8_sync() { cl8_arrive(); cl8_wait(); }

// barrier over the first four warps of the CTA (the 128 threads that run the DFT passes)
__device__ __forceinline__ void cl8_bar128() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

template <typename T, int NC>
__global__ void __launch_bounds__(256, 1)
k_cluster8_iterate(Cx<T>* __restrict__ U, Cx<T>* __restrict__ Dg, DevState* st, const Cluster8Args A) {
    typedef Cl8<T, NC> C;
    extern __shared__ __align__(128) unsigned char cl8_smem[];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), tid = threadIdx.x, lane = tid & 31;
    constexpr long long V = 4096;
    constexpr int NR = NC / 3;
    constexpr uint32_t ES = sizeof(Cx<T>);
    {   // batched contexts: one cluster per lattice (the hardware runs as many clusters side by side as it has room for)
        const int lat = (int)blockIdx.x / C::kCtas;
        U += (size_t)lat * 4 * NC * V;
        Dg += (size_t)lat * 4 * V;
        st += lat;
    }

    Cx<T>* links = reinterpret_cast<Cx<T>*>(cl8_smem);
    Cx<T>* G = links + C::kLinks;
    Cx<T>* D = G + C::kG;                      // Delta / Delta~ of the CTA's sites (padded site order); inbox of the y pushes
    Cx<T>* Tb = D + C::kField;                 // the CTA's 16 (z,t) planes [cc][t][z][kx]; inbox of the z pushes
    Cx<T>* X = Tb + C::kField;                 // inbox of the t pushes
    double* part = reinterpret_cast<double*>(X + C::kField);     // this CTA's (theta, F) partial sums
    __shared__ double red_a[8], red_b[8];

    const int l = tid, lp = cl8_pad(l);
    const int x = l & 7, y = (l >> 3) & 7, zl = l >> 6, zh = rank & 1, t = rank >> 1;
    const long long s = (long long)rank * 256 + l;               // global site index x + 8 (y + 8 (z + 8 t))

#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
        for (int c = 0; c < NC; ++c) links[(mu * NC + c) * 256 + l] = ld_cx(U + (size_t)(mu * NC + c) * V + s);

    // forward neighbours: (rank, local site) of x + mu
    const int lf_x = (l & ~7) | ((l + 1) & 7);
    const int lf_y = (l & ~0x38) | ((l + 8) & 0x38);
    const bool z_remote = zl == 3;
    const int lf_z = z_remote ? (l & 63) : l + 64;
    const unsigned rank_z = z_remote ? (unsigned)(rank ^ 1) : (unsigned)rank;
    const unsigned rank_t = (unsigned)((rank + 2) & 15);
    const int src_x = (lane & ~7) | ((lane - 1) & 7);             // the lane that owns x - 1
    const uint32_t G_z = cl8_map(G + lf_z, rank_z), G_t = cl8_map(G + l, rank_t);
    const uint32_t box_z = cl8_map(Tb + cl8_pad(lf_z), rank_z), box_t = cl8_map(X + lp, rank_t);

    // step C's quotients p2max / (V p2(k)) of this thread's t line (kx, ky = rank/2, kz): loop-invariant
    T sc[8];
    {
        const T* psq = reinterpret_cast<const T*>(A.psq);
        const int kx = tid & 7, kz = (tid >> 3) & 7, ky = rank >> 1;
        const T pxyz = psq[kx] + psq[ky] + psq[kz], num = (T)A.scale_num;
#pragma unroll
        for (int kt = 0; kt < 8; ++kt) sc[kt] = ((kx | ky | kz | kt) == 0) ? T(0) : num / (pxyz + psq[kt]);
    }

    const T ha = (T)A.half_alpha;
    double theta = 0.0, Fval = 0.0;
    long long iter = st->iter;
    const long long max_iter = st->max_iter;
    const double tol = st->tol;
    Cx<T> dreg[4];                                                // Delta of the own site (written back at the end)
#ifdef LGF_CL8_PROF
    long long prof[16] = {};
#endif

    // Steps F + G.  update = false: the links are measured as they are (the call's first pass).
    // g0: g of the own site (step E left it in registers)
    auto update_and_measure = [&](bool update, const Su3<T>& g0) {
        Cx<T> c0(0, 0), c1(0, 0), c2(0, 0);
        T e0 = 0, e1 = 0, retr = 0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            Su3<T> u;
#pragma unroll
            for (int c = 0; c < NC; ++c) u.m[c] = links[(mu * NC + c) * 256 + l];
            if constexpr (NC == 6) rebuild_row2(u);
            if (update) {
                Su3<T> gf;
                if (mu < 2) {
                    const Cx<T>* gsrc = mu == 0 ? G + lf_x : G + lf_y;
#pragma unroll
                    for (int k = 0; k < 6; ++k) gf.m[k] = gsrc[k * 256];
                } else {
                    if (mu == 2) cl8_wait();                        // barrier 3 (arrived after step E): the neighbours' g are in place
                    const uint32_t gsrc = mu == 2 ? G_z : G_t;
#pragma unroll
                    for (int k = 0; k < 6; ++k) gf.m[k] = cl8_ld(gsrc + (uint32_t)k * 256u * ES, T());
                }
                rebuild_row2(gf);
                Cx<T> W[3 * NR];
#pragma unroll
                for (int i = 0; i < NR; ++i)
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        Cx<T> acc = g0.m[3 * i] * u.m[j];
                        fma_cx(acc, g0.m[3 * i + 1], u.m[3 + j]);
                        fma_cx(acc, g0.m[3 * i + 2], u.m[6 + j]);
                        W[3 * i + j] = acc;
                    }
#pragma unroll
                for (int i = 0; i < NR; ++i)
#pragma unroll
                    for (int j = 0; j < 3; ++j) {
                        Cx<T> acc = mulc(W[3 * i], gf.m[3 * j]);
                        fma_cxc(acc, W[3 * i + 1], gf.m[3 * j + 1]);
                        fma_cxc(acc, W[3 * i + 2], gf.m[3 * j + 2]);
                        u.m[3 * i + j] = acc;
                    }
                if constexpr (NC == 6) rebuild_row2(u);            // as K1 sees a 12-real link: row 2 from the stored rows
#pragma unroll
                for (int c = 0; c < NC; ++c) links[(mu * NC + c) * 256 + l] = u.m[c];
            }
            // P(U): packed anti-Hermitian traceless part of this link
            const Cx<T> q0 = u.m[1] - conj(u.m[3]), q1 = u.m[2] - conj(u.m[6]), q2 = u.m[5] - conj(u.m[7]);
            const T tr3 = (u.m[0].im + u.m[4].im + u.m[8].im) / T(3);
            const Cx<T> q3(u.m[0].im - tr3, u.m[4].im - tr3);
            retr += u.m[0].re + u.m[4].re + u.m[8].re;
            c0 = c0 - q0; c1 = c1 - q1; c2 = c2 - q2;
            e0 -= q3.re; e1 -= q3.im;
            if (mu == 0) {                                          // x: the receiver is a lane of this warp
                c0 = c0 + Cx<T>(cl8_shfl(q0.re, src_x), cl8_shfl(q0.im, src_x));
                c1 = c1 + Cx<T>(cl8_shfl(q1.re, src_x), cl8_shfl(q1.im, src_x));
                c2 = c2 + Cx<T>(cl8_shfl(q2.re, src_x), cl8_shfl(q2.im, src_x));
                e0 += cl8_shfl(q3.re, src_x);
                e1 += cl8_shfl(q3.im, src_x);
            } else if (mu == 1) {
                Cx<T>* box = D + cl8_pad(lf_y);
                box[0] = q0; box[C::kPad] = q1; box[2 * C::kPad] = q2; box[3 * C::kPad] = q3;
            } else {
                const uint32_t box = mu == 2 ? box_z : box_t;
                cl8_st(box, q0); cl8_st(box + C::kPad * ES, q1); cl8_st(box + 2 * C::kPad * ES, q2); cl8_st(box + 3 * C::kPad * ES, q3);
            }
        }
        CL8_STAMP(11);
        cl8_sync();                                         // barrier 4: every push has landed
        CL8_STAMP(12);
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const Cx<T>* box = (b == 0 ? D : (b == 1 ? Tb : X)) + lp;
            const Cx<T> p0 = box[0], p1 = box[C::kPad], p2 = box[2 * C::kPad], p3 = box[3 * C::kPad];
            c0 = c0 + p0; c1 = c1 + p1; c2 = c2 + p2;
            e0 += p3.re; e1 += p3.im;
        }
        const T d0 = T(2) * e0, d1 = T(2) * e1, d2 = -(d0 + d1);
        dreg[0] = c0; dreg[1] = c1; dreg[2] = c2; dreg[3] = Cx<T>(d0, d1);
        D[lp] = c0; D[C::kPad + lp] = c1; D[2 * C::kPad + lp] = c2; D[3 * C::kPad + lp] = dreg[3];
        double th = 2.0 * ((double)norm2(c0) + (double)norm2(c1) + (double)norm2(c2)) + (double)d0 * d0 + (double)d1 * d1 +
                    (double)d2 * d2;
        double fn = (double)retr;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            th += __shfl_down_sync(0xffffffffu, th, o);
            fn += __shfl_down_sync(0xffffffffu, fn, o);
        }
        if (lane == 0) { red_a[tid >> 5] = th; red_b[tid >> 5] = fn; }
        __syncthreads();                                            // (also: Delta of the whole CTA is in D)
        if (tid == 0) {
            double a = 0.0, b = 0.0;
#pragma unroll
            for (int w = 0; w < 8; ++w) { a += red_a[w]; b += red_b[w]; }
            part[0] = a; part[1] = b;
        }
    };

    __syncthreads();
    cl8_sync();                                                     // all CTAs are resident before the first remote access
    {
        Su3<T> none;
#pragma unroll
        for (int k = 0; k < 9; ++k) none.m[k] = Cx<T>(0, 0);
        update_and_measure(false, none);
    }

    for (;;) {
        CL8_STAMP(0);
        // ---- A: forward x, y (speculative: if the test below stops the loop, Delta is still in dreg) ----
        if (tid < 128) {
            cl8_line<-1>(D + 9 * tid, 1);
            cl8_bar128();
            cl8_line<-1>(D + 72 * (tid >> 3) + (tid & 7), 9);
        }
        CL8_STAMP(1);
        cl8_sync();                                           // barrier 1
        CL8_STAMP(2);
        // ---- B: pull the 16 (z,t) planes of (ky = rank/2; components 2 (rank%2), 2 (rank%2) + 1): the remote loads are
        //      issued first, the stopping test runs while they are in flight ----
        const int b_kx = tid & 7, b_zlr = (tid >> 3) & 3, b_cc = (tid >> 5) & 1;
        Cx<T> pulled[4];
        {
            const Cx<T>* src = D + (2 * (rank & 1) + b_cc) * C::kPad + 9 * ((rank >> 1) + 8 * b_zlr) + b_kx;
#pragma unroll
            for (int i = 0; i < 4; ++i) pulled[i] = cl8_ld(cl8_map(src, (unsigned)((tid >> 6) + 4 * i)), T());
        }
        {   // theta, F of the current links: every warp sums the 16 partials with the same butterfly
            const uint32_t p = cl8_map(part, (unsigned)(lane & 15));
            double a = cl8_ld_f64(p), b = cl8_ld_f64(p + 8);
#pragma unroll
            for (int o = 8; o > 0; o >>= 1) {
                a += __shfl_xor_sync(0xffffffffu, a, o);
                b += __shfl_xor_sync(0xffffffffu, b, o);
            }
            theta = a / (3.0 * (double)V);
            Fval = b / (12.0 * (double)V);
        }
        if ((theta < tol) || (iter >= max_iter)) break;             // lgf_fix's test (lgf_iterate: tol = -1)
        CL8_STAMP(3);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int rr = (tid >> 6) + 4 * i, z = 4 * (rr & 1) + b_zlr, tt = rr >> 1;
            Tb[((b_cc * 8 + tt) * 8 + z) * 8 + b_kx] = pulled[i];
        }
        __syncthreads();
        CL8_STAMP(4);
        // ---- C: forward z, forward t, scale, inverse t, inverse z (lanes along kx) ----
        if (tid < 128) {
            Cx<T>* zline = Tb + (tid >> 3) * 64 + (tid & 7);        // (cc, t) = tid / 8: z at stride 8
            cl8_line<-1>(zline, 8);
            cl8_bar128();
            {
                Cx<T>* tline = Tb + (tid >> 6) * 512 + ((tid >> 3) & 7) * 8 + (tid & 7);     // (cc, kz, kx): t at stride 64
                Cx<T> v[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) v[j] = tline[64 * j];
                RegFft<8, -1, T>::run(v);
#pragma unroll
                for (int j = 0; j < 8; ++j) v[j] = sc[j] * v[j];
                RegFft<8, +1, T>::run(v);
#pragma unroll
                for (int j = 0; j < 8; ++j) tline[64 * j] = v[j];
            }
            cl8_bar128();
            cl8_line<+1>(zline, 8);
        }
        CL8_STAMP(5);
        cl8_sync();                                           // barrier 2
        CL8_STAMP(6);
        // ---- D: pull the spectrum of the own sites back, inverse y, x ----
        {
            const int z = 4 * zh + zl;
#pragma unroll
            for (int c = 0; c < 4; ++c)
                D[c * C::kPad + lp] = cl8_ld(cl8_map(Tb + (((c & 1) * 8 + t) * 8 + z) * 8 + x, (unsigned)(2 * y + (c >> 1))), T());
        }
        __syncthreads();
        CL8_STAMP(7);
        if (tid < 128) {
            cl8_line<+1>(D + 72 * (tid >> 3) + (tid & 7), 9);
            cl8_bar128();
            cl8_line<+1>(D + 9 * tid, 1);
        }
        __syncthreads();
        CL8_STAMP(8);
        // ---- E: g of the own site (kept in registers; rows 0, 1 to shared memory for the neighbours) ----
        Su3<T> g;
        build_g(g, D[lp], D[C::kPad + lp], D[2 * C::kPad + lp], D[3 * C::kPad + lp], ha);
#pragma unroll
        for (int k = 0; k < 6; ++k) G[k * 256 + l] = g.m[k];
        CL8_STAMP(9);
        __syncthreads();                                            // this CTA's g are complete (x, y neighbours; D is free)
        cl8_arrive();                                         // barrier 3, waited for inside F before the z, t directions
        CL8_STAMP(10);
        // ---- F, G ----
        update_and_measure(true, g);
        ++iter;
        CL8_STAMP(13);
    }

    // ---- write the state back ----
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
#pragma unroll
        for (int c = 0; c < NC; ++c) st_cx(U + (size_t)(mu * NC + c) * V + s, links[(mu * NC + c) * 256 + l]);
#pragma unroll
    for (int c = 0; c < 4; ++c) st_cx(Dg + (size_t)c * V + s, dreg[c]);
#ifdef LGF_CL8_PROF
    if (tid == 0 && (rank == 0 || rank == 7))
        printf("cl8 rank %d: A %lld s1 %lld sum %lld B %lld C %lld s2 %lld D %lld invxy %lld E %lld s3 %lld F %lld s4 %lld G %lld total %lld\n", rank,
               prof[1] - prof[0], prof[2] - prof[1], prof[3] - prof[2], prof[4] - prof[3], prof[5] - prof[4], prof[6] - prof[5], prof[7] - prof[6],
               prof[8] - prof[7], prof[9] - prof[8], prof[10] - prof[9], prof[11] - prof[10], prof[12] - prof[11], prof[13] - prof[12], prof[13] - prof[0]);
#endif
    if (rank == 0 && tid == 0) {
        st->theta = theta;
        st->F = Fval;
        st->iter = iter;
        st->done = 1;
        st->pending = 0;
    }
    cl8_sync();                                                     // no CTA exits while a peer may still read its shared memory
}

}  // namespace lgf
