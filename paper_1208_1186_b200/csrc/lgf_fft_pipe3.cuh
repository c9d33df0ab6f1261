// lgf_fft_pipe3.cuh -- K3 (forward z, forward t, scale by p2max/(V p2(k)), inverse t, inverse z; SURVEY.md §8(a) row K3,
// north_star step 3) for (z,t) planes whose lines do not fit one thread's registers, done in THREE register stages per
// direction instead of four, i.e. five shared-memory passes instead of seven (48 x N_t: three instead of five).
//
// ncu on the two-stage kernel of lgf_fft_pipe.cuh at 64^4 fp64 (profiles/r1_v6_ncu_summary_64x4_f64_12.md) showed it bound
// by its seven lock-step shared-memory passes (mio_throttle the top stall, 114 M shared-memory wavefronts per launch, DRAM
// at 25 %).  A (z,t) plane of Nz x Nt = (A*B) x (C*D) points is a 4-index array; one thread can hold a B x C block of it
// (B*C <= 16..24 elements), so the second z stage and the first t stage run back to back in registers:
//
//   P1  z, stage 1   thread (cx, t,   n2z): DFT_A over m of x[n2z + B m], times w_Nz^{-n2z k1z}    -> position k1z*B + n2z
//   P2  z2 (x) t1    thread (cx, k1z, n2t): DFT_B over n2z for each m, then DFT_C over m of t = n2t + D m
//                                                                                                 -> (k1z*B + k2z, k1t*D + n2t)
//   P3  t, stage 2   thread (cx, zp,  k1t): times w_Nt^{-n2t k1t}, DFT_D over n2t, SCALE, DFT_D^-1, times w_Nt^{+n2t k1t}
//   P4  t1' (x) z2'  thread (cx, k1z, n2t): DFT_C^-1 over k1t, DFT_B^-1 over k2z
//   P5  z, stage 1'  thread (cx, t,   n2z): times w_Nz^{+n2z k1z}, DFT_A^-1 over k1z                -> global, natural order
//
// Every pass is in place per thread (a thread writes exactly the positions it read), so one barrier separates two
// passes.  Every twiddle multiplication sits in the pass where its run-time index (n2z in P1/P5, k1t in P3) is
// uniform across a warp, so the factors are literals selected by a warp-uniform switch (mul_tw<>, no table loads:
// the load/store unit is left to the shared-memory traffic).  When the t line fits the B x C block (D = 1: 48 x 8,
// 48 x 4, 48 x 6) P2, P3 and P4 are ONE pass.  The spectrum order is that of lgf_fft_ct.cuh (position k1*N2 + k2 holds
// frequency k1 + N1*k2); tiles, layout B and the ring are those of lgf_fft_pipe.cuh.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cuda.h>

#include "lgf_fft_pipe.cuh"

namespace lgf {

// Pass bodies.  ROW(t) -> pointer to element (z position 0, cx 0) of row t of the tile in shared memory; element
// (zp, cx) of that row sits at [zp * CX + cx].  `it` enumerates a pass's work items, cx fastest.
template <typename T, class SZ, class ST_, int CX>
struct Zt3 {
    static constexpr int NZ = SZ::kN, NT = ST_::kN, A = SZ::kN1, B = SZ::kN2, C = ST_::kN1, D = ST_::kN2;
    static constexpr int PZ = CX;
    static constexpr int kItems1 = CX * NT * B;      // P1, P5 (whole tile)
    static constexpr int kItems2 = CX * D * A;       // P2, P4 (and the fused P2-P4 when D = 1)
    static constexpr int kItems3 = CX * NZ * C;      // P3

    // P1 on rows [t0, t0 + RT): CX * RT * B items
    template <int RT, class ROW>
    __device__ static __forceinline__ void p1(int it, int t0, ROW&& row) {
        const int cx = it % CX, t = t0 + (it / CX) % RT, n2 = it / (CX * RT);
        Cx<T>* s = row(t) + cx;
        Cx<T> v[A];
        static_for<0, A>([&](auto m) { v[m.value] = s[(n2 + B * m.value) * PZ]; });
        RegFft<A, -1, T>::run(v);
        tw_rows<NZ, A, B, -1, T>(v, n2);
        static_for<0, A>([&](auto k1) { s[(k1.value * B + n2) * PZ] = v[k1.value]; });
    }
    // P5: the tile's rows straight to global memory (natural layout: gz = stride of z, gt = stride of t)
    template <class ROW>
    __device__ static __forceinline__ void p5(int it, ROW&& row, Cx<T>* base, long long gz, long long gt) {
        const int cx = it % CX, t = (it / CX) % NT, n2 = it / (CX * NT);
        const Cx<T>* s = row(t) + cx;
        Cx<T> v[A];
        static_for<0, A>([&](auto k1) { v[k1.value] = s[(k1.value * B + n2) * PZ]; });
        tw_rows<NZ, A, B, +1, T>(v, n2);
        RegFft<A, +1, T>::run(v);
        Cx<T>* gp = base + cx + (size_t)t * gt;
        static_for<0, A>([&](auto m) { st_cx(gp + (size_t)(n2 + B * m.value) * gz, v[m.value]); });
    }
    // row2(lo, hi) -> row holding logical t position lo + D*hi (P2 reads t = n2t + D m and writes position k1t*D + n2t:
    // the same rows).  TWP2: the t twiddles w_Nt^{-+ n2t k1t} are applied here (and in P4) from the table
    // twt[n2t][k1t - 1] = exp(+2 pi i n2t k1t / Nt) in shared memory instead of in P3, which is bound by the FP64 pipe
    // while P2 and P4 are bound by shared memory; n2t0: first n2t of the range this call covers.
    template <bool TWP2, int NN2T = D, class ROW2>
    __device__ static __forceinline__ void p2(int it, ROW2&& row2, const Cx<T>* twt = nullptr, int n2t0 = 0) {
        const int cx = it % CX, n2t = n2t0 + (it / CX) % NN2T, k1z = it / (CX * NN2T);
        const int off = k1z * B * PZ + cx;
        Cx<T> tw[C > 1 ? C - 1 : 1];
        if constexpr (TWP2) static_for<1, C>([&](auto k) { tw[k.value - 1] = twt[n2t * (C - 1) + k.value - 1]; });
        Cx<T> e[C][B];
        static_for<0, C>([&](auto m) {
            const Cx<T>* r = row2(n2t, m.value) + off;
            static_for<0, B>([&](auto j) { e[m.value][j.value] = r[j.value * PZ]; });
            RegFft<B, -1, T>::run(e[m.value]);
        });
        static_for<0, B>([&](auto j) {
            Cx<T> u[C];
            static_for<0, C>([&](auto m) { u[m.value] = e[m.value][j.value]; });
            RegFft<C, -1, T>::run(u);
            if constexpr (TWP2) static_for<1, C>([&](auto k) { u[k.value] = u[k.value] * conj(tw[k.value - 1]); });
            static_for<0, C>([&](auto m) { e[m.value][j.value] = u[m.value]; });
        });
        static_for<0, C>([&](auto k1t) {
            Cx<T>* r = row2(n2t, k1t.value) + off;
            static_for<0, B>([&](auto j) { r[j.value * PZ] = e[k1t.value][j.value]; });
        });
    }
    template <bool TWP2, int NN2T = D, class ROW2>
    __device__ static __forceinline__ void p4(int it, ROW2&& row2, const Cx<T>* twt = nullptr, int n2t0 = 0) {
        const int cx = it % CX, n2t = n2t0 + (it / CX) % NN2T, k1z = it / (CX * NN2T);
        const int off = k1z * B * PZ + cx;
        Cx<T> tw[C > 1 ? C - 1 : 1];
        if constexpr (TWP2) static_for<1, C>([&](auto k) { tw[k.value - 1] = twt[n2t * (C - 1) + k.value - 1]; });
        Cx<T> e[C][B];
        static_for<0, C>([&](auto k1t) {
            const Cx<T>* r = row2(n2t, k1t.value) + off;
            static_for<0, B>([&](auto j) { e[k1t.value][j.value] = r[j.value * PZ]; });
        });
        static_for<0, B>([&](auto j) {
            Cx<T> u[C];
            static_for<0, C>([&](auto m) { u[m.value] = e[m.value][j.value]; });
            if constexpr (TWP2) static_for<1, C>([&](auto k) { u[k.value] = u[k.value] * tw[k.value - 1]; });
            RegFft<C, +1, T>::run(u);
            static_for<0, C>([&](auto m) { e[m.value][j.value] = u[m.value]; });
        });
        static_for<0, C>([&](auto m) {
            RegFft<B, +1, T>::run(e[m.value]);
            Cx<T>* r = row2(n2t, m.value) + off;
            static_for<0, B>([&](auto j) { r[j.value * PZ] = e[m.value][j.value]; });
        });
    }
    // P5 in place (shared memory -> shared memory): the TMA unit stores the tile afterwards
    template <int RT, class ROW>
    __device__ static __forceinline__ void p5s(int it, int r0, ROW&& row) {
        const int cx = it % CX, r = r0 + (it / CX) % RT, n2 = it / (CX * RT);
        Cx<T>* s = row(r) + cx;
        Cx<T> v[A];
        static_for<0, A>([&](auto k1) { v[k1.value] = s[(k1.value * B + n2) * PZ]; });
        tw_rows<NZ, A, B, +1, T>(v, n2);
        RegFft<A, +1, T>::run(v);
        static_for<0, A>([&](auto m) { s[(n2 + B * m.value) * PZ] = v[m.value]; });
    }
    // x, y part of p^2 for the tile's cx-th (x,y) position (K2 left the x and y spectra digit-swapped)
    __device__ static __forceinline__ void momentum_xy(const ZtArgs& A_, long long tile_off, int cx, T& pxy, bool& zero_xy) {
        const long long sxy = tile_off + cx;
        const int ypos = int(sxy / A_.Lx), xpos = int(sxy - (long long)ypos * A_.Lx);
        const int kx = (xpos / A_.x_n2) + A_.x_n1 * (xpos % A_.x_n2), ky = (ypos / A_.y_n2) + A_.y_n1 * (ypos % A_.y_n2);
        pxy = reinterpret_cast<const T*>(A_.psq_x)[kx] + reinterpret_cast<const T*>(A_.psq_y)[ky];
        zero_xy = (kx | ky) == 0;
    }
    // four quotients num / d_i from ONE division (fp64: 20 instead of 36 FP64-pipe instructions; each result carries
    // three more roundings than a plain quotient, ~4e-16 relative); fp32 uses the fast hardware quotient directly
    __device__ static __forceinline__ void quot4(double num, const double* d, double* q) {
        const double p01 = d[0] * d[1], p23 = d[2] * d[3];
        const double r = fast_div(num, p01 * p23);
        const double r01 = r * p23, r23 = r * p01;        // num/(d0 d1), num/(d2 d3)
        q[0] = r01 * d[1]; q[1] = r01 * d[0]; q[2] = r23 * d[3]; q[3] = r23 * d[2];
    }
    __device__ static __forceinline__ void quot4(float num, const float* d, float* q) {
        for (int i = 0; i < 4; ++i) q[i] = fast_div(num, d[i]);
    }
    // TWP2: the twiddles are applied in P2 / P4 (see p2), otherwise here
    template <bool TWP2, class ROW2>
    __device__ static __forceinline__ void p3(int it, ROW2&& row2, const ZtArgs& A_, long long tile_off) {
        const int cx = it % CX, zp = (it / CX) % NZ, k1t = it / (CX * NZ);
        const int off = zp * PZ + cx;
        T pxyz; bool zero;
        momentum_xy(A_, tile_off, cx, pxyz, zero);
        const int kz = SZ::freq_of_pos(zp);
        pxyz += reinterpret_cast<const T*>(A_.psq_z)[kz];
        zero = zero && kz == 0;
        const T num = (T)A_.scale_num;
        Cx<T> v[D];
        static_for<0, D>([&](auto j) { v[j.value] = row2(j.value, k1t)[off]; });
        if constexpr (!TWP2) tw_rows<NT, D, C, -1, T>(v, k1t);
        RegFft<D, -1, T>::run(v);
        if constexpr (D % 4 == 0) {
            static_for<0, D / 4>([&](auto g) {
                T den[4], sc[4];
                static_for<0, 4>([&](auto i) {
                    const int kt = k1t + C * (4 * g.value + i.value);            // frequency held at position k1t*D + k2
                    den[i.value] = (zero && kt == 0) ? T(1) : pxyz + psq_t_half(A_, kt <= NT / 2 ? kt : NT - kt, T());
                });
                quot4(num, den, sc);
                static_for<0, 4>([&](auto i) {
                    const int kt = k1t + C * (4 * g.value + i.value);
                    v[4 * g.value + i.value] = ((zero && kt == 0) ? T(0) : sc[i.value]) * v[4 * g.value + i.value];
                });
            });
        } else {
            static_for<0, D>([&](auto k2) {
                const int kt = k1t + C * k2.value;
                const T den = pxyz + psq_t_half(A_, kt <= NT / 2 ? kt : NT - kt, T());   // p^2 is even in k_t (table by value)
                const T sc = (zero && kt == 0) ? T(0) : fast_div(num, den);
                v[k2.value] = sc * v[k2.value];
            });
        }
        RegFft<D, +1, T>::run(v);
        if constexpr (!TWP2) tw_rows<NT, D, C, +1, T>(v, k1t);
        static_for<0, D>([&](auto j) { row2(j.value, k1t)[off] = v[j.value]; });
    }
    // D = 1 (the whole t line inside the B x C block): P2, P3 and P4 in one pass
    template <class ROW>
    __device__ static __forceinline__ void p234(int it, ROW&& row, const ZtArgs& A_, long long tile_off) {
        static_assert(D == 1, "fused middle pass needs the whole t line in the block");
        const int cx = it % CX, k1z = it / CX;
        const int off = k1z * B * PZ + cx;
        T pxy; bool zero_xy;
        momentum_xy(A_, tile_off, cx, pxy, zero_xy);
        const T num = (T)A_.scale_num;
        Cx<T> e[C][B];
        static_for<0, C>([&](auto m) {
            const Cx<T>* r = row(m.value) + off;
            static_for<0, B>([&](auto j) { e[m.value][j.value] = r[j.value * PZ]; });
            RegFft<B, -1, T>::run(e[m.value]);
        });
        static_for<0, B>([&](auto j) {
            const int kz = k1z + A * j.value;                                    // frequency at z position k1z*B + j
            const T pxyz = pxy + reinterpret_cast<const T*>(A_.psq_z)[kz];
            const bool zero = zero_xy && kz == 0;
            Cx<T> u[C];
            static_for<0, C>([&](auto m) { u[m.value] = e[m.value][j.value]; });
            RegFft<C, -1, T>::run(u);
            static_for<0, C / 2 + 1>([&](auto kt) {                              // one quotient serves k_t and N_t - k_t
                constexpr int k = kt.value;
                const T den = pxyz + psq_t_half(A_, k, T());
                const T sc = (zero && k == 0) ? T(0) : fast_div(num, den);
                u[k] = sc * u[k];
                if constexpr (k != 0 && 2 * k != C) u[C - k] = sc * u[C - k];
            });
            RegFft<C, +1, T>::run(u);
            static_for<0, C>([&](auto m) { e[m.value][j.value] = u[m.value]; });
        });
        static_for<0, C>([&](auto m) {
            RegFft<B, +1, T>::run(e[m.value]);
            Cx<T>* r = row(m.value) + off;
            static_for<0, B>([&](auto j) { r[j.value * PZ] = e[m.value][j.value]; });
        });
    }
};

// Ring of whole tiles, NG thread groups of GT threads (the structure of fft_zt_pipe).
template <typename T, class SZ, class ST_, int CX, int GT, int NG, int NBUF>
__global__ void __launch_bounds__(GT * NG, 1)
fft_zt_pipe3(const Cx<T>* inB, Cx<T>* out, const __grid_constant__ ZtArgs A, const int* done) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    typedef Zt3<T, SZ, ST_, CX> P;
    constexpr int NZ = SZ::kN, NT = ST_::kN, PT = CX * (NZ + 1), TILE = PT * NT;
    static_assert((TILE * sizeof(Cx<T>)) % 16 == 0, "bulk copy alignment");
    static_assert(NBUF >= NG && GT % 32 == 0, "ring");
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(pipe_smem + sizeof(Cx<T>) * (size_t)NBUF * TILE);
    const int tid = threadIdx.x, g = tid / GT, gtid = tid - g * GT;
    const int ntiles = 4 * A.nbatch * A.tiles_per_comp;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const long long gz = A.LxLy, gt = A.LxLy * NZ;

    auto issue = [&](int i) {
        const int buf = i % NBUF;
        const size_t id = (size_t)blockIdx.x + (size_t)i * gridDim.x;
        const uint32_t bytes = (uint32_t)(TILE * sizeof(Cx<T>));
        mbar_arrive_expect_tx(&full[buf], bytes);
        bulk_g2s(bufs + (size_t)buf * TILE, inB + id * (size_t)TILE, bytes, &full[buf]);
    };
    if (tid == 0) {
        for (int b = 0; b < NBUF; ++b) mbar_init(&full[b], 1);
        mbar_fence_init();
        for (int i = 0; i < NBUF && i < my_tiles; ++i) issue(i);
    }
    __syncthreads();

    for (int i = g; i < my_tiles; i += NG) {
        const int buf = i % NBUF;
        Cx<T>* tile = bufs + (size_t)buf * TILE;
        auto row = [&](int t) { return tile + t * PT; };
        const int id = (int)blockIdx.x + i * (int)gridDim.x;
        const int comp = id / A.tiles_per_comp;
        const int tidx = id - comp * A.tiles_per_comp;
        const long long tile_off = (long long)tidx * CX;
        Cx<T>* base = out + (size_t)comp * A.V + tile_off;
        mbar_wait(&full[buf], (uint32_t)((i / NBUF) & 1));

        for (int it = gtid; it < P::kItems1; it += GT) P::template p1<NT>(it, 0, row);
        group_sync<GT, NG>(g);
        if constexpr (P::D == 1) {
            for (int it = gtid; it < P::kItems2; it += GT) P::p234(it, row, A, tile_off);
            group_sync<GT, NG>(g);
        } else {
            auto row2 = [&](int lo, int hi) { return tile + (lo + P::D * hi) * PT; };
            for (int it = gtid; it < P::kItems2; it += GT) P::template p2<false, P::D>(it, row2);
            group_sync<GT, NG>(g);
            for (int it = gtid; it < P::kItems3; it += GT) P::template p3<false>(it, row2, A, tile_off);
            group_sync<GT, NG>(g);
            for (int it = gtid; it < P::kItems2; it += GT) P::template p4<false, P::D>(it, row2);
            group_sync<GT, NG>(g);
        }
        for (int it = gtid; it < P::kItems1; it += GT) P::p5(it, row, base, gz, gt);
        fence_proxy_async();
        group_sync<GT, NG>(g);
        if (i + NBUF < my_tiles && gtid == 0) issue(i + NBUF);
    }
}

// Quarter-tile ring with asynchronous output for planes too large for a ring of whole tiles (64 x 64: a CX = 2 fp64 /
// CX = 4 fp32 tile is 133 KB).  ncu on a half-tile ring with per-thread stores at 64^4 (profiles/r2_k3_*): 43 % of the kernel's warp-time
// sat in P5's scattered 32-byte global stores and the barrier behind them (stall_lg: every STG.128 of a warp is 16 tag
// requests), and the second half-tile's fetch was exposed behind every tile.  Here
//  * P5 runs in place in shared memory and the TMA unit stores the tile (cp.async.bulk.tensor, SASS UTMASTG: a 5-D box
//    whose z extent Nz+1 exceeds the tensor's Nz, so the pad entry of every row is clipped), asynchronously, while the
//    CTA is already transforming the next tile;
//  * the tile travels as four QUARTERS through a ring of six quarter buffers, and layout B stores the t rows in the
//    order [q][m][l], where t = n2t + D m and n2t = q D/4 + l: quarter q holds the rows of its D/4 values of
//    n2t for ALL m, which makes it closed under P1 AND P2 (P2 of one n2t touches t = n2t + D m, m < C), and inside a
//    quarter consecutive n2t are consecutive rows (the lanes of P2 / P4 run along n2t: conflict-free with the padded
//    pitch; the order [n2t][m] measured 106 M bank conflicts per launch).  Both passes run on the first two quarters
//    while the other two are still in flight -- their buffers are the ones the previous tile's first two quarter
//    stores are draining.
// One I/O thread (the CTA's last: idle in the half-tile passes in fp64) owns all bulk groups: it waits for the
// stores' shared-memory reads (wait_group.read) before it re-arms a buffer.
template <typename T, class SZ, class ST_, int CX, int GT>
__global__ void __launch_bounds__(GT, 1)
fft_zt_pipe3q(const Cx<T>* inB, Cx<T>* out, const __grid_constant__ ZtArgs A, const int* done,
              const __grid_constant__ CUtensorMap omap) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    typedef Zt3<T, SZ, ST_, CX> P;
    constexpr int NZ = SZ::kN, NT = ST_::kN, PT = CX * (NZ + 1), QR = NT / 4, QE = PT * QR, NB = 6;
    constexpr int C = P::C, D = P::D, LQ = D / 4;             // LQ: n2t values per quarter
    static_assert(D % 4 == 0 && (QE * sizeof(Cx<T>)) % 128 == 0 && GT % 32 == 0, "quarter tiles");
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    Cx<T>* twt = bufs + (size_t)NB * QE;                       // [n2t][k1t - 1] = exp(+2 pi i n2t k1t / Nt)
    uint64_t* full = reinterpret_cast<uint64_t*>(twt + D * (C - 1));
    const int tid = threadIdx.x;
    const bool io = tid == GT - 1;
    const int ntiles = 4 * A.nbatch * A.tiles_per_comp;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;

    auto issue = [&](int k) {             // quarter k = 4 * (tile index of this CTA) + q
        const int buf = k % NB;
        const size_t id = (size_t)blockIdx.x + (size_t)(k >> 2) * gridDim.x;
        const uint32_t bytes = (uint32_t)(QE * sizeof(Cx<T>));
        mbar_arrive_expect_tx(&full[buf], bytes);
        bulk_g2s(bufs + (size_t)buf * QE, inB + id * (size_t)(4 * QE) + (size_t)(k & 3) * QE, bytes, &full[buf]);
    };
    auto wait_q = [&](int k) { mbar_wait(&full[k % NB], (uint32_t)((k / NB) & 1)); };
    if (io) {
        for (int b = 0; b < NB; ++b) mbar_init(&full[b], 1);
        mbar_fence_init();
        for (int k = 0; k < NB && k < 4 * my_tiles; ++k) issue(k);
    }
    for (int e = tid; e < D * (C - 1); e += GT) {
        const int n2t = e / (C - 1), k1t = e % (C - 1) + 1;
        twt[e] = ldg_cx(reinterpret_cast<const Cx<T>*>(A.twt_inv) + (n2t * k1t) % NT);
    }
    __syncthreads();

    for (int i = 0; i < my_tiles; ++i) {
        const int b0 = (4 * i) % NB;
        auto qbase = [&](int q) { int b = b0 + q; b -= b >= NB ? NB : 0; return bufs + (size_t)b * QE; };
        auto rowp = [&](int r) { const int q = r / QR; return qbase(q) + (r - q * QR) * PT; };                      // physical row
        auto row2 = [&](int lo, int hi) { const int q = lo / LQ; return qbase(q) + (hi * LQ + (lo - q * LQ)) * PT; };  // t position lo + D hi
        const int id = (int)blockIdx.x + i * (int)gridDim.x;
        const int comp = id / A.tiles_per_comp;
        const int tidx = id - comp * A.tiles_per_comp;
        const long long tile_off = (long long)tidx * CX;

#pragma unroll
        for (int h = 0; h < 2; ++h) {
            wait_q(4 * i + 2 * h);
            wait_q(4 * i + 2 * h + 1);
            for (int it = tid; it < CX * 2 * QR * P::B; it += GT) P::template p1<2 * QR>(it, 2 * h * QR, rowp);
            __syncthreads();
            for (int it = tid; it < CX * 2 * LQ * P::A; it += GT) P::template p2<true, 2 * LQ>(it, row2, twt, 2 * h * LQ);
        }
        __syncthreads();
        for (int it = tid; it < P::kItems3; it += GT) P::template p3<true>(it, row2, A, tile_off);
        if (io && i > 0 && i + 1 < my_tiles) {
            // quarters 0, 1 of the NEXT tile go to the buffers of the PREVIOUS tile's quarters 2, 3, whose stores were the
            // last thing issued before this tile and have drained by now
            bulk_wait_group_read<0>();
            issue(4 * i + 4);
            issue(4 * i + 5);
        }
        __syncthreads();
        // after P3 the halves are independent again: P4, P5 and the stores of the first half run (and its two quarter
        // stores drain) while the second half is still being transformed.  The TMA unit serves its requests in order
        // (measured: fetches issued behind the second half's stores landed a whole store-drain late), so the fetch of
        // the next tile's quarters 2, 3 -- into the first half's buffers -- is issued BEFORE the second half's stores.
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            for (int it = tid; it < CX * 2 * LQ * P::A; it += GT) P::template p4<true, 2 * LQ>(it, row2, twt, 2 * h * LQ);
            __syncthreads();
            for (int it = tid; it < CX * 2 * QR * P::B; it += GT) P::template p5s<2 * QR>(it, 2 * h * QR, rowp);
            fence_proxy_async();
            __syncthreads();
            if (io) {
                if (h == 1 && i + 1 < my_tiles) {
                    bulk_wait_group_read<0>();             // this tile's quarter stores 0, 1 have read their buffers
                    issue(4 * i + 6);
                    issue(4 * i + 7);
                }
                // tensor coordinates: (2 reals * xy position, z, t mod D, t div D, component); quarter q holds t mod D in [q LQ, (q+1) LQ)
#pragma unroll
                for (int q = 2 * h; q < 2 * h + 2; ++q) {
                    tma_store_5d(&omap, qbase(q), (int)(2 * tile_off), 0, q * LQ, 0, comp);
                    bulk_commit_group();
                }
            }
        }
    }
    if (io) bulk_wait_group<0>();
}

}  // namespace lgf
