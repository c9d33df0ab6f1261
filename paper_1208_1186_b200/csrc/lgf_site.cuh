// lgf_site.cuh -- per-site kernels: K1 (Delta / theta / F), K5 (g-build + link update),
// boundary layout transposes.  Product code (sm_100a); shares nothing with oracle/.
//
// Device layouts:
//   links  U[mu][c][s]  complex<T>, c = 0..NC-1 row-major matrix element (NC = 9: 18-real,
//                       NC = 6: rows 0,1 only = 12-real), s lexicographic x fastest
//   Delta  D[c][s]      complex<T>, c = 0..3 packed: D01, D02, D12, Im D00 + i Im D11
#pragma once
#include "lgf_math.cuh"


namespace lgf {

struct Geom {
    int L[4];    // Lx, Ly, Lz, Lt
    int nb[4];   // tiles per axis for the per-site kernels; launched as a (nb0, nb1, nb2 * nb3) grid
    long long V;
    // walk order of the (z, t) tiles: blockIdx.z = (zblk * nb3 + bt) * zb + zi, bz = zblk * zb + zi.  zb = nb2 is the
    // plain order (t slowest).  On lattices whose t-slice of links outgrows the L2 (64^4: 100 MB) a z-block of
    // zb tiles is walked through all t before the next z-block starts, so that the t-neighbour data (backward
    // links in K1, forward Delta~ in K5) is re-read from L2 one z-block later, not from DRAM one t-slice later.
    int zb;
    unsigned int zb_magic, nb3_magic;     // ceil(2^32 / zb), ceil(2^32 / nb3)  (0 when the divisor is 1)
    // batched contexts (lgf_create_batch: B independent lattices of the same shape per launch): blockIdx.z =
    // b * nzt + (z,t) tile, nzt = nb2 * nb3; every field of lattice b sits b * (its size) behind lattice 0's
    int nzt;
    unsigned int nzt_magic;
    int nblocks;                          // CTAs per lattice = nb0 * nb1 * nzt (segment of the partials array)
};

// The site kernels are launched on a 3-D grid (x tiles, y tiles, z tiles * t tiles): same CTA order as a linear
// grid, but no runtime integer divisions in the prologue (they were ~100 of k5s's ~600 instructions per thread
// and sat in front of the first load).  All operands are < 2^16, so the multiply-high quotients are exact.
__device__ __forceinline__ unsigned div_magic(unsigned n, unsigned magic) { return magic ? __umulhi(n, magic) : n; }
__device__ __forceinline__ void split_zt(const Geom& g, unsigned bzt, unsigned& bz, unsigned& bt) {
    const unsigned q = div_magic(bzt, g.zb_magic), zi = bzt - q * (unsigned)g.zb;
    const unsigned zblk = div_magic(q, g.nb3_magic);
    bt = q - zblk * (unsigned)g.nb[3];
    bz = zblk * (unsigned)g.zb + zi;
}
__device__ __forceinline__ unsigned linear_block() { return blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z); }
// which lattice of the batch and which (z,t) tile inside it a grid z index means (z < 2^16: exact multiply-high quotient)
struct BatchPos { unsigned b, bzt; };
__device__ __forceinline__ BatchPos batch_pos(const Geom& g, unsigned z) {
    BatchPos p;
    p.b = div_magic(z, g.nzt_magic);
    p.bzt = z - p.b * (unsigned)g.nzt;
    return p;
}
// index of this CTA's (theta, F) partial: lattice b's segment, the CTA's position inside its lattice
__device__ __forceinline__ unsigned partial_index(const Geom& g, const BatchPos& p) {
    return p.b * (unsigned)g.nblocks + blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * p.bzt);
}

// Loop / reduction state, lives in the workspace (device memory).
struct DevState {
    double theta;
    double F;
    long long iter;          // link updates applied since the run started
    int done;                // 1: theta < tol reached (or max_iter) -> later kernels are no-ops
    unsigned int ticket;     // K1 block counter for the last-block reduction
    double tol;
    long long max_iter;
    int cur;                 // which of the two link buffers holds the current field (fused path swaps them)
    int pending;             // K1 has written the partials of an applied update that k1_finish has not folded in yet
};

// Resident CTAs per SM each site kernel is compiled for (= register cap 65536 / (256 * n)); measured
// best of 1..4 per precision and storage at 32^4.
template <typename T, int NC> struct SiteOcc {
#ifdef LGF_K1_OCC
    static constexpr int k1 = LGF_K1_OCC;
#else
    static constexpr int k1 = sizeof(T) == 8 ? 2 : 4;     // fp32 at 4 (64 registers): K1 65.7 -> 61.6 us 18-real, 52.6 -> 49.2 us 12-real at 32^4
#endif
    static constexpr int k5 = sizeof(T) == 8 ? 2 : (NC == 6 ? 4 : 2);
    static constexpr int k5m = sizeof(T) == 8 ? 2 : 3;
};

template <int TX, int TY, int TZ, int TT>
struct SiteTile {
    static constexpr int kThreads = TX * TY * TZ * TT;
    // thread -> lattice coordinates of its site; returns false outside the lattice
    // REVERSE: walk the tiles from the last to the first.  K1 does (it follows K5, which walks forward, so the
    // links K5 wrote last are still in L2 when K1 starts with them).
    // bp: batch_pos of blockIdx.z (REVERSE: of gridDim.z - 1 - blockIdx.z)
    template <bool REVERSE = false>
    __device__ static __forceinline__ bool coords(const Geom& g, const BatchPos& bp, int x[4]) {
        const unsigned bx = REVERSE ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
        const unsigned by = REVERSE ? gridDim.y - 1 - blockIdx.y : blockIdx.y;
        unsigned bz, bt;
        split_zt(g, bp.bzt, bz, bt);
        int t = threadIdx.x;
        x[0] = bx * TX + t % TX; t /= TX;
        x[1] = by * TY + t % TY; t /= TY;
        x[2] = bz * TZ + t % TZ; t /= TZ;
        x[3] = bt * TT + t;
        return x[0] < g.L[0] && x[1] < g.L[1] && x[2] < g.L[2] && x[3] < g.L[3];
    }
};

// (32-bit arithmetic: V < 2^31, a lattice beyond that would need > 1 TB of links)
__device__ __forceinline__ long long site_index(const Geom& g, const int x[4]) {
    return (long long)(x[0] + g.L[0] * (x[1] + g.L[1] * (x[2] + g.L[2] * x[3])));
}
__device__ __forceinline__ long long axis_stride(const Geom& g, int mu) {
    long long s = 1;
    for (int i = 0; i < mu; ++i) s *= g.L[i];
    return s;
}

// Load one link into registers; in 12-real mode rebuild row 2.
// stream: this is the last use of the link in the kernel (L2 evict-first); otherwise a plain load
// (stream is a compile-time constant at every call site once the direction loops are unrolled)
template <typename T, int NC>
__device__ __forceinline__ void load_link(Su3<T>& u, const Cx<T>* __restrict__ U, long long V, int mu, long long s, int stream = 0) {
    const Cx<T>* p = U + (size_t)mu * NC * V + s;
    if (stream) {
        const uint64_t pol = l2_evict_first_policy();
#pragma unroll
        for (int c = 0; c < NC; ++c) u.m[c] = ld_cx_stream(p + (size_t)c * V, pol);
    } else {
#pragma unroll
        for (int c = 0; c < NC; ++c) u.m[c] = ld_cx(p + (size_t)c * V);
    }
    if (NC == 6) rebuild_row2(u);
}

// Deterministic block reduction of two doubles; result valid in thread 0.
template <int NT>
__device__ __forceinline__ void block_sum2(double& a, double& b) {
    __shared__ double sa[NT / 32], sb[NT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = (l < NT / 32) ? sa[l] : 0.0;
        b = (l < NT / 32) ? sb[l] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, o);
            b += __shfl_down_sync(0xffffffffu, b, o);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K1  delta_theta_F  (north_star step 1)
//   M(x) = sum_mu [U_mu(x-mu) - U_mu(x)],  A = M - M^+,  Delta = A - (Tr A/3) 1  -> packed 4 complex
//   theta = (1/(3V)) sum |Delta_ij|^2,  F = (1/(12V)) sum Re Tr U_mu(x); sums in fp64, fixed order.
// mode: 0 = plain measurement; 1 = end of an iteration (skipped if st->done, bumps st->iter and
// evaluates the stopping test theta < tol / iter >= max_iter on the device).
// ---------------------------------------------------------------------------------------------
template <typename T, int NC, class Tile>
__global__ void __launch_bounds__(Tile::kThreads, SiteOcc<T, NC>::k1)
k1_delta_theta_F(const Cx<T>* __restrict__ U, Cx<T>* __restrict__ D, double2* __restrict__ partials,
                 DevState* st, Geom g, int mode) {
    pdl_entry();
#ifndef LGF_K1_FORWARD
    const BatchPos bp = batch_pos(g, gridDim.z - 1 - blockIdx.z);
#else
    const BatchPos bp = batch_pos(g, blockIdx.z);
#endif
    st += bp.b;
    U += (size_t)bp.b * 4 * NC * g.V;
    D += (size_t)bp.b * 4 * g.V;
    if (mode == 1 && *reinterpret_cast<const volatile int*>(&st->done)) return;
    if (mode == 1 && threadIdx.x == 0 && partial_index(g, bp) == bp.b * (unsigned)g.nblocks) st->pending = 1;    // folded in by the next k1_finish
    int x[4];
#ifndef LGF_K1_FORWARD
    const bool valid = Tile::template coords<true>(g, bp, x);
#else
    const bool valid = Tile::template coords<false>(g, bp, x);
#endif
    double th = 0.0, fn = 0.0;
    if (valid) {
        const int s = (int)site_index(g, x);
        // only the anti-Hermitian traceless part of M = sum_mu [U_mu(x-mu) - U_mu(x)] is needed: accumulate its
        // 9 reals link by link (the projection is linear) instead of the full 3x3 sum
        Cx<T> c0(0, 0), c1(0, 0), c2(0, 0);
        T a0 = 0, a1 = 0, a2 = 0, retr = 0;
        int stride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int sb = (x[mu] == 0) ? s + stride * (g.L[mu] - 1) : s - stride;
            // measured at 32^4: evict-first link loads help K1 in fp32 (80 -> 69 us, the Delta it writes stays in
            // L2 for K2) and hurt in fp64 (122 -> 134 us, 18-real: the backward re-reads start missing L2)
            {
                Su3<T> a;
                load_link<T, NC>(a, U, g.V, mu, s, sizeof(T) == 4);
                c0 = c0 - (a.m[1] - conj(a.m[3]));
                c1 = c1 - (a.m[2] - conj(a.m[6]));
                c2 = c2 - (a.m[5] - conj(a.m[7]));
                a0 -= a.m[0].im; a1 -= a.m[4].im; a2 -= a.m[8].im;
                retr += a.m[0].re + a.m[4].re + a.m[8].re;
            }
            {
                Su3<T> b;
                load_link<T, NC>(b, U, g.V, mu, sb, sizeof(T) == 4);
                c0 = c0 + (b.m[1] - conj(b.m[3]));
                c1 = c1 + (b.m[2] - conj(b.m[6]));
                c2 = c2 + (b.m[5] - conj(b.m[7]));
                a0 += b.m[0].im; a1 += b.m[4].im; a2 += b.m[8].im;
            }
            stride *= g.L[mu];
        }
        // diagonal of A = M - M^+ is i * 2 Im M_ii; remove trace/3
        a0 *= T(2); a1 *= T(2); a2 *= T(2);
        const T tr3 = (a0 + a1 + a2) / T(3);
        const T d0 = a0 - tr3, d1 = a1 - tr3, d2 = a2 - tr3;
        const uint64_t keep = l2_evict_last_policy();
        st_cx_keep(D + s, c0, keep);
        st_cx_keep(D + (size_t)g.V + s, c1, keep);
        st_cx_keep(D + (size_t)2 * g.V + s, c2, keep);
        st_cx_keep(D + (size_t)3 * g.V + s, Cx<T>(d0, d1), keep);
        th = 2.0 * ((double)norm2(c0) + (double)norm2(c1) + (double)norm2(c2)) + (double)d0 * d0 +
             (double)d1 * d1 + (double)d2 * d2;
        fn = (double)retr;
    }
    block_sum2<Tile::kThreads>(th, fn);
    if (threadIdx.x == 0) partials[partial_index(g, bp)] = make_double2(th, fn);   // summed by k1_finish
}

// Second half of K1: one CTA sums the per-CTA (theta, F) partials in index order (deterministic, no
// float atomics), publishes theta and F and, at the end of an iteration (mode 1), bumps the
// iteration count and evaluates the stopping test on the device (mode 2: end of a FUSED iteration,
// which additionally swaps the roles of the two link buffers).  A separate tiny launch instead
// of a last-CTA ticket: the K1 CTAs then retire without a fence + atomic tail.
constexpr int kFinishThreads = 1024;
__global__ void __launch_bounds__(kFinishThreads)
k1_finish(const double2* __restrict__ partials, int n, DevState* st, double V, int mode) {
    pdl_entry();
    partials += (size_t)blockIdx.x * n;          // one CTA per lattice of a batched context
    st += blockIdx.x;
    if (mode >= 1 && *reinterpret_cast<volatile int*>(&st->done)) return;
    // mode 3: deferred end of an iteration -- launched beside the NEXT iteration's K2 (and once after the last
    // iteration of a batch); a no-op when the previous K1 has been folded in already
    if (mode == 3 && !*reinterpret_cast<volatile int*>(&st->pending)) return;
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < n; i += kFinishThreads) {
        const double2 p = partials[i];
        a += p.x;
        b += p.y;
    }
    block_sum2<kFinishThreads>(a, b);
    if (threadIdx.x == 0) {
        const double theta = a / (3.0 * V);
        st->theta = theta;
        st->F = b / (12.0 * V);
        if (mode >= 1) {
            st->pending = 0;
            const long long it = st->iter + 1;
            st->iter = it;
            if (mode == 2) st->cur ^= 1;     // fused update: the new links were written to the other buffer
            if (theta < st->tol || it >= st->max_iter) st->done = 1;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// K5  gbuild_update  (north_star steps 4, 5)
//   g(y) = reunitarise(1 + (alpha/2) Dt(y)) for y = x and the four forward neighbours,
//   U'_mu(x) = g(x) U_mu(x) g(x+mu)^+, in place (each link is read and written by one thread only).
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void load_g(Su3<T>& g, const Cx<T>* __restrict__ D, long long V, long long s, T ha) {
    const Cx<T> c0 = ld_cx(D + s), c1 = ld_cx(D + (size_t)V + s), c2 = ld_cx(D + (size_t)2 * V + s),
                c3 = ld_cx(D + (size_t)3 * V + s);
    build_g(g, c0, c1, c2, c3, ha);
}

template <typename T, int NC, class Tile>
__global__ void __launch_bounds__(Tile::kThreads, SiteOcc<T, NC>::k5)
k5_gbuild_update(Cx<T>* __restrict__ U, const Cx<T>* __restrict__ D, const DevState* st, Geom g, T half_alpha) {
    pdl_entry();
    const BatchPos bp = batch_pos(g, blockIdx.z);
    st += bp.b;
    U += (size_t)bp.b * 4 * NC * g.V;
    D += (size_t)bp.b * 4 * g.V;
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    int x[4];
    if (!Tile::coords(g, bp, x)) return;
    const long long s = site_index(g, x);
    constexpr int NR = NC / 3;  // rows to produce: 3 or 2
    Su3<T> g0;
    load_g(g0, D, g.V, s, half_alpha);
    long long stride = 1;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
        const long long sf = (x[mu] == g.L[mu] - 1) ? s - stride * (g.L[mu] - 1) : s + stride;
        Su3<T> gf, u;
        load_g(gf, D, g.V, sf, half_alpha);
        load_link<T, NC>(u, U, g.V, mu, s);
        // W = g0 * u (rows 0..NR-1), then U' = W * gf^+
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
        Cx<T>* p = U + (size_t)mu * NC * g.V + s;
#pragma unroll
        for (int i = 0; i < NR; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                Cx<T> acc = mulc(W[3 * i], gf.m[3 * j]);
                fma_cxc(acc, W[3 * i + 1], gf.m[3 * j + 1]);
                fma_cxc(acc, W[3 * i + 2], gf.m[3 * j + 2]);
                st_cx(p + (size_t)(3 * i + j) * g.V, acc);
            }
        stride *= g.L[mu];
    }
}

// ---------------------------------------------------------------------------------------------
// Boundary transposes: AoS links[s][mu][3][3] (complex<T>) <-> device U[mu][c][s].
// `aos` points at site `s0`; n sites are converted.
// ---------------------------------------------------------------------------------------------
template <typename T, int NC>
__global__ void aos_to_soa(const Cx<T>* __restrict__ aos, Cx<T>* __restrict__ U, long long V, long long s0, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // over n * 36
    if (i >= n * 36) return;
    const long long sl = i / 36;
    const int r = int(i - sl * 36), mu = r / 9, c = r % 9;
    if (c < NC) U[(size_t)(mu * NC + c) * V + s0 + sl] = aos[i];
}

template <typename T, int NC>
__global__ void soa_to_aos(const Cx<T>* __restrict__ U, Cx<T>* __restrict__ aos, long long V, long long s0, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // over n * 4
    if (i >= n * 4) return;
    const long long sl = i / 4;
    const int mu = int(i - sl * 4);
    Su3<T> u;
    load_link<T, NC>(u, U, V, mu, s0 + sl);
#pragma unroll
    for (int c = 0; c < 9; ++c) aos[i * 9 + c] = u.m[c];
}

// packed Delta D[c][s] -> [s][4] (debug/inspection hook)
template <typename T>
__global__ void delta_to_aos(const Cx<T>* __restrict__ D, Cx<T>* __restrict__ out, long long V) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= V * 4) return;
    out[i] = D[(size_t)(i & 3) * V + (i >> 2)];
}

}  // namespace lgf
