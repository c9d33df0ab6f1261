// lgf_site_mu.cuh -- K5 with one thread per (site, direction): four times the threads of the
// thread-per-site kernel, every load of a thread issued in one batch (one load phase instead of
// four).  (The same split was tried for K1 and measured 40 % slower than thread-per-site: it loses
// the in-CTA L1 reuse of the backward links.)
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_site.cuh"


namespace lgf {

// CTA = kSites lattice sites x 4 directions; thread t: site = t % kSites, mu = t / kSites (warp-uniform).
template <int TX, int TY, int TZ, int TT>
struct SiteTileMu {
    static constexpr int kSites = TX * TY * TZ * TT;
    static constexpr int kThreads = 4 * kSites;
    static_assert(kSites % 32 == 0, "mu must be warp-uniform");
    static constexpr int tx = TX, ty = TY, tz = TZ, tt = TT;
    __device__ static __forceinline__ bool coords(const Geom& g, const BatchPos& bp, int ls, int x[4]) {
        const unsigned bx = blockIdx.x, by = blockIdx.y;
        unsigned bz, bt;
        split_zt(g, bp.bzt, bz, bt);
        x[0] = bx * TX + ls % TX; ls /= TX;
        x[1] = by * TY + ls % TY; ls /= TY;
        x[2] = bz * TZ + ls % TZ; ls /= TZ;
        x[3] = bt * TT + ls;
        return x[0] < g.L[0] && x[1] < g.L[1] && x[2] < g.L[2] && x[3] < g.L[3];
    }
};

// stride of direction mu (warp-uniform mu, no dynamic register indexing)
__device__ __forceinline__ void dir_info(const Geom& g, int mu, const int x[4], long long& stride, int& xm, int& Lm) {
    const long long s1 = g.L[0], s2 = s1 * g.L[1], s3 = s2 * g.L[2];
    stride = mu == 0 ? 1 : (mu == 1 ? s1 : (mu == 2 ? s2 : s3));
    xm = mu == 0 ? x[0] : (mu == 1 ? x[1] : (mu == 2 ? x[2] : x[3]));
    Lm = mu == 0 ? g.L[0] : (mu == 1 ? g.L[1] : (mu == 2 ? g.L[2] : g.L[3]));
}

// K5, thread (site, mu): U'_mu(x) = g(x) U_mu(x) g(x+mu)^+; g(x) is rebuilt by each of the four
// direction threads of a site (8 Gram-Schmidt per site instead of 5, no barrier, no shared memory).
template <typename T, int NC, class Tile>
__global__ void __launch_bounds__(Tile::kThreads, SiteOcc<T, NC>::k5m)
k5m_gbuild_update(Cx<T>* __restrict__ U, const Cx<T>* __restrict__ D, const DevState* st, Geom g, T half_alpha) {
    pdl_entry();
    const BatchPos bp = batch_pos(g, blockIdx.z);
    st += bp.b;
    U += (size_t)bp.b * 4 * NC * g.V;
    D += (size_t)bp.b * 4 * g.V;
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    constexpr int NS = Tile::kSites;
    const int ls = threadIdx.x % NS, mu = threadIdx.x / NS;
    int x[4];
    if (!Tile::coords(g, bp, ls, x)) return;
    const long long s = site_index(g, x);
    long long stride; int xm, Lm;
    dir_info(g, mu, x, stride, xm, Lm);
    const long long sf = (xm == Lm - 1) ? s - stride * (Lm - 1) : s + stride;
    constexpr int NR = NC / 3;
    // all loads first
    Cx<T> d0[4], d1[4];
    Su3<T> u;
    Cx<T>* p = U + (size_t)mu * NC * g.V + s;
#pragma unroll
    for (int c = 0; c < 4; ++c) { d0[c] = ld_cx(D + (size_t)c * g.V + s); d1[c] = ld_cx(D + (size_t)c * g.V + sf); }
#pragma unroll
    for (int c = 0; c < NC; ++c) u.m[c] = ld_cx(p + (size_t)c * g.V);
    if (NC == 6) rebuild_row2(u);
    Su3<T> g0;
    build_g(g0, d0[0], d0[1], d0[2], d0[3], half_alpha);
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
    Su3<T> gf;
    build_g(gf, d1[0], d1[1], d1[2], d1[3], half_alpha);
#pragma unroll
    for (int i = 0; i < NR; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            Cx<T> acc = mulc(W[3 * i], gf.m[3 * j]);
            fma_cxc(acc, W[3 * i + 1], gf.m[3 * j + 1]);
            fma_cxc(acc, W[3 * i + 2], gf.m[3 * j + 2]);
            st_cx(p + (size_t)(3 * i + j) * g.V, acc);
        }
}

// ---------------------------------------------------------------------------------------------
// K5, thread (site, mu) with g shared through shared memory: every g of the tile and of its four
// forward halo faces is built ONCE by one thread (instead of 5-8 times per site), the link loads
// are issued before the g phase so that they overlap it, and a single barrier separates the two.
// Requires every L_mu to be a multiple of the tile extent (no ragged tiles).
// ---------------------------------------------------------------------------------------------
template <int TX, int TY, int TZ, int TT>
struct SiteTileS {
    static constexpr int tx = TX, ty = TY, tz = TZ, tt = TT;
    static constexpr int kSites = TX * TY * TZ * TT;
    static constexpr int kThreads = 4 * kSites;
    static constexpr int HX = TY * TZ * TT, HY = TX * TZ * TT, HZ = TX * TY * TT, HT = TX * TY * TZ;
    static constexpr int OX = kSites, OY = OX + HX, OZ = OY + HY, OT = OZ + HZ, NG = OT + HT;   // g slots
    static_assert(kSites % 32 == 0, "mu must be warp-uniform");
};

template <typename T, int NC, class Tile, int MINB>
__global__ void __launch_bounds__(Tile::kThreads, MINB)
k5s_gbuild_update(Cx<T>* __restrict__ U, const Cx<T>* __restrict__ D, const DevState* st, Geom g, T half_alpha) {
    pdl_entry();
    const BatchPos bp = batch_pos(g, blockIdx.z);
    st += bp.b;
    U += (size_t)bp.b * 4 * NC * g.V;
    D += (size_t)bp.b * 4 * g.V;
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    constexpr int TX = Tile::tx, TY = Tile::ty, TZ = Tile::tz, TT = Tile::tt, NS = Tile::kSites, NG = Tile::NG, NR = NC / 3;
    __shared__ Cx<T> G[9 * NG];
    unsigned bz, bt;
    split_zt(g, bp.bzt, bz, bt);
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = bz * TZ, t0 = bt * TT;
    const int s1 = g.L[0], s2 = s1 * g.L[1], s3 = s2 * g.L[2];      // 32-bit site arithmetic (V < 2^31)
    const int tid = threadIdx.x, ls = tid % NS, mu = tid / NS;
    const int lx = ls % TX, ly = (ls / TX) % TY, lz = (ls / (TX * TY)) % TZ, lt = ls / (TX * TY * TZ);
    const int s = (x0 + lx) + s1 * (y0 + ly) + s2 * (z0 + lz) + s3 * (t0 + lt);
    // ---- this thread's link: loads in flight during the whole g phase ----
    Su3<T> u;
    Cx<T>* p = U + (size_t)mu * NC * g.V + s;
#pragma unroll
    for (int c = 0; c < NC; ++c) u.m[c] = ld_cx(p + (size_t)c * g.V);
    // ---- g of the tile and of its forward halo faces, one item per thread ----
    for (int i = tid; i < NG; i += Tile::kThreads) {
        int ax, ay, az, at;           // local coordinates of the item's site (may equal the tile extent: halo)
        if (i < Tile::OX) { ax = i % TX; ay = (i / TX) % TY; az = (i / (TX * TY)) % TZ; at = i / (TX * TY * TZ); }
        else if (i < Tile::OY) { const int h = i - Tile::OX; ax = TX; ay = h % TY; az = (h / TY) % TZ; at = h / (TY * TZ); }
        else if (i < Tile::OZ) { const int h = i - Tile::OY; ax = h % TX; ay = TY; az = (h / TX) % TZ; at = h / (TX * TZ); }
        else if (i < Tile::OT) { const int h = i - Tile::OZ; ax = h % TX; ay = h / TX % TY; az = TZ; at = h / (TX * TY); }
        else { const int h = i - Tile::OT; ax = h % TX; ay = (h / TX) % TY; az = h / (TX * TY); at = TT; }
        int gx = x0 + ax, gy = y0 + ay, gz = z0 + az, gt = t0 + at;
        if (gx >= g.L[0]) gx -= g.L[0];
        if (gy >= g.L[1]) gy -= g.L[1];
        if (gz >= g.L[2]) gz -= g.L[2];
        if (gt >= g.L[3]) gt -= g.L[3];
        Su3<T> gg;
        load_g(gg, D, g.V, gx + s1 * gy + s2 * gz + s3 * gt, half_alpha);
#pragma unroll
        for (int c = 0; c < 9; ++c) G[c * NG + i] = gg.m[c];
    }
    __syncthreads();
    // ---- U' = g(x) U g(x+mu)^+ ----
    int f;
    if (mu == 0) f = lx + 1 < TX ? ls + 1 : Tile::OX + ly + TY * (lz + TZ * lt);
    else if (mu == 1) f = ly + 1 < TY ? ls + TX : Tile::OY + lx + TX * (lz + TZ * lt);
    else if (mu == 2) f = lz + 1 < TZ ? ls + TX * TY : Tile::OZ + lx + TX * (ly + TY * lt);
    else f = lt + 1 < TT ? ls + TX * TY * TZ : Tile::OT + lx + TX * (ly + TY * lz);
    if (NC == 6) rebuild_row2(u);
    Cx<T> W[3 * NR];
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        const Cx<T> a0 = G[(3 * i) * NG + ls], a1 = G[(3 * i + 1) * NG + ls], a2 = G[(3 * i + 2) * NG + ls];
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            Cx<T> acc = a0 * u.m[j];
            fma_cx(acc, a1, u.m[3 + j]);
            fma_cx(acc, a2, u.m[6 + j]);
            W[3 * i + j] = acc;
        }
    }
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        const Cx<T> b0 = G[(3 * j) * NG + f], b1 = G[(3 * j + 1) * NG + f], b2 = G[(3 * j + 2) * NG + f];
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            Cx<T> acc = mulc(W[3 * i], b0);
            fma_cxc(acc, W[3 * i + 1], b1);
            fma_cxc(acc, W[3 * i + 2], b2);
            st_cx(p + (size_t)(3 * i + j) * g.V, acc);
        }
    }
}

}  // namespace lgf
