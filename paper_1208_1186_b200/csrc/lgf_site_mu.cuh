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
    __device__ static __forceinline__ bool coords(const Geom& g, int ls, int x[4]) {
        int b = blockIdx.x;
        const int bx = b % g.nb[0]; b /= g.nb[0];
        const int by = b % g.nb[1]; b /= g.nb[1];
        const int bz = b % g.nb[2]; b /= g.nb[2];
        const int bt = b;
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
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    constexpr int NS = Tile::kSites;
    const int ls = threadIdx.x % NS, mu = threadIdx.x / NS;
    int x[4];
    if (!Tile::coords(g, ls, x)) return;
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

}  // namespace lgf
