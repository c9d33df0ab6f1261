// lgf_site_fused.cuh -- K5 and K1 of consecutive iterations fused into one marching kernel
// (SURVEY.md §8(f) rank 1): the update kernel also emits Delta, theta and F of the NEW links, so the
// links are read once and written once per iteration (8 n_l + 16 reals per site instead of
// 12 n_l + 16) and K1 runs stand-alone only for the very first measurement.
//
//   U'_mu(x)  = g(x) U_mu(x) g(x+mu)^+                                   (north_star steps 4, 5)
//   Delta'(x) = sum_mu [ q_mu(x-mu) - q_mu(x) ],   q_mu(x) = P(U'_mu(x))  (north_star step 1)
// with P(M) = (M - M^+) - (1/3) Tr(M - M^+), packed like Delta (c0 = P01, c1 = P02, c2 = P12,
// c3 = Im P00 + i Im P11): the projection is linear, so it is taken per link and only its 8 reals
// travel between sites.
//
// Work decomposition.  A CTA owns a (x,y,z) tile of TX*TY*TZ sites (TX = Lx: the x direction wraps
// inside the tile) and MARCHES along t, one t-slice per step, over a contiguous range of the
// global slice sequence (column-major: tile column, then t), so that any grid size balances to
// within one slice.  Per step:
//   * g of the slice (built once per site, at the previous step) sits in shared memory, G[c][site];
//     the forward y/z halo g's are built by the face rows.  Matrix operands of the 3x3 products
//     are read from there, which keeps the register footprint at ~128.
//   * q_mu of the slice is exchanged through shared memory (Q[mu][c][site]); the backward y/z face
//     rows recompute their halo links U'_mu(x-mu) (owned by the neighbouring tile) from the OLD field;
//     the backward t neighbour is the thread's own previous step (registers).
// Because halo links are recomputed from the old field, the update is out of place: the links
// live in two buffers that swap roles every iteration (DevState::cur says which one is current).
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_site.cuh"

namespace lgf {

template <int TX_, int TY_, int TZ_>
struct MarchTile {
    static constexpr int TX = TX_, TY = TY_, TZ = TZ_;
    static constexpr int NS = TX * TY * TZ;          // sites per t-slice of the tile = threads
    static constexpr int HY = TX * TZ, HZ = TX * TY; // forward halo sites (y face, z face)
    static constexpr int NG = NS + HY + HZ;          // g slots
    template <typename T> static constexpr size_t smem_bytes() { return sizeof(Cx<T>) * (size_t)(9 * NG + 12 * NS); }
};

struct MarchGeom {
    int L[4];
    long long V;
    int nby, nbz;             // tiles along y, z
    long long nslices;        // nby * nbz * Lt
};

// q = P(u): packed anti-Hermitian traceless part of a 3x3 matrix (see header)
template <typename T>
__device__ __forceinline__ void project_ah(const Su3<T>& u, Cx<T> q[4]) {
    q[0] = u.m[1] - conj(u.m[3]);
    q[1] = u.m[2] - conj(u.m[6]);
    q[2] = u.m[5] - conj(u.m[7]);
    const T a0 = T(2) * u.m[0].im, a1 = T(2) * u.m[4].im, a2 = T(2) * u.m[8].im;
    const T tr3 = (a0 + a1 + a2) / T(3);
    q[3] = Cx<T>(a0 - tr3, a1 - tr3);
}

// out = A u B^+ with A, B read element-wise through accessors (shared memory or registers).
// Rows 0..NR-1 by products; NR = 2: row 2 = conj(row0 x row1) (12-real mode).
template <typename T, int NR, class FA, class FB>
__device__ __forceinline__ void sandwich(Su3<T>& out, const Su3<T>& u, FA&& A, FB&& B) {
    Cx<T> W[3 * NR];
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        const Cx<T> a0 = A(3 * i), a1 = A(3 * i + 1), a2 = A(3 * i + 2);
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
        const Cx<T> b0 = B(3 * j), b1 = B(3 * j + 1), b2 = B(3 * j + 2);
#pragma unroll
        for (int i = 0; i < NR; ++i) {
            Cx<T> acc = mulc(W[3 * i], b0);
            fma_cxc(acc, W[3 * i + 1], b1);
            fma_cxc(acc, W[3 * i + 2], b2);
            out.m[3 * i + j] = acc;
        }
    }
    if (NR == 2) rebuild_row2(out);
}

template <typename T, int NC>
__device__ __forceinline__ void store_link(const Su3<T>& u, Cx<T>* __restrict__ U, long long V, int mu, long long s) {
    Cx<T>* p = U + (size_t)mu * NC * V + s;
#pragma unroll
    for (int c = 0; c < NC; ++c) st_cx(p + (size_t)c * V, u.m[c]);
}

template <typename T, int NC> struct FusedOcc { static constexpr int value = 2; };

template <typename T, int NC, class Tile, int MINB>
__global__ void __launch_bounds__(Tile::NS, MINB)
k51_update_delta(const Cx<T>* __restrict__ U0, const Cx<T>* __restrict__ U1, const Cx<T>* __restrict__ Dt,
                 Cx<T>* __restrict__ Dout, double2* __restrict__ partials, const DevState* st, MarchGeom g, T ha) {
    extern __shared__ __align__(16) unsigned char fused_smem[];
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    constexpr int TX = Tile::TX, TY = Tile::TY, TZ = Tile::TZ, NS = Tile::NS, NG = Tile::NG, NR = NC / 3;
    Cx<T>* G = reinterpret_cast<Cx<T>*>(fused_smem);     // [9][NG]
    Cx<T>* Q = G + 9 * NG;                               // [3][4][NS]
    const int cur = *reinterpret_cast<const volatile int*>(&st->cur);
    const Cx<T>* __restrict__ Uin = cur ? U1 : U0;
    Cx<T>* __restrict__ Uout = const_cast<Cx<T>*>(cur ? U0 : U1);

    const int tid = threadIdx.x;
    const int lx = tid % TX, ly = (tid / TX) % TY, lz = tid / (TX * TY);
    const int Lx = g.L[0], Ly = g.L[1], Lz = g.L[2], Lt = g.L[3];
    const long long V = g.V, sy = Lx, sz = (long long)Lx * Ly, stt = sz * Lz;
    // in-tile neighbours (x always wraps inside the tile; y/z wrap inside only if the tile spans the axis)
    const bool wrap_y = (Ly == TY), wrap_z = (Lz == TZ);
    const int fx = tid - lx + (lx + 1 == TX ? 0 : lx + 1), bx = tid - lx + (lx == 0 ? TX - 1 : lx - 1);
    const bool fy_in = (ly + 1 < TY) || wrap_y, by_in = (ly > 0) || wrap_y;
    const bool fz_in = (lz + 1 < TZ) || wrap_z, bz_in = (lz > 0) || wrap_z;
    const int fy = fy_in ? (ly + 1 < TY ? tid + TX : tid - TX * (TY - 1)) : NS + lx + TX * lz;
    const int fz = fz_in ? (lz + 1 < TZ ? tid + TX * TY : tid - TX * TY * (TZ - 1)) : NS + Tile::HY + lx + TX * ly;
    const int by = ly > 0 ? tid - TX : tid + TX * (TY - 1);
    const int bz = lz > 0 ? tid - TX * TY : tid + TX * TY * (TZ - 1);

    // this CTA's contiguous range of the slice sequence (column-major: tile column, then t)
    const long long q0 = g.nslices * (long long)blockIdx.x / gridDim.x;
    const long long q1 = g.nslices * (long long)(blockIdx.x + 1) / gridDim.x;
    double th = 0.0, fn = 0.0;
    Cx<T> qtp[4];                       // q_t(x - t) carried from the previous step
    long long sxyz = 0, yf_off = 0, zf_off = 0, yb_off = 0, zb_off = 0;

    auto own_g = [&](int c) { return G[c * NG + tid]; };

    for (long long q = q0; q < q1; ++q) {
        const int col = (int)(q / Lt), t = (int)(q - (long long)col * Lt);
        if (q == q0 || t == 0) {
            // ---- new column (or first step): coordinates, g of the first slice, q_t of the slice behind ----
            const int tby = col % g.nby, tbz = col / g.nby;
            const int y = tby * TY + ly, z = tbz * TZ + lz;
            sxyz = lx + sy * y + sz * z;
            yf_off = (y + 1 == Ly) ? -(long long)(Ly - 1) * sy : sy;
            yb_off = (y == 0) ? (long long)(Ly - 1) * sy : -sy;
            zf_off = (z + 1 == Lz) ? -(long long)(Lz - 1) * sz : sz;
            zb_off = (z == 0) ? (long long)(Lz - 1) * sz : -sz;
            const long long s = sxyz + (long long)t * stt;
            const long long sb = s + (t == 0 ? (long long)(Lt - 1) * stt : -stt);
            Su3<T> g0, gb, u, un;
            load_g(g0, Dt, V, s, ha);
            load_g(gb, Dt, V, sb, ha);
            load_link<T, NC>(u, Uin, V, 3, sb);
            sandwich<T, NR>(un, u, [&](int c) { return gb.m[c]; }, [&](int c) { return g0.m[c]; });
            project_ah(un, qtp);
            __syncthreads();            // the previous column's last reads of G are done
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + tid] = g0.m[c];
        }
        const long long s = sxyz + (long long)t * stt;
        // ---- (1) forward halo g's of this slice, built by the face rows ----
        if (!fy_in) {
            Su3<T> gh;
            load_g(gh, Dt, V, s + yf_off, ha);
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + fy] = gh.m[c];
        }
        if (!fz_in) {
            Su3<T> gh;
            load_g(gh, Dt, V, s + zf_off, ha);
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + fz] = gh.m[c];
        }
        __syncthreads();                // (a) g of the slice and of its forward halo is in place
        Cx<T> acc[4] = {qtp[0], qtp[1], qtp[2], qtp[3]};
        T retr = 0;
        // ---- (2) links mu = x, y, z ----
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) {
            const int f = mu == 0 ? fx : (mu == 1 ? fy : fz);
            Su3<T> u, un;
            load_link<T, NC>(u, Uin, V, mu, s);
            sandwich<T, NR>(un, u, own_g, [&](int c) { return G[c * NG + f]; });
            store_link<T, NC>(un, Uout, V, mu, s);
            retr += un.m[0].re + un.m[4].re + un.m[8].re;
            Cx<T> qq[4];
            project_ah(un, qq);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                acc[c] = acc[c] - qq[c];
                Q[(mu * 4 + c) * NS + tid] = qq[c];
            }
        }
        __syncthreads();                // (b) q_mu of the slice is in place; nobody reads G's neighbours any more
        // ---- (3) backward contributions ----
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] = acc[c] + Q[(0 * 4 + c) * NS + bx];
        if (by_in) {
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] + Q[(1 * 4 + c) * NS + by];
        } else {
            Su3<T> gb, u, un;
            load_g(gb, Dt, V, s + yb_off, ha);
            load_link<T, NC>(u, Uin, V, 1, s + yb_off);
            sandwich<T, NR>(un, u, [&](int c) { return gb.m[c]; }, own_g);
            Cx<T> qq[4];
            project_ah(un, qq);
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] + qq[c];
        }
        if (bz_in) {
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] + Q[(2 * 4 + c) * NS + bz];
        } else {
            Su3<T> gb, u, un;
            load_g(gb, Dt, V, s + zb_off, ha);
            load_link<T, NC>(u, Uin, V, 2, s + zb_off);
            sandwich<T, NR>(un, u, [&](int c) { return gb.m[c]; }, own_g);
            Cx<T> qq[4];
            project_ah(un, qq);
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] + qq[c];
        }
        // ---- link mu = t: g(x+t) is built here and becomes the next step's g ----
        {
            const long long sf = s + (t == Lt - 1 ? -(long long)(Lt - 1) * stt : stt);
            Su3<T> gt, u, un;
            load_g(gt, Dt, V, sf, ha);
            load_link<T, NC>(u, Uin, V, 3, s);
            sandwich<T, NR>(un, u, own_g, [&](int c) { return gt.m[c]; });
            store_link<T, NC>(un, Uout, V, 3, s);
            retr += un.m[0].re + un.m[4].re + un.m[8].re;
            project_ah(un, qtp);
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] - qtp[c];
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + tid] = gt.m[c];     // own slot: read by others only after the next (a)
        }
        // ---- Delta', theta, F of the new links at this site ----
        st_cx(Dout + s, acc[0]);
        st_cx(Dout + (size_t)V + s, acc[1]);
        st_cx(Dout + (size_t)2 * V + s, acc[2]);
        st_cx(Dout + (size_t)3 * V + s, acc[3]);
        const T d2 = -(acc[3].re + acc[3].im);
        th += 2.0 * ((double)norm2(acc[0]) + (double)norm2(acc[1]) + (double)norm2(acc[2])) + (double)acc[3].re * acc[3].re +
              (double)acc[3].im * acc[3].im + (double)d2 * d2;
        fn += (double)retr;
    }
    block_sum2<NS>(th, fn);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fn);
}

}  // namespace lgf
