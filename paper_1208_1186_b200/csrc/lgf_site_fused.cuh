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

template <int TX_, int TY_, int TZ_, bool STAGE_ = false>
struct MarchTile {
    static constexpr int TX = TX_, TY = TY_, TZ = TZ_;
    // STAGE: every thread keeps the links and the Delta~ it needs at the NEXT step in flight as
    // cp.async copies into its own shared-memory slots (no registers, no barrier: a thread reads back
    // only what it copied itself), so global latency is off the critical path of the march.
    static constexpr bool kStage = STAGE_;
    static constexpr int NS = TX * TY * TZ;          // sites per t-slice of the tile = threads
    static constexpr int HY = TX * TZ, HZ = TX * TY; // halo sites of one y face / one z face
    static constexpr int NG = NS + HY + HZ;          // g slots: the slice + its forward y and z halo
    static constexpr int NH = HY + HZ;               // q slots of the backward halo links
    static constexpr bool kShflX = (TX == 32);       // a warp is one x row: q_x travels by shuffle
    static constexpr int NQ = kShflX ? 2 : 3;        // directions exchanged through shared memory
    template <typename T, int NC> static constexpr size_t smem_bytes() {
        return sizeof(Cx<T>) * (size_t)(9 * NG + 4 * NQ * NS + 4 * NH + (kStage ? (4 * NC + 4) * NS : 0));
    }
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


// shuffle a complex number from lane `src` of the warp
__device__ __forceinline__ Cx<double> shfl_cx(Cx<double> v, int src) {
    return Cx<double>(__shfl_sync(0xffffffffu, v.re, src), __shfl_sync(0xffffffffu, v.im, src));
}
__device__ __forceinline__ Cx<float> shfl_cx(Cx<float> v, int src) {
    return Cx<float>(__shfl_sync(0xffffffffu, v.re, src), __shfl_sync(0xffffffffu, v.im, src));
}
// per-thread asynchronous global -> shared copy of one complex number (LDGSTS), and its group fences
__device__ __forceinline__ void cp_async_cx(Cx<double>* dst, const Cx<double>* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_cx(Cx<float>* dst, const Cx<float>* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// pull the 128-byte line holding p towards L2 ahead of the next step's loads
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <typename T, int NC, class Tile, int MINB>
__global__ void __launch_bounds__(Tile::NS, MINB)
k51_update_delta(const Cx<T>* __restrict__ U0, const Cx<T>* __restrict__ U1, const Cx<T>* __restrict__ Dt,
                 Cx<T>* __restrict__ Dout, double2* __restrict__ partials, const DevState* st, MarchGeom g, T ha) {
    pdl_entry();
    extern __shared__ __align__(16) unsigned char fused_smem[];
    if (*reinterpret_cast<const volatile int*>(&st->done)) return;
    constexpr int TX = Tile::TX, TY = Tile::TY, TZ = Tile::TZ, NS = Tile::NS, NG = Tile::NG, NH = Tile::NH, NR = NC / 3;
    constexpr int HY = Tile::HY;
    constexpr bool SHX = Tile::kShflX;
    constexpr int QY = SHX ? 0 : 1, QZ = SHX ? 1 : 2;   // planes of Q holding q_y, q_z (q_x in plane 0 unless shuffled)
    Cx<T>* G = reinterpret_cast<Cx<T>*>(fused_smem);     // [9][NG]   g of the slice + forward halo
    Cx<T>* Q = G + 9 * NG;                               // [NQ][4][NS]  q_mu of the slice
    Cx<T>* QH = Q + 4 * Tile::NQ * NS;                   // [4][NH]   q of the backward halo links
    constexpr bool STG = Tile::kStage;
    Cx<T>* S = QH + 4 * NH;                              // [4*NC][NS] staged links of the step (STG)
    Cx<T>* SD = S + 4 * NC * NS;                         // [4][NS]    staged Delta~(x+t) of the step (STG)
    const int cur = *reinterpret_cast<const volatile int*>(&st->cur);
    const Cx<T>* __restrict__ Uin = cur ? U1 : U0;
    Cx<T>* __restrict__ Uout = const_cast<Cx<T>*>(cur ? U0 : U1);

    const int tid = threadIdx.x;
    const int lx = tid % TX, ly = (tid / TX) % TY, lz = tid / (TX * TY);
    const int Lx = g.L[0], Ly = g.L[1], Lz = g.L[2], Lt = g.L[3];
    const long long V = g.V, sy = Lx, sz = (long long)Lx * Ly, stt = sz * Lz;
    const bool wrap_y = (Ly == TY), wrap_z = (Lz == TZ);
    const int nhy = wrap_y ? 0 : HY, nh = nhy + (wrap_z ? 0 : Tile::HZ);     // halo items of this lattice
    const int fx = tid - lx + (lx + 1 == TX ? 0 : lx + 1), bx = tid - lx + (lx == 0 ? TX - 1 : lx - 1);
    const bool fy_in = (ly + 1 < TY) || wrap_y, by_in = (ly > 0) || wrap_y;
    const bool fz_in = (lz + 1 < TZ) || wrap_z, bz_in = (lz > 0) || wrap_z;
    const int fy = fy_in ? (ly + 1 < TY ? tid + TX : tid - TX * (TY - 1)) : NS + lx + TX * lz;
    const int fz = fz_in ? (lz + 1 < TZ ? tid + TX * TY : tid - TX * TY * (TZ - 1)) : NS + HY + lx + TX * ly;
    const int by = by_in ? (ly > 0 ? tid - TX : tid + TX * (TY - 1)) : lx + TX * lz;              // Q slot, or QH item
    const int bz = bz_in ? (lz > 0 ? tid - TX * TY : tid + TX * TY * (TZ - 1)) : nhy + lx + TX * ly;
    const long long sloc = lx + sy * ly + sz * lz;       // this thread's site relative to the tile origin
    const bool pf_lane = (lx % (int)(128 / sizeof(Cx<T>))) == 0;

    const long long q0 = g.nslices * (long long)blockIdx.x / gridDim.x;
    const long long q1 = g.nslices * (long long)(blockIdx.x + 1) / gridDim.x;
    double th = 0.0, fn = 0.0;
    Cx<T> qtp[4];                       // q_t(x - t), carried from the previous step
    long long s0 = 0, yf_off = 0, zf_off = 0, yb_off = 0, zb_off = 0;   // tile origin (t = 0) and face offsets

    auto own_g = [&](int c) { return G[c * NG + tid]; };
    // halo item h -> site offset (relative to the slice's tile origin) of a y-face / z-face position
    auto item_site = [&](int h, bool& is_y) -> long long {
        is_y = h < nhy;
        const int k = is_y ? h : h - nhy;
        const int a = k % TX, b = k / TX;
        return is_y ? a + sz * b : a + sy * b;
    };

    // STG: this thread's copies for slice index qq, batch b (0..2: link b; 3: link t and Delta~(x+t));
    // one commit per batch, also when there is nothing left to copy, so that the group count stays 4 per step
    auto stage_issue = [&](long long qq, int b) {
        if (qq < q1) {
            const int c2 = (int)(qq / Lt), t2 = (int)(qq - (long long)c2 * Lt);
            const long long sn = sy * ((c2 % g.nby) * TY) + sz * ((c2 / g.nby) * TZ) + sloc + (long long)t2 * stt;
#pragma unroll
            for (int c = 0; c < NC; ++c) cp_async_cx(S + (b * NC + c) * NS + tid, Uin + (size_t)(b * NC + c) * V + sn);
            if (b == 3) {
                const long long sfn = sn + (t2 == Lt - 1 ? -(long long)(Lt - 1) * stt : stt);
#pragma unroll
                for (int c = 0; c < 4; ++c) cp_async_cx(SD + c * NS + tid, Dt + (size_t)c * V + sfn);
            }
        }
        cp_async_commit();
    };
    auto staged_link = [&](Su3<T>& u, int b) {
#pragma unroll
        for (int c = 0; c < NC; ++c) u.m[c] = S[(b * NC + c) * NS + tid];
        if (NC == 6) rebuild_row2(u);
    };
    if (STG) {
#pragma unroll
        for (int b = 0; b < 4; ++b) stage_issue(q0, b);
    }

    for (long long q = q0; q < q1; ++q) {
        const int col = (int)(q / Lt), t = (int)(q - (long long)col * Lt);
        if (q == q0 || t == 0) {
            // ---- new column (or first step): tile origin, g of the first slice, q_t of the slice behind ----
            const int y0 = (col % g.nby) * TY, z0 = (col / g.nby) * TZ;
            s0 = sy * y0 + sz * z0;
            yf_off = (long long)((y0 + TY) % Ly - y0) * sy;
            yb_off = (long long)((y0 + Ly - 1) % Ly - y0) * sy;
            zf_off = (long long)((z0 + TZ) % Lz - z0) * sz;
            zb_off = (long long)((z0 + Lz - 1) % Lz - z0) * sz;
            const long long s = s0 + sloc + (long long)t * stt;
            const long long sb = s + (t == 0 ? (long long)(Lt - 1) * stt : -stt);
            Su3<T> g0, gb, u, un;
            load_g(g0, Dt, V, s, ha);
            load_g(gb, Dt, V, sb, ha);
            load_link<T, NC>(u, Uin, V, 3, sb);
            sandwich<T, NR>(un, u, [&](int c) { return gb.m[c]; }, [&](int c) { return g0.m[c]; });
            project_ah(un, qtp);
            __syncthreads();            // uniform branch; the previous column is completely done
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + tid] = g0.m[c];
        }
        const long long sbase = s0 + (long long)t * stt;
        const long long s = sbase + sloc;
        // ---- (1) forward halo g's of this slice, one item per thread ----
        for (int h = tid; h < nh; h += NS) {
            bool is_y;
            const long long hs = sbase + item_site(h, is_y) + (is_y ? yf_off : zf_off);
            Su3<T> gh;
            load_g(gh, Dt, V, hs, ha);
            const int slot = NS + (is_y ? h : HY + (h - nhy));
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + slot] = gh.m[c];
        }
        // next slice's lines towards L2 while this one is being worked on
        if (!STG && pf_lane && t + 1 < Lt) {
#pragma unroll
            for (int mu = 0; mu < 4; ++mu)
#pragma unroll
                for (int c = 0; c < NC; ++c) prefetch_l2(Uin + (size_t)(mu * NC + c) * V + s + stt);
            if (t + 2 < Lt) {
#pragma unroll
                for (int c = 0; c < 4; ++c) prefetch_l2(Dt + (size_t)c * V + s + 2 * stt);
            }
        }
        __syncthreads();                // (a) g of the slice and of its forward halo is in place
        Cx<T> acc[4] = {qtp[0], qtp[1], qtp[2], qtp[3]};
        T retr = 0;
        // ---- (2) links mu = x, y, z of this site ----
#pragma unroll
        for (int mu = 0; mu < 3; ++mu) {
            const int f = mu == 0 ? fx : (mu == 1 ? fy : fz);
            Su3<T> u, un;
            if (STG) {
                cp_async_wait<3>();                 // the batch issued one step ago has landed
                staged_link(u, mu);
                stage_issue(q + 1, mu);             // same slots, next slice
            } else {
                load_link<T, NC>(u, Uin, V, mu, s);
            }
            sandwich<T, NR>(un, u, own_g, [&](int c) { return G[c * NG + f]; });
            store_link<T, NC>(un, Uout, V, mu, s);
            retr += un.m[0].re + un.m[4].re + un.m[8].re;
            Cx<T> qq[4];
            project_ah(un, qq);
            if (SHX && mu == 0) {
                // the warp is this x row: q_x(x - 1) comes from the lane to the left (periodic)
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[c] = (acc[c] - qq[c]) + shfl_cx(qq[c], (lx + 31) & 31);
            } else {
                const int plane = mu == 0 ? 0 : (mu == 1 ? QY : QZ);
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    acc[c] = acc[c] - qq[c];
                    Q[(plane * 4 + c) * NS + tid] = qq[c];
                }
            }
        }
        // ---- backward halo links (owned by the neighbouring tiles), one item per thread ----
        for (int h = tid; h < nh; h += NS) {
            bool is_y;
            const long long loc = item_site(h, is_y);
            const long long hs = sbase + loc + (is_y ? yb_off : zb_off);
            // the face site this link ends on: (a, 0, b) for a y item, (a, b, 0) for a z item
            const int k = is_y ? h : h - nhy;
            const int ts = is_y ? (k % TX) + TX * TY * (k / TX) : k;
            Su3<T> gb, u, un;
            load_g(gb, Dt, V, hs, ha);
            load_link<T, NC>(u, Uin, V, is_y ? 1 : 2, hs);
            sandwich<T, NR>(un, u, [&](int c) { return gb.m[c]; }, [&](int c) { return G[c * NG + ts]; });
            Cx<T> qq[4];
            project_ah(un, qq);
#pragma unroll
            for (int c = 0; c < 4; ++c) QH[c * NH + h] = qq[c];
        }
        __syncthreads();                // (b) q_mu of the slice and of the halo links is in place
        // ---- (3) backward contributions, then the t link ----
        if (!SHX) {
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] + Q[(0 * 4 + c) * NS + bx];
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] = acc[c] + (by_in ? Q[(QY * 4 + c) * NS + by] : QH[c * NH + by]);
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] = acc[c] + (bz_in ? Q[(QZ * 4 + c) * NS + bz] : QH[c * NH + bz]);
        {
            // g(x+t) is built here and becomes the next step's g
            const long long sf = s + (t == Lt - 1 ? -(long long)(Lt - 1) * stt : stt);
            Su3<T> gt, u, un;
            if (STG) {
                cp_async_wait<3>();
                build_g(gt, SD[tid], SD[NS + tid], SD[2 * NS + tid], SD[3 * NS + tid], ha);
                staged_link(u, 3);
                stage_issue(q + 1, 3);
            } else {
                load_g(gt, Dt, V, sf, ha);
                load_link<T, NC>(u, Uin, V, 3, s);
            }
            sandwich<T, NR>(un, u, own_g, [&](int c) { return gt.m[c]; });
            store_link<T, NC>(un, Uout, V, 3, s);
            retr += un.m[0].re + un.m[4].re + un.m[8].re;
            project_ah(un, qtp);
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = acc[c] - qtp[c];
#pragma unroll
            for (int c = 0; c < 9; ++c) G[c * NG + tid] = gt.m[c];     // own slot: others read it only after the next (a)
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
