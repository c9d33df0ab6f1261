// lgf_fft_pipe.cuh -- persistent, asynchronously fed versions of the compile-time-sized FFT passes
// (K2, K3, K4 of SURVEY.md §8(a)); the default path when a lattice's extents are instantiated.
//
// One CTA per SM loops over its tiles.  A tile is fetched into shared memory by the TMA unit
// (cp.async.bulk row copies completing on an mbarrier) while the CTA's threads are still
// transforming earlier tiles: NG groups of GT threads each own one tile at a time, NBUF >= NG tile
// buffers form a ring, and the group that has finished tile i re-arms its buffer for tile i + NBUF.
// Global memory latency is therefore taken off the critical path of every tile but the first NBUF.
//
// To make K3's tiles contiguous in memory (one tile = one dense block instead of Lz*Lt scattered
// CX-site chunks), the spectrum travels between the kernels in two layouts:
//   natural   D[c][t][z][y][x]                       (K1 -> K2 input, K3 output -> K4 -> K5)
//   layout B  D'[c][chunk][t][z + pad][j], (y,x) position q = chunk*CXB + j   (K2 output -> K3 input;
//             one pad z-entry per t row, so that a tile is stored exactly as it sits in shared memory
//             and arrives with ONE bulk copy; bulk copies cost ~55 cycles each in the SM's TMA unit)
// K2 scatters CXB-site chunks into layout B, K3 scatters them back; the reads of all three kernels
// are dense.  K2 and K3 are out of place (two Delta-sized buffers ping-pong), K4 is in place.
// The in-register line transforms and the digit-swapped spectrum order are those of lgf_fft_ct.cuh.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_async.cuh"
#include "lgf_fft_ct.cuh"

namespace lgf {

// num / den (den > 0, both in the normal range).  fp64: reciprocal seed (~20 bits) + two Newton steps,
// then one residual correction of the quotient, which reproduces the correctly rounded IEEE quotient
// (so the scale factors agree bit for bit with a plain division) in ~9 instructions instead of the
// ~25 of the generic division sequence with its range checks.
__device__ __forceinline__ float fast_div(float num, float den) { return __fdividef(num, den); }
__device__ __forceinline__ double fast_div(double num, double den) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(den));
    r = fma(fma(-den, r, 1.0), r, r);
    r = fma(fma(-den, r, 1.0), r, r);
    const double q = num * r;
    return fma(fma(-den, q, num), r, q);
}

template <int GT, int NG>
__device__ __forceinline__ void group_sync(int g) {
    if (NG == 1) __syncthreads();
    else named_bar_sync(1 + g, GT);
}

struct XyPipeArgs {
    const void* twx_fwd; const void* twx_inv;
    const void* twy_fwd; const void* twy_inv;
    int nplanes;            // 4 * Lz * Lt
    int planes_per_comp;    // Lz * Lt
    int nz;                 // Lz
    int cxb_shift;          // layout-B chunk = 1 << cxb_shift sites (K3's CX)
    int chunks_per_comp;    // Lx * Ly >> cxb_shift
    int pt;                 // layout-B t pitch in elements: CX * (Lz + 1)
    int tile_elems;         // layout-B tile size in elements: pt * Lt
    // order of the t rows inside a layout-B tile: with t = n2 + perm_d * m (n2 < perm_d, m < perm_c) and n2 = perm_lq * q + l,
    // row rho(t) = (q * perm_c + m) * perm_lq + l.  perm_c = 1, perm_d = perm_lq = Lt is the natural order; the quarter-ring
    // K3 of lgf_fft_pipe3.cuh asks for the (C, D) split of its t lines with perm_lq = D / 4.
    int perm_c, perm_d, perm_lq;
    int store_tiles, nstores;   // fft_xy_pipe_io's tensor stores: layout-B tiles per store (box extent, <= 256), stores per plane
};

// Shared-memory planes are dense (one bulk copy per tile); bank conflicts of the passes that walk
// along y are removed by an XOR swizzle of the column index with the low bits of the row index,
// applied from the first stage's write-back on:  element (row, col) lives at row*NX + (col ^ (row & mask)).
template <typename T, int NX> struct XySwz {
    static constexpr int kSlots = (int)(128 / sizeof(Cx<T>));          // elements per 128 bytes
    static constexpr int mask = (NX < kSlots ? NX : kSlots) - 1;
};

// v[k] *= exp(SIGN 2 pi i r k / N) for k = 1..NK-1; r in [0, NR) is a run-time value that is uniform across the warp at
// every call site (the branches below do not diverge); the factors are compile-time literals.
template <int N, int NK, int NR, int SIGN, typename T>
__device__ __forceinline__ void tw_rows(Cx<T>* v, int r) {
    static_for<1, NR>([&](auto rr) {
        if (r == rr.value) static_for<1, NK>([&](auto k) { v[k.value] = mul_tw<rr.value * k.value, N, SIGN, T>(v[k.value]); });
    });
}

// K2 in THREE register stages per plane instead of four (the structure of lgf_fft_pipe3.cuh's K3, here for the (x,y)
// plane): with y lines split N_y = A*B (A first, 12 or 16) and x lines N_x = C*D (C = 4 first, D = 12 or 16)
//   P1  thread (x, n2y):    DFT_A over m of rows n2y + B m, times w_Ny^{-n2y k1y}        (lanes along x; dense in, swizzled out)
//   P2  thread (n2x, k1y):  DFT_B over the rows k1y*B + j, then DFT_C over the columns n2x + D m   (a B x C block; lanes along x)
//   P3  thread (y, k1x):    times w_Nx^{-j k1x}, DFT_D over the columns k1x*D + j         (lanes along y)
// The spectrum is left in the digit-swapped order of LineSplit<Ny, A> / LineSplit<Nx, C>; K4 inverts it with its
// two-stage passes on the same splits.  P1's output columns are another lane's input columns: a warp-level barrier
// separates its loads from its stores (the swizzle permutes inside aligned 8- or 16-element groups: inside a warp).
template <typename T, class SX, class SY, int PB, int GT, int NG>
__device__ __forceinline__ void xy3_forward_passes(Cx<T>* tile, int g, int gtid) {
    constexpr int NX = SX::kN, NY = SY::kN, PLANE = NX * NY, SW = XySwz<T, NX>::mask;
    constexpr int A = SY::kN1, B = SY::kN2, C = SX::kN1, D = SX::kN2;
    static_assert(B > 1 && D > 1 && B * C <= 16, "three-stage K2: the middle block must fit the registers");
    static_assert((PB * NX * B) % 32 == 0, "P1 must fill whole warps (its lanes exchange positions)");
    for (int it = gtid; it < PB * NX * B; it += GT) {
        const int x = it % NX, n2 = (it / NX) % B, pl = it / (NX * B);
        Cx<T>* s = tile + pl * PLANE;
        Cx<T> v[A];
        static_for<0, A>([&](auto m) { v[m.value] = s[(n2 + B * m.value) * NX + x]; });
        __syncwarp();
        RegFft<A, -1, T>::run(v);
        tw_rows<NY, A, B, -1, T>(v, n2);
        static_for<0, A>([&](auto k1) { constexpr int r0 = k1.value * B; const int r = r0 + n2; s[r * NX + (x ^ (r & SW))] = v[k1.value]; });
    }
    named_bar_sync(1 + g, GT);
    for (int it = gtid; it < PB * D * A; it += GT) {
        const int n2x = it % D, k1y = (it / D) % A, pl = it / (D * A);
        Cx<T>* s = tile + pl * PLANE + k1y * B * NX;
        Cx<T> e[C][B];
        static_for<0, C>([&](auto m) {
            static_for<0, B>([&](auto j) { e[m.value][j.value] = s[j.value * NX + ((n2x + D * m.value) ^ ((k1y * B + j.value) & SW))]; });
            RegFft<B, -1, T>::run(e[m.value]);
        });
        static_for<0, B>([&](auto j) {
            Cx<T> u[C];
            static_for<0, C>([&](auto m) { u[m.value] = e[m.value][j.value]; });
            RegFft<C, -1, T>::run(u);
            static_for<0, C>([&](auto k1x) { s[j.value * NX + ((k1x.value * D + n2x) ^ ((k1y * B + j.value) & SW))] = u[k1x.value]; });
        });
    }
    named_bar_sync(1 + g, GT);
    for (int it = gtid; it < PB * NY * C; it += GT) {
        const int y = it % NY, k1x = (it / NY) % C, pl = it / (NY * C);
        Cx<T>* s = tile + pl * PLANE + y * NX;
        const int sw = y & SW;
        Cx<T> v[D];
        static_for<0, D>([&](auto j) { v[j.value] = s[(k1x * D + j.value) ^ sw]; });
        tw_rows<NX, D, C, -1, T>(v, k1x);
        RegFft<D, -1, T>::run(v);
        static_for<0, D>([&](auto j) { s[(k1x * D + j.value) ^ sw] = v[j.value]; });
    }
    named_bar_sync(1 + g, GT);
}

// K2 (SIGN = -1: natural in -> layout B out) / K4 (SIGN = +1: natural in -> natural out, in place
// allowed); tile = PB contiguous (x,y) planes.
template <typename T, class SX, class SY, int SIGN, int PB, int GT, int NG, int NBUF, bool THREE = false>
__global__ void __launch_bounds__(GT * NG, 1)
fft_xy_pipe(const Cx<T>* in, Cx<T>* out, const XyPipeArgs A, const int* done) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    constexpr int NX = SX::kN, NY = SY::kN, PLANE = NX * NY, TILE = PB * PLANE, SW = XySwz<T, NX>::mask;
    static_assert((PLANE * sizeof(Cx<T>)) % 128 == 0, "bulk copy alignment");
    static_assert(NBUF >= NG && GT % 32 == 0 && NX % 8 == 0, "ring");
    // the swizzling first stage exchanges positions between lanes of one warp: whole warps only
    static_assert((PB * NX * SY::kN2) % 32 == 0 && (PB * NX * SY::kN1) % 32 == 0, "first stage must fill whole warps");
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(pipe_smem + sizeof(Cx<T>) * (size_t)NBUF * TILE);
    const int tid = threadIdx.x, g = tid / GT, gtid = tid - g * GT;
    const int ntiles = (A.nplanes + PB - 1) / PB;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const Cx<T>* twx = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twx_fwd : A.twx_inv);
    const Cx<T>* twy = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twy_fwd : A.twy_inv);

    // one thread arms buffer i % NBUF for this CTA's i-th tile: the planes of a tile are contiguous
    auto issue = [&](int i) {
        const int buf = i % NBUF;
        const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
        const int nvalid = min(PB, A.nplanes - plane0);
        const uint32_t bytes = (uint32_t)(nvalid * PLANE * sizeof(Cx<T>));
        mbar_arrive_expect_tx(&full[buf], bytes);
        bulk_g2s(bufs + (size_t)buf * TILE, in + (size_t)plane0 * PLANE, bytes, &full[buf]);
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
        const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
        const int nvalid = min(PB, A.nplanes - plane0);
        mbar_wait(&full[buf], (uint32_t)((i / NBUF) & 1));
        // (planes past nvalid hold stale data: they are transformed like the others, never stored)

        if constexpr (SIGN < 0 && THREE) {
            xy3_forward_passes<T, SX, SY, PB, GT, NG>(tile, g, gtid);
        } else if (SIGN < 0) {
            // ---- y axis: A (threads along x; dense in, swizzled out), B ----
            for (int it = gtid; it < PB * NX * SY::kN2; it += GT) {
                const int x = it % NX, n2 = (it / NX) % SY::kN2, pl = it / (NX * SY::kN2);
                Cx<T>* s = tile + pl * PLANE;
                stage_A_fwd<T, SY, 1>(n2, twy, [&](int p) { return s[p * NX + x]; },
                                      [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; });
            }
            group_sync<GT, NG>(g);
            if constexpr (SY::kN2 > 1) {
                for (int it = gtid; it < PB * NX * SY::kN1; it += GT) {
                    const int x = it % NX, k1 = (it / NX) % SY::kN1, pl = it / (NX * SY::kN1);
                    Cx<T>* s = tile + pl * PLANE;
                    stage_B<T, SY, 1, 0>(k1, twy, [&](int p) { return s[p * NX + (x ^ (p & SW))]; },
                                         [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; }, NoScale());
                }
                group_sync<GT, NG>(g);
            }
        } else {
            // ---- inverse y: B', A' (the first of them dense in, swizzled out) ----
            if constexpr (SY::kN2 > 1) {
                for (int it = gtid; it < PB * NX * SY::kN1; it += GT) {
                    const int x = it % NX, k1 = (it / NX) % SY::kN1, pl = it / (NX * SY::kN1);
                    Cx<T>* s = tile + pl * PLANE;
                    stage_B<T, SY, 0, 1, 1>(k1, twy, [&](int p) { return s[p * NX + x]; },
                                            [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; }, NoScale());
                }
                group_sync<GT, NG>(g);
                for (int it = gtid; it < PB * NX * SY::kN2; it += GT) {
                    const int x = it % NX, n2 = (it / NX) % SY::kN2, pl = it / (NX * SY::kN2);
                    Cx<T>* s = tile + pl * PLANE;
                    stage_A_inv<T, SY>(n2, [&](int p) { return s[p * NX + (x ^ (p & SW))]; },
                                       [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; });
                }
            } else {
                for (int it = gtid; it < PB * NX; it += GT) {
                    const int x = it % NX, pl = it / NX;
                    Cx<T>* s = tile + pl * PLANE;
                    stage_A_inv<T, SY, 1>(0, [&](int p) { return s[p * NX + x]; },
                                          [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; });
                }
            }
            group_sync<GT, NG>(g);
        }
        // ---- x axis (threads along y; every position swizzled by the row's low bits) ----
        if (SIGN < 0) {
            if constexpr (!THREE) {
                for (int it = gtid; it < PB * NY * SX::kN2; it += GT) {
                    const int y = it % NY, n2 = (it / NY) % SX::kN2, pl = it / (NY * SX::kN2);
                    Cx<T>* s = tile + pl * PLANE + y * NX;
                    const int sw = y & SW;
                    stage_A_fwd<T, SX>(n2, twx, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; });
                }
                group_sync<GT, NG>(g);
                if constexpr (SX::kN2 > 1) {
                    for (int it = gtid; it < PB * NY * SX::kN1; it += GT) {
                        const int y = it % NY, k1 = (it / NY) % SX::kN1, pl = it / (NY * SX::kN1);
                        Cx<T>* s = tile + pl * PLANE + y * NX;
                        const int sw = y & SW;
                        stage_B<T, SX, 1, 0>(k1, twx, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; }, NoScale());
                    }
                    group_sync<GT, NG>(g);
                }
            }
            // ---- scatter CXB-site chunks into layout B (its tiles are stored padded, as K3 wants them in smem) ----
            const int cxb_mask = (1 << A.cxb_shift) - 1;
            for (int pl = 0; pl < nvalid; ++pl) {
                const int gp = plane0 + pl;
                const int comp = gp / A.planes_per_comp, zt = gp - comp * A.planes_per_comp;
                const int t = zt / A.nz, z = zt - t * A.nz;
                const int tm = t / A.perm_d, tn = t - tm * A.perm_d, tq = tn / A.perm_lq;
                const int rho = (tq * A.perm_c + tm) * A.perm_lq + (tn - tq * A.perm_lq);
                Cx<T>* dbase = out + (size_t)comp * A.chunks_per_comp * A.tile_elems + (size_t)rho * A.pt + ((size_t)z << A.cxb_shift);
                const Cx<T>* sp = tile + pl * PLANE;
#pragma unroll 4
                for (int q = gtid; q < PLANE; q += GT) {
                    const int x = q % NX, y = q / NX;
                    st_cx(dbase + (size_t)(q >> A.cxb_shift) * A.tile_elems + (q & cxb_mask), sp[y * NX + (x ^ (y & SW))]);
                }
            }
        } else {
            if constexpr (SX::kN2 > 1) {
                for (int it = gtid; it < PB * NY * SX::kN1; it += GT) {
                    const int y = it % NY, k1 = (it / NY) % SX::kN1, pl = it / (NY * SX::kN1);
                    Cx<T>* s = tile + pl * PLANE + y * NX;
                    const int sw = y & SW;
                    stage_B<T, SX, 0, 1>(k1, twx, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; }, NoScale());
                }
                group_sync<GT, NG>(g);
            }
            for (int it = gtid; it < PB * NY * SX::kN2; it += GT) {
                const int y = it % NY, n2 = (it / NY) % SX::kN2, pl = it / (NY * SX::kN2);
                Cx<T>* s = tile + pl * PLANE + y * NX;
                const int sw = y & SW;
                stage_A_inv<T, SX>(n2, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; });
            }
            group_sync<GT, NG>(g);
            // ---- coalesced copy-out, natural layout ----
            Cx<T>* base = out + (size_t)plane0 * PLANE;
            const uint64_t keep = l2_evict_last_policy();      // Delta~ is K5's next read
#pragma unroll 4
            for (int e = gtid; e < nvalid * PLANE; e += GT) {
                const int x = e % NX, y = (e / NX) % NY, pl = e / PLANE;
                st_cx_keep(base + e, tile[pl * PLANE + y * NX + (x ^ (y & SW))], keep);
            }
        }
        // ---- hand the buffer back to the TMA unit for tile i + NBUF ----
        fence_proxy_async();
        group_sync<GT, NG>(g);
        if (i + NBUF < my_tiles && gtid == 0) issue(i + NBUF);
    }
}

// K3: layout B in -> forward z, forward t, scale by p2max/(V p2(k)), inverse t, inverse z -> natural out.
// Tile = CX contiguous (x,y) positions x the whole (z,t) plane of one component.
template <typename T, class SZ, class ST_, int CX, int GT, int NG, int NBUF>
__global__ void __launch_bounds__(GT * NG, 1)
fft_zt_pipe(const Cx<T>* inB, Cx<T>* out, const ZtArgs A, const int* done) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    constexpr int NZ = SZ::kN, NT = ST_::kN, PZ = CX, PT = CX * (NZ + 1), TILE = PT * NT;
    static_assert((TILE * sizeof(Cx<T>)) % 16 == 0, "bulk copy alignment");
    static_assert(NBUF >= NG && GT % 32 == 0, "ring");
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(pipe_smem + sizeof(Cx<T>) * (size_t)NBUF * TILE);
    const int tid = threadIdx.x, g = tid / GT, gtid = tid - g * GT;
    const int ntiles = 4 * A.nbatch * A.tiles_per_comp;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const long long gz = A.LxLy, gt = A.LxLy * NZ;
    const Cx<T>* twz_f = reinterpret_cast<const Cx<T>*>(A.twz_fwd);
    const Cx<T>* twz_i = reinterpret_cast<const Cx<T>*>(A.twz_inv);
    const Cx<T>* twt_f = reinterpret_cast<const Cx<T>*>(A.twt_fwd);
    const Cx<T>* twt_i = reinterpret_cast<const Cx<T>*>(A.twt_inv);

    // one thread arms buffer i % NBUF: layout-B tiles are stored padded exactly as they sit in shared memory
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
        const int id = (int)blockIdx.x + i * (int)gridDim.x;
        const int comp = id / A.tiles_per_comp;
        const int tidx = id - comp * A.tiles_per_comp;
        const long long tile_off = (long long)tidx * CX;
        Cx<T>* base = out + (size_t)comp * A.V + tile_off;
        mbar_wait(&full[buf], (uint32_t)((i / NBUF) & 1));

        // ---- z forward: A, B (in shared memory) ----
        for (int it = gtid; it < CX * NT * SZ::kN2; it += GT) {
            const int cx = it % CX, t = (it / CX) % NT, n2 = it / (CX * NT);
            Cx<T>* s = tile + cx + t * PT;
            stage_A_fwd<T, SZ>(n2, twz_f, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { s[p * PZ] = v; });
        }
        group_sync<GT, NG>(g);
        if constexpr (SZ::kN2 > 1) {
            for (int it = gtid; it < CX * NT * SZ::kN1; it += GT) {
                const int cx = it % CX, t = (it / CX) % NT, k1 = it / (CX * NT);
                Cx<T>* s = tile + cx + t * PT;
                stage_B<T, SZ, 1, 0>(k1, twz_i, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { s[p * PZ] = v; }, NoScale());
            }
            group_sync<GT, NG>(g);
        }
        // ---- t: forward, scale, inverse ----
        {
            constexpr int NLT = CX * NZ;
            auto line_momentum = [&](int cx, int zp, T& pxyz, bool& zero_xyz) {
                const long long sxy = tile_off + cx;
                const int ypos = int(sxy / A.Lx), xpos = int(sxy - (long long)ypos * A.Lx);
                const int kx = (xpos / A.x_n2) + A.x_n1 * (xpos % A.x_n2), ky = (ypos / A.y_n2) + A.y_n1 * (ypos % A.y_n2);
                const int kz = SZ::freq_of_pos(zp);
                pxyz = reinterpret_cast<const T*>(A.psq_x)[kx] + reinterpret_cast<const T*>(A.psq_y)[ky] +
                       reinterpret_cast<const T*>(A.psq_z)[kz];
                zero_xyz = (kx | ky | kz) == 0;
            };
            const T* pt = reinterpret_cast<const T*>(A.psq_t);
            const T num = (T)A.scale_num;
            if constexpr (ST_::kN2 > 1) {
                for (int it = gtid; it < NLT * ST_::kN2; it += GT) {
                    const int cx = it % CX, zp = (it / CX) % NZ, n2 = it / NLT;
                    Cx<T>* s = tile + cx + zp * PZ;
                    stage_A_fwd<T, ST_>(n2, twt_f, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; });
                }
                group_sync<GT, NG>(g);
                for (int it = gtid; it < NLT * ST_::kN1; it += GT) {
                    const int cx = it % CX, zp = (it / CX) % NZ, k1 = it / NLT;
                    Cx<T>* s = tile + cx + zp * PZ;
                    T pxyz; bool zero_xyz;
                    line_momentum(cx, zp, pxyz, zero_xyz);
                    auto scale = [&](int k2) -> T {
                        const int kt = k1 + ST_::kN1 * k2;
                        const T den = pxyz + __ldg(pt + kt);
                        return (zero_xyz && kt == 0) ? T(0) : fast_div(num, den);
                    };
                    stage_B<T, ST_, 1, 1>(k1, twt_i, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; }, scale);
                }
                group_sync<GT, NG>(g);
                for (int it = gtid; it < NLT * ST_::kN2; it += GT) {
                    const int cx = it % CX, zp = (it / CX) % NZ, n2 = it / NLT;
                    Cx<T>* s = tile + cx + zp * PZ;
                    stage_A_inv<T, ST_>(n2, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; });
                }
                group_sync<GT, NG>(g);
            } else {
                for (int it = gtid; it < NLT; it += GT) {
                    const int cx = it % CX, zp = it / CX;
                    Cx<T>* s = tile + cx + zp * PZ;
                    T pxyz; bool zero_xyz;
                    line_momentum(cx, zp, pxyz, zero_xyz);
                    Cx<T> v[NT];
                    static_for<0, NT>([&](auto m) { v[m.value] = s[m.value * PT]; });
                    RegFft<NT, -1, T>::run(v);
                    // p^2 is even in k_t: one quotient scales modes k_t and N_t - k_t
                    static_for<0, NT / 2 + 1>([&](auto kt) {
                        constexpr int k = kt.value;
                        const T den = pxyz + psq_t_half(A, k, T());
                        const T sc = (zero_xyz && k == 0) ? T(0) : fast_div(num, den);
                        v[k] = sc * v[k];
                        if constexpr (k != 0 && 2 * k != NT) v[NT - k] = sc * v[NT - k];
                    });
                    RegFft<NT, +1, T>::run(v);
                    static_for<0, NT>([&](auto m) { s[m.value * PT] = v[m.value]; });
                }
                group_sync<GT, NG>(g);
            }
        }
        // ---- z inverse: B' in shared memory, A' straight to global (natural layout) ----
        if constexpr (SZ::kN2 > 1) {
            for (int it = gtid; it < CX * NT * SZ::kN1; it += GT) {
                const int cx = it % CX, t = (it / CX) % NT, k1 = it / (CX * NT);
                Cx<T>* s = tile + cx + t * PT;
                stage_B<T, SZ, 0, 1>(k1, twz_i, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { s[p * PZ] = v; }, NoScale());
            }
            group_sync<GT, NG>(g);
        }
        for (int it = gtid; it < CX * NT * SZ::kN2; it += GT) {
            const int cx = it % CX, t = (it / CX) % NT, n2 = it / (CX * NT);
            Cx<T>* gp = base + cx + (size_t)t * gt;
            const Cx<T>* s = tile + cx + t * PT;
            stage_A_inv<T, SZ>(n2, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { st_cx(gp + (size_t)p * gz, v); });
        }
        fence_proxy_async();
        group_sync<GT, NG>(g);
        if (i + NBUF < my_tiles && gtid == 0) issue(i + NBUF);
    }
}

}  // namespace lgf
