// lgf_fft_pipe_io.cuh -- K2 / K4 asynchronously fed AND drained: the variant of fft_xy_pipe
// (lgf_fft_pipe.cuh) whose output leaves through the TMA unit.  Used where the output chunks are small and the field
// lives in HBM (64 x 64 planes: 32-byte chunks of layout B); on L2-resident lattices (32^4, 48^3 x 8) the extra
// un-swizzle pass and the store -> drain -> re-fetch chain of the I/O lane cost more than the per-thread scatter
// (measured: K2 25.8 -> 32.2 us at 32^4 fp64, 660 -> 500 us at 64^4 fp64).
//
// One CTA per SM loops over its tiles.  NG groups of GT compute threads each own one tile at a time; NBUF >= NG + 1
// tile buffers form a ring; ONE extra warp (the I/O warp, one active lane) owns every asynchronous copy:
//   fetch   a tile arrives through one cp.async.bulk (TMA unit, SASS UBLKCP) completing on the mbarrier full[buf];
//   drain   a group that has finished a tile leaves its OUTPUT in the tile buffer (dense, un-swizzled) and arrives on
//           done[buf]; the I/O lane then stores it with the TMA unit -- a TENSOR store (cp.async.bulk.tensor, SASS UTMASTG)
//           where the output is a scatter (K2 into layout B, K3 into the natural layout), one bulk copy where it is
//           contiguous (K4) -- waits until the store has read the buffer (bulk wait_group.read) and re-arms it.
// Why the TMA unit stores: a microbenchmark of K3's output pattern on B200 (1.07 GB in chunks of CX sites x 16 B, 64 KB
// apart) wrote 1.17 / 2.3 / 4.7 TB/s with per-thread stores at 32 / 64 / 128-byte chunks (the SM's store path takes one
// 128-byte-line request every ~6 cycles, full or not) against 3.8 / 4.8 / 5.3 TB/s through tensor stores with the same
// chunks as the innermost box dimension, and 6.1 TB/s dense.  ncu had shown the per-thread scatter as the top stall
// (stall_lg) of K3 at 64^4.
//
// To make K3's tiles contiguous in memory (one tile = one dense block instead of Lz*Lt scattered CX-site chunks), the
// spectrum travels between the kernels in two layouts:
//   natural   D[c][t][z][y][x]                       (K1 -> K2 input, K3 output -> K4 -> K5)
//   layout B  D'[c][chunk][t][z + pad][j], (y,x) position q = chunk*CXB + j   (K2 output -> K3 input;
//             one pad z-entry per t row, so that a tile is stored exactly as it sits in shared memory
//             and arrives with ONE bulk copy; bulk copies cost ~55 cycles each in the SM's TMA unit)
// K2 and K3 are out of place (two Delta-sized buffers ping-pong), K4 is in place.
// The in-register line transforms and the digit-swapped spectrum order are those of lgf_fft_ct.cuh.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cuda.h>

#include "lgf_fft_pipe.cuh"

namespace lgf {

// The I/O lane's loop, shared by the ring kernels: fetch the first NBUF tiles, then for every tile of this CTA in order
// wait until its group is done with it, store it (STORE(i, buffer index)), wait until the store has read the buffer and
// fetch tile i + NBUF into it.  FETCH(i) arms full[i % NBUF] and issues the bulk copy.
template <int NBUF, class FETCH, class STORE>
__device__ __forceinline__ void io_lane_loop(int my_tiles, uint64_t* done, FETCH&& fetch, STORE&& store) {
    for (int i = 0; i < NBUF && i < my_tiles; ++i) fetch(i);
    for (int i = 0; i < my_tiles; ++i) {
        mbar_wait(&done[i % NBUF], (uint32_t)((i / NBUF) & 1));
        store(i, i % NBUF);
        bulk_commit_group();
        bulk_wait_group_read<0>();
        if (i + NBUF < my_tiles) fetch(i + NBUF);
    }
    bulk_wait_group<0>();          // the last stores' global writes are performed before the CTA exits
}

// K2 (SIGN = -1: natural in -> layout B out) / K4 (SIGN = +1: natural in -> natural out, in place
// allowed); tile = PB contiguous (x,y) planes.
// `bmap`: CUtensorMap of layout B as the 4-D tensor (2 reals x CXB sites, z, t row, tile) -- used by K2 only.
template <typename T, class SX, class SY, int SIGN, int PB, int GT, int NG, int NBUF, bool THREE = false>
__global__ void __launch_bounds__(GT * NG + 32, 1)
fft_xy_pipe_io(const Cx<T>* in, Cx<T>* out, const __grid_constant__ XyPipeArgs A, const int* done_flag,
            const __grid_constant__ CUtensorMap bmap) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done_flag && *reinterpret_cast<const volatile int*>(done_flag)) return;
    constexpr int NX = SX::kN, NY = SY::kN, PLANE = NX * NY, TILE = PB * PLANE, SW = XySwz<T, NX>::mask;
    static_assert((PLANE * sizeof(Cx<T>)) % 128 == 0, "bulk copy alignment");
    static_assert(NBUF > NG && GT % 32 == 0 && NX % 8 == 0, "ring");
    // the swizzling first stage exchanges positions between lanes of one warp: whole warps only
    static_assert((PB * NX * SY::kN2) % 32 == 0 && (PB * NX * SY::kN1) % 32 == 0, "first stage must fill whole warps");
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(pipe_smem + sizeof(Cx<T>) * (size_t)NBUF * TILE);
    uint64_t* done = full + NBUF;
    const int tid = threadIdx.x, g = tid / GT, gtid = tid - g * GT;
    const int ntiles = (A.nplanes + PB - 1) / PB;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const Cx<T>* twx = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twx_fwd : A.twx_inv);
    const Cx<T>* twy = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twy_fwd : A.twy_inv);

    if (tid == 0) {
        for (int b = 0; b < NBUF; ++b) { mbar_init(&full[b], 1); mbar_init(&done[b], 1); }
        mbar_fence_init();
    }
    __syncthreads();
    if (g == NG) {
        // ---- the I/O warp: fetches, stores and buffer re-arming (see the file header) ----
        if (gtid != 0) return;
        auto fetch = [&](int i) {          // the planes of a tile are contiguous
            const int buf = i % NBUF;
            const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
            const int nvalid = min(PB, A.nplanes - plane0);
            const uint32_t bytes = (uint32_t)(nvalid * PLANE * sizeof(Cx<T>));
            mbar_arrive_expect_tx(&full[buf], bytes);
            bulk_g2s(bufs + (size_t)buf * TILE, in + (size_t)plane0 * PLANE, bytes, &full[buf]);
        };
        auto store = [&](int i, int buf) {
            const Cx<T>* tile = bufs + (size_t)buf * TILE;
            const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
            const int nvalid = min(PB, A.nplanes - plane0);
            if (SIGN < 0) {
                // layout B: plane (comp, t, z) holds the j-th site of tile q / CXB at [tile][rho(t)][z][j]
                for (int pl = 0; pl < nvalid; ++pl) {
                    const int gp = plane0 + pl;
                    const int comp = gp / A.planes_per_comp, zt = gp - comp * A.planes_per_comp;
                    const int t = zt / A.nz, z = zt - t * A.nz;
                    const int tm = t / A.perm_d, tn = t - tm * A.perm_d, tq = tn / A.perm_lq;
                    const int rho = (tq * A.perm_c + tm) * A.perm_lq + (tn - tq * A.perm_lq);
                    for (int sidx = 0; sidx < A.nstores; ++sidx)
                        tma_store_4d(&bmap, tile + pl * PLANE + ((size_t)sidx * A.store_tiles << A.cxb_shift), 0, z, rho,
                                     comp * A.chunks_per_comp + sidx * A.store_tiles);
                }
            } else {
                bulk_s2g(out + (size_t)plane0 * PLANE, tile, (uint32_t)(nvalid * PLANE * sizeof(Cx<T>)));
            }
        };
        io_lane_loop<NBUF>(my_tiles, done, fetch, store);
        return;
    }

    for (int i = g; i < my_tiles; i += NG) {
        const int buf = i % NBUF;
        Cx<T>* tile = bufs + (size_t)buf * TILE;
        mbar_wait(&full[buf], (uint32_t)((i / NBUF) & 1));
        // (planes past the last valid one hold stale data: they are transformed like the others, never stored)

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
            named_bar_sync(1 + g, GT);
            if constexpr (SY::kN2 > 1) {
                for (int it = gtid; it < PB * NX * SY::kN1; it += GT) {
                    const int x = it % NX, k1 = (it / NX) % SY::kN1, pl = it / (NX * SY::kN1);
                    Cx<T>* s = tile + pl * PLANE;
                    stage_B<T, SY, 1, 0>(k1, twy, [&](int p) { return s[p * NX + (x ^ (p & SW))]; },
                                         [&](int p, Cx<T> v) { s[p * NX + (x ^ (p & SW))] = v; }, NoScale());
                }
                named_bar_sync(1 + g, GT);
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
                named_bar_sync(1 + g, GT);
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
            named_bar_sync(1 + g, GT);
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
                named_bar_sync(1 + g, GT);
                if constexpr (SX::kN2 > 1) {
                    for (int it = gtid; it < PB * NY * SX::kN1; it += GT) {
                        const int y = it % NY, k1 = (it / NY) % SX::kN1, pl = it / (NY * SX::kN1);
                        Cx<T>* s = tile + pl * PLANE + y * NX;
                        const int sw = y & SW;
                        stage_B<T, SX, 1, 0>(k1, twx, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; }, NoScale());
                    }
                    named_bar_sync(1 + g, GT);
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
                named_bar_sync(1 + g, GT);
            }
            for (int it = gtid; it < PB * NY * SX::kN2; it += GT) {
                const int y = it % NY, n2 = (it / NY) % SX::kN2, pl = it / (NY * SX::kN2);
                Cx<T>* s = tile + pl * PLANE + y * NX;
                const int sw = y & SW;
                stage_A_inv<T, SX>(n2, [&](int p) { return s[p ^ sw]; }, [&](int p, Cx<T> v) { s[p ^ sw] = v; });
            }
            named_bar_sync(1 + g, GT);
        }
        // ---- un-swizzle in place: the TMA unit stores a dense tile.  One thread owns one aligned group of SW + 1
        // elements of a row (the swizzle permutes inside such a group); it walks the group's slots in an order
        // rotated by its item index, so that the lanes of a shared-memory access phase hit different banks ----
        {
            constexpr int G = SW + 1, NGRP = NX / G;
            for (int it = gtid; it < PB * NY * NGRP; it += GT) {
                const int grp = it % NGRP, y = (it / NGRP) % NY, pl = it / (NGRP * NY);
                Cx<T>* row = tile + pl * PLANE + y * NX + grp * G;
                const int sw = y & SW, rot = it & (G - 1);
                Cx<T> e[G];
                static_for<0, G>([&](auto j) { e[j.value] = row[(j.value + rot) & (G - 1)]; });
                static_for<0, G>([&](auto j) { row[((j.value + rot) & (G - 1)) ^ sw] = e[j.value]; });
            }
        }
        // ---- hand the finished tile to the I/O lane ----
        fence_proxy_async();
        named_bar_sync(1 + g, GT);
        if (gtid == 0) mbar_arrive(&done[buf]);
    }
}

}  // namespace lgf
