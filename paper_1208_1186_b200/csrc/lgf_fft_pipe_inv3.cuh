// lgf_fft_pipe_inv3.cuh -- K4 (inverse DFT along x and y) in THREE register stages per plane,
// the mirror image of xy3_forward_passes (lgf_fft_pipe.cuh) on the digit-swapped spectrum K2 leaves:
//   Q1  thread (y, k1x):    DFT_D^-1 over the columns k1x*D + k2x, times w_Nx^{+n2x k1x}          (lanes along y)
//   Q2  thread (n2x, k1y):  DFT_C^-1 over the columns k1x*D + n2x, then DFT_B^-1 over the rows k1y*B + k2y   (a B x C block)
//   Q3  thread (x, n2y):    times w_Ny^{+n2y k1y}, DFT_A^-1 over the rows k1y*B + n2y  -> global memory, natural order,
//                           coalesced along x (no copy-out pass)
// The digit order forces the 16-point x stage first, i.e. a first pass whose lanes run along y over a densely loaded
// tile -- a 32-way bank conflict.  The tile is therefore fetched by a TMA TENSOR load whose box is one column (fp32: two)
// WIDER than the plane: the out-of-range column is zero-filled and gives the shared-memory rows an odd pitch
// (N_x + 1 elements), so that lanes along y AND lanes along x are conflict-free without any swizzle (fp32: the pitch
// must stay a multiple of 16 bytes, N_x + 2 elements: Q1 alone keeps a 2-way conflict).
// Shared-memory traffic per plane: the fetch + Q1 (read, write) + Q2 (read, write) + Q3 (read) = 6 traversals
// instead of 10 for the two-stage kernel (fetch, four passes, copy-out).
// Lines that fit one thread's registers (32 points, LineSplit<N, N>) run the same scheme in TWO stages: whole x lines in
// place, whole y lines straight to global memory.
// Ring of NBUF tile buffers and NG thread groups as in fft_xy_pipe.  Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include "lgf_fft_pipe.cuh"

namespace lgf {

// global -> shared TENSOR load of a 3-D box (SASS UTMALDG), completing on `bar` as box-size bytes of transaction count
__device__ __forceinline__ void tma_load_3d(void* dst_smem, const void* tmap, int c0, int c1, int c2, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
                 : "memory");
}

template <typename T> struct XyPad { static constexpr int value = sizeof(T) == 8 ? 1 : 2; };

// `imap`: CUtensorMap of the natural-layout Delta~ field as the 3-D tensor (2 reals x N_x, N_y, planes).
template <typename T, class SX, class SY, int PB, int GT, int NG, int NBUF>
__global__ void __launch_bounds__(GT * NG, 1)
fft_xy_inv3(const Cx<T>* in, Cx<T>* out, const __grid_constant__ XyPipeArgs A_, const int* done,
            const __grid_constant__ CUtensorMap imap) {
    pdl_entry();
    extern __shared__ __align__(128) unsigned char pipe_smem[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    constexpr int NX = SX::kN, NY = SY::kN, P = NX + XyPad<T>::value, PLANE = P * NY, TILE = PB * PLANE;
    constexpr int A = SY::kN1, B = SY::kN2, C = SX::kN1, D = SX::kN2;
    constexpr bool WHOLE = (B == 1 && D == 1);       // lines that fit one thread's registers (32 points): Q1 and Q3 only
    static_assert(WHOLE || (B > 1 && D > 1 && B * C <= 16), "three-stage K4: the middle block must fit the registers");
    static_assert((TILE * sizeof(Cx<T>)) % 128 == 0 && (P * sizeof(Cx<T>)) % 16 == 0, "tensor-load alignment");
    // NBUF % NG == 0: a buffer is always re-armed by the group that consumes it.  With NG = 2, NBUF = 3 (the groups hand
    // buffers to each other, as fft_xy_pipe does without trouble) this kernel ended in "unspecified launch failure" on
    // the GPU once a CTA had more than ~55 tiles (fp64, 64^4 and 16 x 48^3x12); cause not found.
    static_assert(NBUF >= NG && NBUF % NG == 0 && GT % 32 == 0, "ring");
    (void)in;
    Cx<T>* bufs = reinterpret_cast<Cx<T>*>(pipe_smem);
    uint64_t* full = reinterpret_cast<uint64_t*>(pipe_smem + sizeof(Cx<T>) * (size_t)NBUF * TILE);
    const int tid = threadIdx.x, g = tid / GT, gtid = tid - g * GT;
    const int ntiles = (A_.nplanes + PB - 1) / PB;
    const int my_tiles = (int)blockIdx.x < ntiles ? (ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;

    // one thread arms buffer i % NBUF for this CTA's i-th tile; planes past the last one are zero-filled like the pad column
    auto issue = [&](int i) {
        const int buf = i % NBUF;
        const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
        mbar_arrive_expect_tx(&full[buf], (uint32_t)(TILE * sizeof(Cx<T>)));
        tma_load_3d(bufs + (size_t)buf * TILE, &imap, 0, 0, plane0, &full[buf]);
    };
    if (tid == 0) {
        for (int b = 0; b < NBUF; ++b) mbar_init(&full[b], 1);
        mbar_fence_init();
        for (int i = 0; i < NBUF && i < my_tiles; ++i) issue(i);
    }
    __syncthreads();
    const uint64_t keep = l2_evict_last_policy();          // Delta~ is K5's next read

    for (int i = g; i < my_tiles; i += NG) {
        const int buf = i % NBUF;
        Cx<T>* tile = bufs + (size_t)buf * TILE;
        const int plane0 = ((int)blockIdx.x + i * (int)gridDim.x) * PB;
        const int nvalid = min(PB, A_.nplanes - plane0);
        mbar_wait(&full[buf], (uint32_t)((i / NBUF) & 1));

        if constexpr (WHOLE) {
            // ---- whole x lines in place (lanes along y: the odd pitch keeps them conflict-free) ----
            for (int it = gtid; it < PB * NY; it += GT) {
                Cx<T>* s = tile + (it / NY) * PLANE + (it % NY) * P;
                Cx<T> v[NX];
                static_for<0, NX>([&](auto j) { v[j.value] = s[j.value]; });
                RegFft<NX, +1, T>::run(v);
                static_for<0, NX>([&](auto j) { s[j.value] = v[j.value]; });
            }
            group_sync<GT, NG>(g);
            // ---- whole y lines, straight to global memory (lanes along x: coalesced) ----
            for (int it = gtid; it < PB * NX; it += GT) {
                const int x = it % NX, pl = it / NX;
                if (pl < nvalid) {
                    const Cx<T>* s = tile + pl * PLANE + x;
                    Cx<T> v[NY];
                    static_for<0, NY>([&](auto k) { v[k.value] = s[k.value * P]; });
                    RegFft<NY, +1, T>::run(v);
                    Cx<T>* gp = out + (size_t)(plane0 + pl) * (NX * NY) + x;
                    static_for<0, NY>([&](auto k) { st_cx_keep(gp + (size_t)k.value * NX, v[k.value], keep); });
                }
            }
        } else {
        // ---- Q1: x, 16-point stage (lanes along y) ----
        for (int it = gtid; it < PB * NY * C; it += GT) {
            const int y = it % NY, k1x = (it / NY) % C, pl = it / (NY * C);
            Cx<T>* s = tile + pl * PLANE + y * P + k1x * D;
            Cx<T> v[D];
            static_for<0, D>([&](auto j) { v[j.value] = s[j.value]; });
            RegFft<D, +1, T>::run(v);
            tw_rows<NX, D, C, +1, T>(v, k1x);
            static_for<0, D>([&](auto j) { s[j.value] = v[j.value]; });
        }
        group_sync<GT, NG>(g);
        // ---- Q2: the B x C block: x, 4-point stage; y, 4-point stage (lanes along x) ----
        for (int it = gtid; it < PB * D * A; it += GT) {
            const int n2x = it % D, k1y = (it / D) % A, pl = it / (D * A);
            Cx<T>* s = tile + pl * PLANE + k1y * B * P + n2x;
            Cx<T> e[C][B];
            static_for<0, B>([&](auto j) {
                Cx<T> u[C];
                static_for<0, C>([&](auto k) { u[k.value] = s[j.value * P + k.value * D]; });
                RegFft<C, +1, T>::run(u);
                static_for<0, C>([&](auto m) { e[m.value][j.value] = u[m.value]; });
            });
            static_for<0, C>([&](auto m) {
                RegFft<B, +1, T>::run(e[m.value]);
                static_for<0, B>([&](auto j) { s[j.value * P + m.value * D] = e[m.value][j.value]; });
            });
        }
        group_sync<GT, NG>(g);
        // ---- Q3: y, 16-point stage, straight to global memory (lanes along x: coalesced) ----
        for (int it = gtid; it < PB * NX * B; it += GT) {
            const int x = it % NX, n2y = (it / NX) % B, pl = it / (NX * B);
            if (pl < nvalid) {
                const Cx<T>* s = tile + pl * PLANE + n2y * P + x;
                Cx<T> v[A];
                static_for<0, A>([&](auto k1) { v[k1.value] = s[k1.value * B * P]; });
                tw_rows<NY, A, B, +1, T>(v, n2y);
                RegFft<A, +1, T>::run(v);
                Cx<T>* gp = out + (size_t)(plane0 + pl) * (NX * NY) + (size_t)n2y * NX + x;
                static_for<0, A>([&](auto m) { st_cx_keep(gp + (size_t)m.value * B * NX, v[m.value], keep); });
            }
        }
        }
        // ---- hand the buffer back to the TMA unit for tile i + NBUF ----
        fence_proxy_async();
        group_sync<GT, NG>(g);
        if (i + NBUF < my_tiles && gtid == 0) issue(i + NBUF);
    }
}

}  // namespace lgf
