// lgf_fft_pipe_inst.cuh -- registry of the pipelined FFT kernels (lgf_fft_pipe.cuh).
// lgf_fft_pipe_f64.cu / lgf_fft_pipe_f32.cu instantiate the tables; lgf_api.cu looks kernels up by
// lattice extents.  A lattice runs on this path when BOTH its (x,y) and its (z,t) extents are
// instantiated (K2 writes layout B for exactly the chunk size K3 was compiled for).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace lgf {

struct XyPipeEntry {
    int nx, ny;
    int x_n1, y_n1;          // first-stage radices (digit-swapped spectrum order, see lgf_fft_ct.cuh)
    int pb;                  // planes per tile
    int threads;             // GT * NG (+ 32 for the kernels with an I/O warp)
    int nbuf;
    size_t smem;
    const void* k_fwd;       // fft_xy_pipe<..., -1, ...>  natural -> layout B
    const void* k_inv;       // fft_xy_pipe<..., +1, ...>  natural -> natural (nullptr: forward-only entry)
    int io;                  // 1: fft_xy_pipe_io (I/O warp, TMA tensor stores into layout B; takes the layout-B CUtensorMap)
    int inv3;                // 1: inverse-only entry, fft_xy_inv3 (padded TMA tensor load; takes the Delta~ plane CUtensorMap); k_fwd = nullptr
};
struct ZtPipeEntry {
    int nz, nt;
    int cx;                  // tile width = layout-B chunk (power of two, divides Lx*Ly)
    int threads;
    int nbuf;
    size_t smem;
    const void* kernel;      // fft_zt_pipe<...>  layout B -> natural
    // tstore = 1: the quarter-ring kernel fft_zt_pipe3q, which stores quarter tiles through the TMA unit and takes the 5-D
    // CUtensorMap of the natural-layout Delta~ field as its fifth argument; layout B then holds the t rows quarter by
    // quarter (XyPipeArgs::perm_*; perm_c x perm_d = the kernel's split of the t lines).  0, 1, nt for the ring kernels.
    int tstore, perm_c, perm_d;
};

// precision: 0 = float, 1 = double; LGF_XYP_VARIANT / LGF_ZTP_VARIANT pick the v-th match (A/B knob)
const XyPipeEntry* find_xy_pipe(int precision, int nx, int ny);
const XyPipeEntry* find_xy_pipe_inv(int precision, int nx, int ny, const XyPipeEntry* fwd);
const ZtPipeEntry* find_zt_pipe(int precision, int nz, int nt, long long LxLy);
cudaError_t prepare_pipe_kernels(int precision);

const XyPipeEntry* xy_pipe_table_f64(int* n);
const ZtPipeEntry* zt_pipe_table_f64(int* n);
const XyPipeEntry* xy_pipe_table_f32(int* n);
const ZtPipeEntry* zt_pipe_table_f32(int* n);

}  // namespace lgf
