// lgf_fft_inst.cuh -- registry of the compile-time-sized FFT kernels (lgf_fft_ct.cuh).
// lgf_fft_inst_f64.cu / lgf_fft_inst_f32.cu instantiate the tables; lgf_api.cu looks kernels up
// by lattice extents and launches them through cudaLaunchKernel.  Sizes that are not in the
// tables run on the generic runtime-radix kernels of lgf_fft.cuh.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace lgf {

struct XyCtEntry {
    int nx, ny;              // plane extents
    int x_n1, y_n1;          // first-stage radices (N1); N2 = N / N1
    int pb;                  // planes per CTA
    int threads;
    size_t smem;
    const void* k_fwd;       // fft_xy_ct<..., -1, ...>
    const void* k_inv;       // fft_xy_ct<..., +1, ...>
};
struct ZtCtEntry {
    int nz, nt;
    int cx;                  // contiguous (x,y)-plane sites per CTA; must divide Lx*Ly
    int threads;
    size_t smem;
    const void* kernel;      // fft_zt_ct<...>
};

// precision: 0 = float, 1 = double (LGF_F32 / LGF_F64)
const XyCtEntry* find_xy_ct(int precision, int nx, int ny);
const ZtCtEntry* find_zt_ct(int precision, int nz, int nt, long long LxLy);
cudaError_t prepare_ct_kernels(int precision);   // raises the dynamic shared memory limits once

const XyCtEntry* xy_table_f64(int* n);
const ZtCtEntry* zt_table_f64(int* n);
const XyCtEntry* xy_table_f32(int* n);
const ZtCtEntry* zt_table_f32(int* n);

}  // namespace lgf
