// lgf_fft_inst.cu -- lookup over the instantiation tables of the compile-time-sized FFT kernels.
#include "lgf_fft_inst.cuh"

namespace lgf {

static const XyCtEntry* xy_tab(int precision, int* n) { return precision ? xy_table_f64(n) : xy_table_f32(n); }
static const ZtCtEntry* zt_tab(int precision, int* n) { return precision ? zt_table_f64(n) : zt_table_f32(n); }

const XyCtEntry* find_xy_ct(int precision, int nx, int ny) {
    int n = 0;
    const XyCtEntry* t = xy_tab(precision, &n);
    for (int i = 0; i < n; ++i)
        if (t[i].nx == nx && t[i].ny == ny) return &t[i];
    return nullptr;
}
const ZtCtEntry* find_zt_ct(int precision, int nz, int nt, long long LxLy) {
    int n = 0;
    const ZtCtEntry* t = zt_tab(precision, &n);
    for (int i = 0; i < n; ++i)
        if (t[i].nz == nz && t[i].nt == nt && LxLy % t[i].cx == 0) return &t[i];
    return nullptr;
}
cudaError_t prepare_ct_kernels(int precision) {
    int n = 0;
    const XyCtEntry* x = xy_tab(precision, &n);
    for (int i = 0; i < n; ++i) {
        if (x[i].smem <= 48 * 1024) continue;
        cudaError_t e = cudaFuncSetAttribute(x[i].k_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)x[i].smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(x[i].k_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)x[i].smem);
        if (e != cudaSuccess) return e;
    }
    const ZtCtEntry* z = zt_tab(precision, &n);
    for (int i = 0; i < n; ++i) {
        if (z[i].smem <= 48 * 1024) continue;
        cudaError_t e = cudaFuncSetAttribute(z[i].kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)z[i].smem);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace lgf
