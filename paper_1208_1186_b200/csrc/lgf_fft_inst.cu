// lgf_fft_inst.cu -- lookup over the instantiation tables of the compile-time-sized FFT kernels.
#include "lgf_fft_inst.cuh"
#include "lgf_fft_pipe_inst.cuh"

#include <cstdlib>

namespace lgf {

static const XyCtEntry* xy_tab(int precision, int* n) { return precision ? xy_table_f64(n) : xy_table_f32(n); }
static const ZtCtEntry* zt_tab(int precision, int* n) { return precision ? zt_table_f64(n) : zt_table_f32(n); }

// Several entries may serve the same extents (different splits / tile sizes): the first one is the
// tuned default; LGF_XY_VARIANT / LGF_ZT_VARIANT = v select the v-th match (developer A/B knob).
static const char* knob(const char* name) {       // developer knobs are honoured only with LGF_DEVKNOBS=1 (see lgf_api.cu)
    const char* on = getenv("LGF_DEVKNOBS");
    return (on && atoi(on) != 0) ? getenv(name) : nullptr;
}
static int variant(const char* name) {
    const char* e = knob(name);
    return e ? atoi(e) : 0;
}

const XyCtEntry* find_xy_ct(int precision, int nx, int ny) {
    int n = 0, skip = variant("LGF_XY_VARIANT");
    const XyCtEntry* t = xy_tab(precision, &n);
    const XyCtEntry* last = nullptr;
    for (int i = 0; i < n; ++i)
        if (t[i].nx == nx && t[i].ny == ny) {
            last = &t[i];
            if (skip-- == 0) return last;
        }
    return last;
}
const ZtCtEntry* find_zt_ct(int precision, int nz, int nt, long long LxLy) {
    int n = 0, skip = variant("LGF_ZT_VARIANT");
    const ZtCtEntry* t = zt_tab(precision, &n);
    const ZtCtEntry* last = nullptr;
    for (int i = 0; i < n; ++i)
        if (t[i].nz == nz && t[i].nt == nt && LxLy % t[i].cx == 0) {
            last = &t[i];
            if (skip-- == 0) return last;
        }
    return last;
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


// ---- pipelined kernels (lgf_fft_pipe.cuh) ----
static const XyPipeEntry* xyp_tab(int precision, int* n) { return precision ? xy_pipe_table_f64(n) : xy_pipe_table_f32(n); }
static const ZtPipeEntry* ztp_tab(int precision, int* n) { return precision ? zt_pipe_table_f64(n) : zt_pipe_table_f32(n); }

// K4 may run on another entry than K2 as long as the line splits agree (both read and write the natural layout on
// their own): LGF_XYP_INV_VARIANT = v picks the v-th such entry.
const XyPipeEntry* find_xy_pipe_inv(int precision, int nx, int ny, const XyPipeEntry* fwd) {
    int n = 0;
    const XyPipeEntry* t = xyp_tab(precision, &n);
    auto matches = [&](const XyPipeEntry& x) { return x.nx == nx && x.ny == ny && x.x_n1 == fwd->x_n1 && x.y_n1 == fwd->y_n1 && x.k_inv; };
    if (const char* e = knob("LGF_XYP_INV_VARIANT")) {       // the v-th entry that can invert K2's line splits
        int skip = atoi(e);
        const XyPipeEntry* last = nullptr;
        for (int i = 0; i < n; ++i)
            if (matches(t[i])) {
                last = &t[i];
                if (skip-- == 0) return last;
            }
        return last;
    }
    for (int i = 0; i < n; ++i)                               // default: the three-stage inverse where one is instantiated,
        if (matches(t[i]) && t[i].inv3) return &t[i];
    if (fwd->k_inv) return fwd;                               // else K2's own entry,
    for (int i = 0; i < n; ++i)                               // else (forward-only K2 entries) the first that fits
        if (matches(t[i])) return &t[i];
    return nullptr;
}
const XyPipeEntry* find_xy_pipe(int precision, int nx, int ny) {
    int n = 0, skip = variant("LGF_XYP_VARIANT");
    const XyPipeEntry* t = xyp_tab(precision, &n);
    const XyPipeEntry* last = nullptr;
    for (int i = 0; i < n; ++i)
        if (t[i].nx == nx && t[i].ny == ny && t[i].k_fwd) {
            last = &t[i];
            if (skip-- == 0) return last;
        }
    return last;
}
const ZtPipeEntry* find_zt_pipe(int precision, int nz, int nt, long long LxLy) {
    int n = 0, skip = variant("LGF_ZTP_VARIANT");
    const ZtPipeEntry* t = ztp_tab(precision, &n);
    const ZtPipeEntry* last = nullptr;
    for (int i = 0; i < n; ++i)
        if (t[i].nz == nz && t[i].nt == nt && LxLy % t[i].cx == 0) {
            last = &t[i];
            if (skip-- == 0) return last;
        }
    return last;
}
cudaError_t prepare_pipe_kernels(int precision) {
    int n = 0;
    const XyPipeEntry* x = xyp_tab(precision, &n);
    for (int i = 0; i < n; ++i) {
        cudaError_t e = x[i].k_fwd ? cudaFuncSetAttribute(x[i].k_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)x[i].smem) : cudaSuccess;
        if (e == cudaSuccess && x[i].k_inv) e = cudaFuncSetAttribute(x[i].k_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)x[i].smem);
        if (e != cudaSuccess) return e;
    }
    const ZtPipeEntry* z = ztp_tab(precision, &n);
    for (int i = 0; i < n; ++i) {
        cudaError_t e = cudaFuncSetAttribute(z[i].kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)z[i].smem);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace lgf
