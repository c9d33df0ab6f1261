// fp32 instantiations of the compile-time-sized FFT kernels (see lgf_fft_inst_f64.cu).
#include "lgf_fft_inst_impl.cuh"

namespace lgf {
using namespace inst;
typedef float T;

const XyCtEntry* xy_table_f32(int* n) {
    static const XyCtEntry tab[] = {
        XyInst<T, 8, 8, 8, 8, 16>::entry(),
        XyInst<T, 16, 16, 16, 16, 8>::entry(),
        XyInst<T, 32, 32, 32, 32, 4>::entry(),
        XyInst<T, 32, 32, 32, 32, 2>::entry(),
        XyInst<T, 32, 8, 32, 8, 1>::entry(),
        XyInst<T, 32, 8, 32, 8, 2>::entry(),
        XyInst<T, 32, 16, 32, 16, 2>::entry(),
        XyInst<T, 32, 32, 32, 32, 8>::entry(),
        XyInst<T, 48, 8, 48, 8, 1>::entry(),
        XyInst<T, 64, 8, 64, 8, 1>::entry(),
    };
    *n = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}
const ZtCtEntry* zt_table_f32(int* n) {
    static const ZtCtEntry tab[] = {
        ZtInst<T, 8, 8, 8, 8, 8>::entry(),
        ZtInst<T, 16, 16, 16, 16, 8>::entry(),
        ZtInst<T, 32, 32, 32, 32, 4>::entry(),   // measured: 31 us vs 35 us for CX = 8 at 32^4
        ZtInst<T, 32, 32, 32, 32, 8>::entry(),
        ZtInst<T, 32, 8, 32, 8, 8>::entry(),
        ZtInst<T, 32, 8, 32, 8, 4>::entry(),
        ZtInst<T, 32, 16, 32, 16, 8>::entry(),
        ZtInst<T, 32, 8, 32, 32, 8>::entry(),
        ZtInst<T, 32, 32, 32, 8, 8>::entry(),
        ZtInst<T, 48, 8, 8, 8, 8>::entry(),
        ZtInst<T, 64, 8, 64, 8, 4>::entry(),
    };
    *n = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}
}  // namespace lgf
