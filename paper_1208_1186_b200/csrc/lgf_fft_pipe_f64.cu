// fp64 instantiations of the pipelined FFT kernels.  <T, N, N1, M, M1, PB|CX, GT, NG, NBUF>:
// N1 = N means "whole line in registers"; 48 = 8*6 and 64 = 8*8 take two register stages.
#include "lgf_fft_pipe_inst_impl.cuh"

namespace lgf {
using namespace pinst;
typedef double T;

const XyPipeEntry* xy_pipe_table_f64(int* n) {
    static const XyPipeEntry tab[] = {
        XyP<T, 8, 8, 8, 8, 16, 128, 2, 3>::entry(),
        XyP<T, 16, 16, 16, 16, 8, 128, 2, 3>::entry(),
        XyP<T, 32, 32, 32, 32, 2, 64, 4, 6>::entry(),      // 2-plane tiles, four thread groups: K2 28.0 -> 25.9 us, K4 26.0 -> 24.2 us
        XyP<T, 32, 32, 32, 32, 4, 128, 2, 3>::entry(),
        XyP<T, 32, 32, 32, 32, 4, 128, 3, 3>::entry(),
        XyP<T, 48, 8, 48, 8, 2, 192, 2, 3>::entry(),     // 576 / 768 items per stage: whole rounds of 192 threads
        XyP<T, 48, 8, 48, 8, 1, 256, 2, 4>::entry(),
        XyP<T, 64, 8, 64, 8, 1, 256, 2, 3>::entry(),
    };
    *n = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}
const ZtPipeEntry* zt_pipe_table_f64(int* n) {
    static const ZtPipeEntry tab[] = {
        ZtP<T, 8, 8, 8, 8, 8, 64, 2, 3>::entry(),
        ZtP<T, 16, 16, 16, 16, 4, 64, 2, 3>::entry(),
        ZtP<T, 32, 32, 32, 32, 4, 128, 2, 3>::entry(),
        ZtP<T, 32, 32, 32, 32, 2, 64, 4, 6>::entry(),
        ZtP<T, 32, 32, 32, 32, 4, 128, 3, 3>::entry(),
        ZtP3<T, 48, 16, 8, 8, 8, 192, 2, 4>::entry(),          // three register stages (lgf_fft_pipe3.cuh): 3 passes instead of 5
        ZtP3<T, 48, 16, 8, 8, 8, 128, 3, 4>::entry(),
        ZtP<T, 48, 8, 8, 8, 8, 128, 3, 4>::entry(),
        // the paper's other finite-temperature shapes 48^3 x N_t, N_t = 4, 6, 12
        ZtP3<T, 48, 16, 4, 4, 8, 192, 2, 4>::entry(),
        ZtP<T, 48, 8, 4, 4, 8, 128, 3, 4>::entry(),
        ZtP3<T, 48, 16, 6, 6, 8, 192, 2, 4>::entry(),
        ZtP<T, 48, 8, 6, 6, 8, 128, 3, 4>::entry(),
        ZtP<T, 48, 8, 12, 12, 8, 128, 2, 3>::entry(),        // 384 / 512 / 384 items: whole rounds of 128 threads
        ZtP<T, 48, 8, 8, 8, 8, 256, 2, 4>::entry(),
        ZtP3Q<T, 64, 16, 64, 4, 2, 512>::entry(),             // quarter ring, TMA tensor store of the output
        ZtP3H<T, 64, 16, 64, 4, 2, 512>::entry(),             // 5 shared-memory passes instead of 7
        ZtP3<T, 64, 16, 64, 4, 2, 512, 1, 1>::entry(),
        ZtPH<T, 64, 8, 64, 8, 2, 512>::entry(),
        ZtP<T, 64, 8, 64, 8, 2, 512, 1, 1>::entry(),
    };
    *n = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}
}  // namespace lgf
