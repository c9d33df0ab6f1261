// fp64 instantiations of the pipelined FFT kernels.  <T, N, N1, M, M1, PB|CX, GT, NG, NBUF>:
// N1 = N means "whole line in registers"; 48 and 64-point lines take two register stages (K2, K4: 8 x 6, 8 x 8) or
// share three stages per plane (K3: 16 x 3 with the t line, 16 x 4 with 4 x 16).  The first entry for an extent is
// the default; later ones are reachable through LGF_XYP_VARIANT / LGF_ZTP_VARIANT (with LGF_DEVKNOBS=1) for A/B runs.
#include "lgf_fft_pipe_inst_impl.cuh"

namespace lgf {
using namespace pinst;
typedef double T;

const XyPipeEntry* xy_pipe_table_f64(int* n) {
    static const XyPipeEntry tab[] = {
        XyP<T, 8, 8, 8, 8, 16, 128, 2, 3>::entry(),
        XyP<T, 16, 16, 16, 16, 8, 128, 2, 3>::entry(),
        XyP<T, 32, 32, 32, 32, 2, 64, 4, 6>::entry(),
        XyP<T, 32, 32, 32, 32, 4, 128, 2, 3>::entry(),
        XyInv3<T, 32, 32, 32, 32, 2, 64, 3, 6>::entry(),    // K4 at 32 x 32: whole lines on a padded TMA tile, last stage to global
        XyP3<T, 48, 4, 48, 12, 2, 192, 2, 3>::entry(),      // K2 in three stages (12*4 x 4*12); its own K4 (two stages): LGF_XYP_INV_VARIANT=0
        XyInv3<T, 48, 4, 48, 12, 1, 192, 2, 4>::entry(),    // K4: three stages on a padded tile (one round of 192 threads per stage)
        XyP<T, 48, 8, 48, 8, 2, 192, 2, 3>::entry(),     // 576 / 768 items per stage: whole rounds of 192 threads
        XyP<T, 48, 8, 48, 8, 1, 256, 2, 4>::entry(),
        // K2: three stages (16*4 x 4*16), TMA-drained, ONE compute group: with two groups + the I/O warp (17 warps) a
        // scheduler holds five warps, ptxas caps the kernel at 96 registers (104-byte stack frame) and that build failed
        // intermittently on the GPU (5 of 10 bench runs: "unspecified launch failure"); 9 warps leave 170 registers
        XyPIO3<T, 64, 4, 64, 16, 1, 256, 1, 3>::entry(),
        XyInv3<T, 64, 4, 64, 16, 1, 256, 1, 3>::entry(),    // its K4: three stages on a padded tile
        XyP<T, 64, 4, 64, 16, 1, 256, 2, 3>::entry(),       // (K4 in two stages: LGF_XYP_INV_VARIANT=1)
        XyPIO<T, 64, 8, 64, 8, 1, 256, 2, 3>::entry(),      // K2: 32-byte chunks of layout B leave through the TMA unit
        XyP<T, 64, 8, 64, 8, 1, 256, 2, 3>::entry(),        // K4 (and K2 as variant 1)
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
        ZtP3<T, 48, 16, 8, 8, 8, 128, 3, 4>::entry(),        // three groups of 128: 48^3 x 8 K3 30.8 -> 29.4 us (fp64), 21.8 -> 20.9 us (fp32)
        ZtP3<T, 48, 16, 8, 8, 8, 192, 2, 4>::entry(),
        ZtP<T, 48, 8, 8, 8, 8, 128, 3, 4>::entry(),
        // the paper's other finite-temperature shapes 48^3 x N_t, N_t = 4, 6, 12
        ZtP3<T, 48, 16, 4, 4, 8, 192, 2, 4>::entry(),
        ZtP3<T, 48, 16, 6, 6, 8, 192, 2, 4>::entry(),
        ZtP3<T, 48, 16, 12, 12, 8, 128, 2, 3>::entry(),       // 3 x 12 block per thread (36 elements): P2-P4 in one pass
        ZtP<T, 48, 8, 12, 12, 8, 128, 2, 3>::entry(),        // 384 / 512 / 384 items: whole rounds of 128 threads
        ZtP3Q<T, 64, 16, 64, 4, 2, 512>::entry(),
    };
    *n = (int)(sizeof(tab) / sizeof(tab[0]));
    return tab;
}
}  // namespace lgf
