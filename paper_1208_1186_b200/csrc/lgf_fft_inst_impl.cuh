// lgf_fft_inst_impl.cuh -- included by the two instantiation units with LGF_INST_T defined.
#pragma once
#include "lgf_fft_ct.cuh"
#include "lgf_fft_inst.cuh"

namespace lgf {
namespace inst {

constexpr int round32(int v) { return (v + 31) / 32 * 32; }
constexpr int imax(int a, int b) { return a > b ? a : b; }
constexpr int imin(int a, int b) { return a < b ? a : b; }

// thread count: enough for the widest stage, capped (stages loop over their items)
constexpr int pick_threads(int max_items, int cap) { return imin(imax(round32(max_items), 64), cap); }

template <typename T, int NX, int X1, int NY, int Y1, int PB, int MINB = 1>
struct XyInst {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr int kItems = imax(imax(PB * NX * SY::kN2, SY::kN2 > 1 ? PB * NX * SY::kN1 : 0),
                                       imax(PB * NY * SX::kN2, SX::kN2 > 1 ? PB * NY * SX::kN1 : 0));
    static constexpr int kThreads = pick_threads(kItems, 512);
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)PB * (NX + 1) * NY;
    static XyCtEntry entry() {
        return XyCtEntry{NX, NY, X1, Y1, PB, kThreads, kSmem,
                         (const void*)&fft_xy_ct<T, SX, SY, -1, PB, kThreads, MINB>,
                         (const void*)&fft_xy_ct<T, SX, SY, +1, PB, kThreads, MINB>};
    }
};

template <typename T, int NZ, int Z1, int NT, int T1, int CX, int MINB = 1>
struct ZtInst {
    typedef LineSplit<NZ, Z1> SZ;
    typedef LineSplit<NT, T1> ST_;
    static constexpr int kItems = imax(imax(CX * NT * SZ::kN2, SZ::kN2 > 1 ? CX * NT * SZ::kN1 : 0),
                                       imax(CX * NZ * ST_::kN2, ST_::kN2 > 1 ? CX * NZ * ST_::kN1 : 0));
    static constexpr int kThreads = pick_threads(kItems, 512);
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)CX * (NZ + 1) * NT;
    static ZtCtEntry entry() {
        return ZtCtEntry{NZ, NT, CX, kThreads, kSmem, (const void*)&fft_zt_ct<T, SZ, ST_, CX, kThreads, MINB>};
    }
};

}  // namespace inst
}  // namespace lgf
