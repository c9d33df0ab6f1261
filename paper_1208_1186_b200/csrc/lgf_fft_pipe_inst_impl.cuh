// lgf_fft_pipe_inst_impl.cuh -- entry builders shared by the two instantiation units.
#pragma once
#include "lgf_fft_pipe.cuh"
#include "lgf_fft_pipe3.cuh"
#include "lgf_fft_pipe_io.cuh"
#include "lgf_fft_pipe_inv3.cuh"
#include "lgf_fft_pipe_inst.cuh"

namespace lgf {
namespace pinst {

template <typename T, int NX, int X1, int NY, int Y1, int PB, int GT, int NG, int NBUF>
struct XyP {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * PB * NX * NY + 8 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static XyPipeEntry entry() {
        return XyPipeEntry{NX, NY, X1, Y1, PB, GT * NG, NBUF, kSmem,
                           (const void*)&fft_xy_pipe<T, SX, SY, -1, PB, GT, NG, NBUF>,
                           (const void*)&fft_xy_pipe<T, SX, SY, +1, PB, GT, NG, NBUF>, 0};
    }
};

// K2 in three register stages per plane (xy3_forward_passes); K4 on the same line splits in two stages
template <typename T, int NX, int X1, int NY, int Y1, int PB, int GT, int NG, int NBUF>
struct XyP3 {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * PB * NX * NY + 8 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static XyPipeEntry entry() {
        return XyPipeEntry{NX, NY, X1, Y1, PB, GT * NG, NBUF, kSmem,
                           (const void*)&fft_xy_pipe<T, SX, SY, -1, PB, GT, NG, NBUF, true>,
                           (const void*)&fft_xy_pipe<T, SX, SY, +1, PB, GT, NG, NBUF, false>, 0};
    }
};
// ... and through the I/O warp
template <typename T, int NX, int X1, int NY, int Y1, int PB, int GT, int NG, int NBUF>
struct XyPIO3 {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * PB * NX * NY + 16 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static XyPipeEntry entry() {
        return XyPipeEntry{NX, NY, X1, Y1, PB, GT * NG + 32, NBUF, kSmem,
                           (const void*)&fft_xy_pipe_io<T, SX, SY, -1, PB, GT, NG, NBUF, true>, nullptr, 1};
    }
};

// K4 in three register stages on a padded tile (fft_xy_inv3); inverse only: K2 of the lattice is the XyP3 / XyPIO3 entry
// with the same line splits
template <typename T, int NX, int X1, int NY, int Y1, int PB, int GT, int NG, int NBUF>
struct XyInv3 {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * PB * (NX + XyPad<T>::value) * NY + 8 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static XyPipeEntry entry() {
        return XyPipeEntry{NX, NY, X1, Y1, PB, GT * NG, NBUF, kSmem, nullptr,
                           (const void*)&fft_xy_inv3<T, SX, SY, PB, GT, NG, NBUF>, 0, 1};
    }
};

// K2 through the I/O warp and TMA tensor stores (fft_xy_pipe_io); K4 of such a lattice runs on a plain XyP entry
template <typename T, int NX, int X1, int NY, int Y1, int PB, int GT, int NG, int NBUF>
struct XyPIO {
    typedef LineSplit<NX, X1> SX;
    typedef LineSplit<NY, Y1> SY;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * PB * NX * NY + 16 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static XyPipeEntry entry() {
        return XyPipeEntry{NX, NY, X1, Y1, PB, GT * NG + 32, NBUF, kSmem,
                           (const void*)&fft_xy_pipe_io<T, SX, SY, -1, PB, GT, NG, NBUF>, nullptr, 1};
    }
};

template <typename T, int NZ, int Z1, int NT, int T1, int CX, int GT, int NG, int NBUF>
struct ZtP {
    typedef LineSplit<NZ, Z1> SZ;
    typedef LineSplit<NT, T1> ST_;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * CX * (NZ + 1) * NT + 8 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static_assert((CX & (CX - 1)) == 0, "CX must be a power of two");
    static ZtPipeEntry entry() {
        return ZtPipeEntry{NZ, NT, CX, GT * NG, NBUF, kSmem, (const void*)&fft_zt_pipe<T, SZ, ST_, CX, GT, NG, NBUF>, 0, 1, NT};
    }
};

// three-register-stage K3 (lgf_fft_pipe3.cuh): ring of whole tiles / half-tile ring
template <typename T, int NZ, int Z1, int NT, int T1, int CX, int GT, int NG, int NBUF>
struct ZtP3 {
    typedef LineSplit<NZ, Z1> SZ;
    typedef LineSplit<NT, T1> ST_;
    static constexpr size_t kSmem = sizeof(Cx<T>) * (size_t)NBUF * CX * (NZ + 1) * NT + 8 * NBUF;
    static_assert(kSmem <= 227 * 1024, "tile ring exceeds shared memory");
    static_assert((CX & (CX - 1)) == 0, "CX must be a power of two");
    static ZtPipeEntry entry() {
        return ZtPipeEntry{NZ, NT, CX, GT * NG, NBUF, kSmem, (const void*)&fft_zt_pipe3<T, SZ, ST_, CX, GT, NG, NBUF>, 0, 1, NT};
    }
};
// quarter ring + TMA tensor store (fft_zt_pipe3q)
template <typename T, int NZ, int Z1, int NT, int T1, int CX, int GT>
struct ZtP3Q {
    typedef LineSplit<NZ, Z1> SZ;
    typedef LineSplit<NT, T1> ST_;
    static constexpr size_t kSmem = sizeof(Cx<T>) * ((size_t)6 * CX * (NZ + 1) * (NT / 4) + (size_t)(NT / T1) * (T1 - 1)) + 8 * 6;
    static_assert(kSmem <= 227 * 1024, "quarter-tile ring exceeds shared memory");
    static_assert((CX & (CX - 1)) == 0, "CX must be a power of two");
    static ZtPipeEntry entry() {
        return ZtPipeEntry{NZ, NT, CX, GT, 6, kSmem, (const void*)&fft_zt_pipe3q<T, SZ, ST_, CX, GT>, 1, T1, NT / T1};
    }
};

}  // namespace pinst
}  // namespace lgf
