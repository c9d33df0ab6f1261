// lgf_fft_ct.cuh -- compile-time-sized FFT pass kernels (the fast path of K2, K3, K4).
//
// A line of length N = N1*N2 is transformed in at most two register stages (lgf_regfft.cuh):
//   forward   A : thread (line, n2) holds x[n2 + N2 m], m < N1   -> DFT_N1 over m -> * w_N^{n2 k1}
//                 and writes Y[k1][n2] back to the SAME positions (position k1*N2 + n2)
//             B : thread (line, k1) holds Y[k1][n2], n2 < N2     -> DFT_N2 over n2 -> X[k1 + N1 k2],
//                 written back to the SAME positions (position k1*N2 + k2)
//   inverse   B': thread (line, k1): DFT_N2^-1 over k2 -> * w_N^{-n2 k1};  A': DFT_N1^-1 over k1.
// Every stage is in place per thread, so a stage needs one barrier (to hand lines to the next
// thread mapping) and no scratch copy.  The price is that the spectrum sits in the digit-swapped
// order  position p = k1*N2 + k2  <->  frequency k = k1 + N1*k2; nothing but the p^2 scale in K3
// looks at frequencies, and it un-swaps with two compile-time divisions.  N2 = 1 is the
// "full line in registers" case (natural order).
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_regfft.cuh"

namespace lgf {

template <int N, int N1> struct LineSplit {
    static_assert(N % N1 == 0, "N1 must divide N");
    static constexpr int kN = N, kN1 = N1, kN2 = N / N1;
    // frequency held at position p after the forward transform
    __host__ __device__ static constexpr int freq_of_pos(int p) { return (p / kN2) + N1 * (p % kN2); }
};

// ---- the four stage bodies; LD(pos) / ST(pos, value) address one line, pos in [0, N) ----------
// tw: table exp(-2 pi i j / N) (forward) or exp(+2 pi i j / N) (inverse), j < N, in global memory.
// WSYNC = 1: a warp-level barrier between the loads and the stores, for callers whose store addresses
// are another lane's load addresses (the swizzling first stage of lgf_fft_pipe.cuh).
template <typename T, class S, int WSYNC = 0, class LD, class ST>
__device__ __forceinline__ void stage_A_fwd(int n2, const Cx<T>* __restrict__ tw, LD&& ld, ST&& st) {
    Cx<T> v[S::kN1];
    static_for<0, S::kN1>([&](auto m) { v[m.value] = ld(n2 + S::kN2 * m.value); });
    if constexpr (WSYNC) __syncwarp();
    RegFft<S::kN1, -1, T>::run(v);
    if constexpr (S::kN2 > 1) {
        static_for<1, S::kN1>([&](auto k1) { v[k1.value] = v[k1.value] * ldg_cx(tw + n2 * k1.value); });
    }
    static_for<0, S::kN1>([&](auto k1) { st(k1.value * S::kN2 + n2, v[k1.value]); });
}
template <typename T, class S, int WSYNC = 0, class LD, class ST>
__device__ __forceinline__ void stage_A_inv(int n2, LD&& ld, ST&& st) {
    Cx<T> v[S::kN1];
    static_for<0, S::kN1>([&](auto k1) { v[k1.value] = ld(k1.value * S::kN2 + n2); });
    if constexpr (WSYNC) __syncwarp();
    RegFft<S::kN1, +1, T>::run(v);
    static_for<0, S::kN1>([&](auto m) { st(n2 + S::kN2 * m.value, v[m.value]); });
}
struct NoScale {};

// B forward, optional scale (SC(k2) -> multiplier for frequency k1 + N1 k2), B' inverse: all on the
// same thread <-> element mapping, so they chain in registers.
template <typename T, class S, int DO_FWD, int DO_INV, int WSYNC = 0, class LD, class ST, class SC>
__device__ __forceinline__ void stage_B(int k1, const Cx<T>* __restrict__ tw_inv, LD&& ld, ST&& st, SC&& sc) {
    Cx<T> v[S::kN2];
    static_for<0, S::kN2>([&](auto j) { v[j.value] = ld(k1 * S::kN2 + j.value); });
    if constexpr (WSYNC) __syncwarp();
    if constexpr (DO_FWD) {
        RegFft<S::kN2, -1, T>::run(v);
        if constexpr (!std::is_same<typename std::decay<SC>::type, NoScale>::value) {
            static_for<0, S::kN2>([&](auto k2) { v[k2.value] = sc(k2.value) * v[k2.value]; });
        }
    }
    if constexpr (DO_INV) {
        RegFft<S::kN2, +1, T>::run(v);
        static_for<1, S::kN2>([&](auto n2) { v[n2.value] = v[n2.value] * ldg_cx(tw_inv + n2.value * k1); });
    }
    static_for<0, S::kN2>([&](auto j) { st(k1 * S::kN2 + j.value, v[j.value]); });
}
struct XyArgs {
    const void* twx_fwd; const void* twx_inv;
    const void* twy_fwd; const void* twy_inv;
    int nplanes;                      // 4 * Lz * Lt
};

// K2 (SIGN = -1) / K4 (SIGN = +1): PB contiguous (x,y) planes per CTA.
template <typename T, class SX, class SY, int SIGN, int PB, int NTHREADS, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB)
fft_xy_ct(Cx<T>* __restrict__ D, const XyArgs A, const int* done) {
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    constexpr int NX = SX::kN, NY = SY::kN, PX = NX + 1, PLANE = PX * NY;
    Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
    const int plane0 = blockIdx.x * PB;
    Cx<T>* base = D + (size_t)plane0 * (NX * NY);
    const int tid = threadIdx.x;
    const Cx<T>* twx = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twx_fwd : A.twx_inv);
    const Cx<T>* twy = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? A.twy_fwd : A.twy_inv);

    // ---- y axis, first stage straight from global memory (threads run along x: coalesced) ----
    if (SIGN < 0) {
        constexpr int NTH = PB * NX * SY::kN2;
        for (int it = tid; it < NTH; it += NTHREADS) {
            const int x = it % NX, n2 = (it / NX) % SY::kN2, pl = it / (NX * SY::kN2);
            if (plane0 + pl < A.nplanes) {
                const Cx<T>* g = base + (size_t)pl * (NX * NY) + x;
                Cx<T>* s = tile + pl * PLANE + x;
                stage_A_fwd<T, SY>(n2, twy, [&](int p) { return ld_cx(g + p * NX); }, [&](int p, Cx<T> v) { s[p * PX] = v; });
            }
        }
        __syncthreads();
        if constexpr (SY::kN2 > 1) {
            constexpr int NTB = PB * NX * SY::kN1;
            for (int it = tid; it < NTB; it += NTHREADS) {
                const int x = it % NX, k1 = (it / NX) % SY::kN1, pl = it / (NX * SY::kN1);
                Cx<T>* s = tile + pl * PLANE + x;
                stage_B<T, SY, 1, 0>(k1, twy, [&](int p) { return s[p * PX]; }, [&](int p, Cx<T> v) { s[p * PX] = v; }, NoScale());
            }
            __syncthreads();
        }
        // ---- x axis (threads run along y; row pitch PX is odd: conflict-free) ----
        {
            constexpr int NTH2 = PB * NY * SX::kN2;
            for (int it = tid; it < NTH2; it += NTHREADS) {
                const int y = it % NY, n2 = (it / NY) % SX::kN2, pl = it / (NY * SX::kN2);
                Cx<T>* s = tile + pl * PLANE + y * PX;
                stage_A_fwd<T, SX>(n2, twx, [&](int p) { return s[p]; }, [&](int p, Cx<T> v) { s[p] = v; });
            }
            __syncthreads();
        }
        if constexpr (SX::kN2 > 1) {
            constexpr int NTB = PB * NY * SX::kN1;
            for (int it = tid; it < NTB; it += NTHREADS) {
                const int y = it % NY, k1 = (it / NY) % SX::kN1, pl = it / (NY * SX::kN1);
                Cx<T>* s = tile + pl * PLANE + y * PX;
                stage_B<T, SX, 1, 0>(k1, twx, [&](int p) { return s[p]; }, [&](int p, Cx<T> v) { s[p] = v; }, NoScale());
            }
            __syncthreads();
        }
    } else {
        // inverse: y axis B' (from global), A'; then x axis B', A'
        if constexpr (SY::kN2 > 1) {
            constexpr int NTB = PB * NX * SY::kN1;
            for (int it = tid; it < NTB; it += NTHREADS) {
                const int x = it % NX, k1 = (it / NX) % SY::kN1, pl = it / (NX * SY::kN1);
                if (plane0 + pl < A.nplanes) {
                    const Cx<T>* g = base + (size_t)pl * (NX * NY) + x;
                    Cx<T>* s = tile + pl * PLANE + x;
                    stage_B<T, SY, 0, 1>(k1, twy, [&](int p) { return ld_cx(g + p * NX); }, [&](int p, Cx<T> v) { s[p * PX] = v; }, NoScale());
                }
            }
            __syncthreads();
            constexpr int NTH = PB * NX * SY::kN2;
            for (int it = tid; it < NTH; it += NTHREADS) {
                const int x = it % NX, n2 = (it / NX) % SY::kN2, pl = it / (NX * SY::kN2);
                Cx<T>* s = tile + pl * PLANE + x;
                stage_A_inv<T, SY>(n2, [&](int p) { return s[p * PX]; }, [&](int p, Cx<T> v) { s[p * PX] = v; });
            }
            __syncthreads();
        } else {
            constexpr int NTH = PB * NX;
            for (int it = tid; it < NTH; it += NTHREADS) {
                const int x = it % NX, pl = it / NX;
                if (plane0 + pl < A.nplanes) {
                    const Cx<T>* g = base + (size_t)pl * (NX * NY) + x;
                    Cx<T>* s = tile + pl * PLANE + x;
                    stage_A_inv<T, SY>(0, [&](int p) { return ld_cx(g + p * NX); }, [&](int p, Cx<T> v) { s[p * PX] = v; });
                }
            }
            __syncthreads();
        }
        if constexpr (SX::kN2 > 1) {
            constexpr int NTB = PB * NY * SX::kN1;
            for (int it = tid; it < NTB; it += NTHREADS) {
                const int y = it % NY, k1 = (it / NY) % SX::kN1, pl = it / (NY * SX::kN1);
                Cx<T>* s = tile + pl * PLANE + y * PX;
                stage_B<T, SX, 0, 1>(k1, twx, [&](int p) { return s[p]; }, [&](int p, Cx<T> v) { s[p] = v; }, NoScale());
            }
            __syncthreads();
        }
        {
            constexpr int NTH2 = PB * NY * SX::kN2;
            for (int it = tid; it < NTH2; it += NTHREADS) {
                const int y = it % NY, n2 = (it / NY) % SX::kN2, pl = it / (NY * SX::kN2);
                Cx<T>* s = tile + pl * PLANE + y * PX;
                stage_A_inv<T, SX>(n2, [&](int p) { return s[p]; }, [&](int p, Cx<T> v) { s[p] = v; });
            }
            __syncthreads();
        }
    }
    // ---- coalesced copy-out ----
    constexpr int ELEMS = PB * NX * NY;
#pragma unroll 4
    for (int e = tid; e < ELEMS; e += NTHREADS) {
        const int x = e % NX, y = (e / NX) % NY, pl = e / (NX * NY);
        if (plane0 + pl < A.nplanes) st_cx(base + e, tile[pl * PLANE + y * PX + x]);
    }
}

struct ZtArgs {
    const void* twz_fwd; const void* twz_inv;
    const void* twt_fwd; const void* twt_inv;
    const void* psq_x; const void* psq_y; const void* psq_z; const void* psq_t;
    long long V;
    long long LxLy;
    int Lx;
    int tiles_per_comp;               // LxLy / CX
    int nbatch;                       // lattices per launch (batched contexts): components run over 4 * nbatch
    double scale_num;                 // p2max / V
    int x_n1, x_n2, y_n1, y_n2;       // how K2 split the x and y lines (digit-swapped spectrum order)
    // psq_t[k] for k = 0..Lt/2, by value (read as constant-bank operands by the whole-line t pass of the pipelined K3;
    // the table is symmetric, psq_t[Lt - k] = psq_t[k], so one quotient serves both modes); Lt <= 64
    double psq_t_half_d[33];
    float psq_t_half_f[33];
};
__device__ __forceinline__ double psq_t_half(const ZtArgs& A, int k, double) { return A.psq_t_half_d[k]; }
__device__ __forceinline__ float psq_t_half(const ZtArgs& A, int k, float) { return A.psq_t_half_f[k]; }

// K3: forward z, forward t, scale, inverse t, inverse z on CX contiguous (x,y)-plane sites.
template <typename T, class SZ, class ST_, int CX, int NTHREADS, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB)
fft_zt_ct(Cx<T>* __restrict__ D, const ZtArgs A, const int* done) {
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    constexpr int NZ = SZ::kN, NT = ST_::kN, PZ = CX, PT = CX * (NZ + 1);
    Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
    const int comp = blockIdx.x / A.tiles_per_comp;
    const int tidx = blockIdx.x - comp * A.tiles_per_comp;
    const long long tile_off = (long long)tidx * CX;
    Cx<T>* base = D + (size_t)comp * A.V + tile_off;
    const long long gz = A.LxLy, gt = A.LxLy * NZ;
    const int tid = threadIdx.x;
    const Cx<T>* twz_f = reinterpret_cast<const Cx<T>*>(A.twz_fwd);
    const Cx<T>* twz_i = reinterpret_cast<const Cx<T>*>(A.twz_inv);
    const Cx<T>* twt_f = reinterpret_cast<const Cx<T>*>(A.twt_fwd);
    const Cx<T>* twt_i = reinterpret_cast<const Cx<T>*>(A.twt_inv);

    // ---- z forward: A from global, B in smem ----
    {
        constexpr int NTH = CX * NT * SZ::kN2;
        for (int it = tid; it < NTH; it += NTHREADS) {
            const int cx = it % CX, t = (it / CX) % NT, n2 = it / (CX * NT);
            const Cx<T>* g = base + cx + (size_t)t * gt;
            Cx<T>* s = tile + cx + t * PT;
            stage_A_fwd<T, SZ>(n2, twz_f, [&](int p) { return ld_cx(g + (size_t)p * gz); }, [&](int p, Cx<T> v) { s[p * PZ] = v; });
        }
        __syncthreads();
    }
    if constexpr (SZ::kN2 > 1) {
        constexpr int NTB = CX * NT * SZ::kN1;
        for (int it = tid; it < NTB; it += NTHREADS) {
            const int cx = it % CX, t = (it / CX) % NT, k1 = it / (CX * NT);
            Cx<T>* s = tile + cx + t * PT;
            stage_B<T, SZ, 1, 0>(k1, twz_i, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { s[p * PZ] = v; }, NoScale());
        }
        __syncthreads();
    }
    // ---- t: A forward | B forward, scale, B' inverse | A' inverse (or the whole line in registers) ----
    {
        constexpr int NLT = CX * NZ;                 // t lines in the tile
        auto line_momentum = [&](int cx, int zp, T& pxyz, bool& zero_xyz) {
            // x, y frequencies from the tile position (un-swapping K2's order), z from zp
            const long long sxy = tile_off + cx;
            const int ypos = int(sxy / A.Lx), xpos = int(sxy - (long long)ypos * A.Lx);
            const int kx = (xpos / A.x_n2) + A.x_n1 * (xpos % A.x_n2), ky = (ypos / A.y_n2) + A.y_n1 * (ypos % A.y_n2);
            const int kz = SZ::freq_of_pos(zp);
            pxyz = reinterpret_cast<const T*>(A.psq_x)[kx] + reinterpret_cast<const T*>(A.psq_y)[ky] +
                   reinterpret_cast<const T*>(A.psq_z)[kz];
            zero_xyz = (kx | ky | kz) == 0;
        };
        const T* pt = reinterpret_cast<const T*>(A.psq_t);
        const T num = (T)A.scale_num;
        if constexpr (ST_::kN2 > 1) {
            for (int it = tid; it < NLT * ST_::kN2; it += NTHREADS) {
                const int cx = it % CX, zp = (it / CX) % NZ, n2 = it / NLT;
                Cx<T>* s = tile + cx + zp * PZ;
                stage_A_fwd<T, ST_>(n2, twt_f, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; });
            }
            __syncthreads();
            for (int it = tid; it < NLT * ST_::kN1; it += NTHREADS) {
                const int cx = it % CX, zp = (it / CX) % NZ, k1 = it / NLT;
                Cx<T>* s = tile + cx + zp * PZ;
                T pxyz; bool zero_xyz;
                line_momentum(cx, zp, pxyz, zero_xyz);
                auto scale = [&](int k2) -> T {
                    const int kt = k1 + ST_::kN1 * k2;
                    const T den = pxyz + __ldg(pt + kt);
                    return (zero_xyz && kt == 0) ? T(0) : num / den;
                };
                stage_B<T, ST_, 1, 1>(k1, twt_i, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; }, scale);
            }
            __syncthreads();
            for (int it = tid; it < NLT * ST_::kN2; it += NTHREADS) {
                const int cx = it % CX, zp = (it / CX) % NZ, n2 = it / NLT;
                Cx<T>* s = tile + cx + zp * PZ;
                stage_A_inv<T, ST_>(n2, [&](int p) { return s[p * PT]; }, [&](int p, Cx<T> v) { s[p * PT] = v; });
            }
            __syncthreads();
        } else {
            for (int it = tid; it < NLT; it += NTHREADS) {
                const int cx = it % CX, zp = it / CX;
                Cx<T>* s = tile + cx + zp * PZ;
                T pxyz; bool zero_xyz;
                line_momentum(cx, zp, pxyz, zero_xyz);
                Cx<T> v[NT];
                static_for<0, NT>([&](auto m) { v[m.value] = s[m.value * PT]; });
                RegFft<NT, -1, T>::run(v);
                static_for<0, NT>([&](auto kt) {
                    const T den = pxyz + __ldg(pt + kt.value);
                    const T sc = (zero_xyz && kt.value == 0) ? T(0) : num / den;
                    v[kt.value] = sc * v[kt.value];
                });
                RegFft<NT, +1, T>::run(v);
                static_for<0, NT>([&](auto m) { s[m.value * PT] = v[m.value]; });
            }
            __syncthreads();
        }
    }
    // ---- z inverse: B' in smem, A' straight to global ----
    if constexpr (SZ::kN2 > 1) {
        constexpr int NTB = CX * NT * SZ::kN1;
        for (int it = tid; it < NTB; it += NTHREADS) {
            const int cx = it % CX, t = (it / CX) % NT, k1 = it / (CX * NT);
            Cx<T>* s = tile + cx + t * PT;
            stage_B<T, SZ, 0, 1>(k1, twz_i, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { s[p * PZ] = v; }, NoScale());
        }
        __syncthreads();
    }
    {
        constexpr int NTH = CX * NT * SZ::kN2;
        for (int it = tid; it < NTH; it += NTHREADS) {
            const int cx = it % CX, t = (it / CX) % NT, n2 = it / (CX * NT);
            Cx<T>* g = base + cx + (size_t)t * gt;
            const Cx<T>* s = tile + cx + t * PT;
            stage_A_inv<T, SZ>(n2, [&](int p) { return s[p * PZ]; }, [&](int p, Cx<T> v) { st_cx(g + (size_t)p * gz, v); });
        }
    }
}

}  // namespace lgf
