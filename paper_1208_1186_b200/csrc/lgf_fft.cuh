// lgf_fft.cuh -- batched mixed-radix (2/3/4/8) 4D FFT passes over the packed Delta field, done in
// three kernels (north_star subsystem (c)):
//   K2  forward DFT along x and y          (tile = one contiguous Lx*Ly plane of one component)
//   K3  forward z,t; scale by p2max/(V p2(k)), zero mode -> 0; inverse t,z
//                                           (tile = CX contiguous sites x the whole Lz*Lt plane)
//   K4  inverse DFT along y and x
// Each CTA holds its tile in shared memory; a 1D transform is a sequence of Stockham auto-sort
// stages, every thread doing radix-R butterflies in registers (read all -> barrier -> write all),
// so the spectrum is in natural order and K3 can index the p^2 tables directly.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_math.cuh"

namespace lgf {

constexpr int kMaxStages = 16;   // 4 bits per stage in Axis::radices

// One lattice direction as the FFT kernels see it (all scalars: kernel parameters are never
// indexed dynamically, so nothing is copied to local memory).
struct Axis {
    int N;                        // extent L_mu = product of the radices
    int nstages;
    unsigned long long radices;   // stage s has radix (radices >> 4s) & 15, each in {2,3,4,8}
    const void* tw_fwd;           // Cx<T>[N]: exp(-2 pi i j / N)
    const void* tw_inv;           // Cx<T>[N]: exp(+2 pi i j / N)
    const void* psq;              // T[N]: 4 sin^2(pi k / N)
};

// K2 / K4: tile = one contiguous (x,y) plane of one packed component.
struct XyPass {
    Axis ax, ay;
    int pitch;                    // shared-memory row pitch in elements (Lx + pad)
};

// K3: tile = CX contiguous sites of the (x,y) plane x the whole (z,t) plane of one component.
struct ZtPass {
    Axis az, at;
    int cx;                       // contiguous sites per tile
    int pz, pt;                   // shared-memory strides of the z and t axes (elements)
    long long gz, gt;             // global strides of z and t (elements): LxLy, LxLyLz
    int tiles_per_comp;           // LxLy / cx
    int Lx;
    const void* psq_x;            // T[Lx], T[Ly]
    const void* psq_y;
    double scale_num;             // p2max / V   (SURVEY.md §8(c) readings #5, #7)
};

template <int SIGN, typename T> __device__ __forceinline__ Cx<T> rot90(Cx<T> a) {
    // multiply by exp(SIGN * i pi/2)
    return SIGN < 0 ? mul_mi(a) : mul_i(a);
}

template <int R, int SIGN, typename T> struct Dft;

template <int SIGN, typename T> struct Dft<2, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const Cx<T> a = v[0] + v[1], b = v[0] - v[1];
        v[0] = a; v[1] = b;
    }
};
template <int SIGN, typename T> struct Dft<3, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const T h = T(0.86602540378443864676372317075294);  // sqrt(3)/2
        const Cx<T> t = v[1] + v[2];
        const Cx<T> m = Cx<T>(v[0].re - T(0.5) * t.re, v[0].im - T(0.5) * t.im);
        const Cx<T> s = rot90<SIGN>(h * (v[1] - v[2]));
        v[0] = v[0] + t;
        v[1] = m + s;
        v[2] = m - s;
    }
};
template <int SIGN, typename T> struct Dft<4, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const Cx<T> b0 = v[0] + v[2], b1 = v[0] - v[2], b2 = v[1] + v[3], b3 = rot90<SIGN>(v[1] - v[3]);
        v[0] = b0 + b2; v[2] = b0 - b2; v[1] = b1 + b3; v[3] = b1 - b3;
    }
};
template <int SIGN, typename T> struct Dft<8, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const T r = T(0.70710678118654752440084436210485);  // sqrt(1/2)
        Cx<T> e[4], o[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { e[i] = v[i] + v[i + 4]; o[i] = v[i] - v[i + 4]; }
        // o[m] *= exp(SIGN * 2 pi i m / 8)
        o[1] = (SIGN < 0) ? Cx<T>(r * (o[1].re + o[1].im), r * (o[1].im - o[1].re))
                          : Cx<T>(r * (o[1].re - o[1].im), r * (o[1].im + o[1].re));
        o[2] = rot90<SIGN>(o[2]);
        o[3] = (SIGN < 0) ? Cx<T>(r * (o[3].im - o[3].re), -r * (o[3].re + o[3].im))
                          : Cx<T>(-r * (o[3].re + o[3].im), r * (o[3].re - o[3].im));
        Dft<4, SIGN, T>::run(e);
        Dft<4, SIGN, T>::run(o);
#pragma unroll
        for (int i = 0; i < 4; ++i) { v[2 * i] = e[i]; v[2 * i + 1] = o[i]; }
    }
};

// elements a thread may hold in registers during one stage
constexpr int kElemsPerThread = 16;
template <int R> struct MaxItems { static constexpr int value = kElemsPerThread / R; };

// One Stockham stage of radix R over every line of the tile along `axis`.
template <typename T, int R, int SIGN>
__device__ __forceinline__ void fft_stage(Cx<T>* tile, int N, int pN, int nA, int pA, int nB, int pB, int Ns,
                                          const Cx<T>* __restrict__ tw) {
    constexpr int MAXI = MaxItems<R>::value;
    Cx<T> v[MAXI][R];
    int outbase[MAXI];
    const int nbf = N / R;
    const int items = nA * nB * nbf;
    const int tstep = N / (Ns * R);
#pragma unroll
    for (int i = 0; i < MAXI; ++i) {
        const int item = threadIdx.x + i * blockDim.x;
        outbase[i] = -1;
        if (item < items) {
            const int a = item % nA, q = item / nA;
            const int b = q % nB, j = q / nB;
            const int off = a * pA + b * pB;
            const int k = j % Ns;
#pragma unroll
            for (int m = 0; m < R; ++m) v[i][m] = tile[off + (j + m * nbf) * pN];
            if (Ns > 1) {
#pragma unroll
                for (int m = 1; m < R; ++m) {
                    const Cx<T> w = ld_cx(tw + m * k * tstep);
                    v[i][m] = v[i][m] * w;
                }
            }
            Dft<R, SIGN, T>::run(v[i]);
            outbase[i] = off + ((j - k) * R + k) * pN;
        } else {
            // defined on every path: keeps the register arrays from becoming loop-carried
#pragma unroll
            for (int m = 0; m < R; ++m) v[i][m] = Cx<T>(0, 0);
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < MAXI; ++i) {
        if (outbase[i] >= 0) {
#pragma unroll
            for (int m = 0; m < R; ++m) tile[outbase[i] + m * Ns * pN] = v[i][m];
        }
    }
    __syncthreads();
}

template <typename T, int SIGN>
__device__ __forceinline__ void fft_axis(Cx<T>* tile, const Axis& ax, int pN, int nA, int pA, int nB, int pB) {
    const Cx<T>* tw = reinterpret_cast<const Cx<T>*>(SIGN < 0 ? ax.tw_fwd : ax.tw_inv);
    int Ns = 1;
    for (int st = 0; st < ax.nstages; ++st) {
        const int R = int((ax.radices >> (4 * st)) & 15ull);
        switch (R) {
            case 8: fft_stage<T, 8, SIGN>(tile, ax.N, pN, nA, pA, nB, pB, Ns, tw); break;
            case 4: fft_stage<T, 4, SIGN>(tile, ax.N, pN, nA, pA, nB, pB, Ns, tw); break;
            case 3: fft_stage<T, 3, SIGN>(tile, ax.N, pN, nA, pA, nB, pB, Ns, tw); break;
            default: fft_stage<T, 2, SIGN>(tile, ax.N, pN, nA, pA, nB, pB, Ns, tw); break;
        }
        Ns *= R;
    }
}

template <typename T> struct FftBounds { static constexpr int kMaxThreads = sizeof(T) == 8 ? 512 : 1024; };

// K2 (SIGN = -1: forward x then y) and K4 (SIGN = +1: inverse y then x).  One CTA per plane per
// component: blockIdx.x = comp * Lz*Lt + plane, and the plane is contiguous: base = blockIdx.x * LxLy.
template <typename T, int SIGN>
__global__ void __launch_bounds__(FftBounds<T>::kMaxThreads, 1)
fft_xy_kernel(Cx<T>* __restrict__ D, const XyPass P, const int* done) {
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
    const int nx = P.ax.N, ny = P.ay.N;
    Cx<T>* base = D + (size_t)blockIdx.x * nx * ny;
    const int elems = nx * ny;
    for (int e = threadIdx.x; e < elems; e += blockDim.x) {
        const int y = e / nx, x = e - y * nx;
        tile[x + y * P.pitch] = ld_cx(base + e);
    }
    __syncthreads();
    if (SIGN < 0) {
        fft_axis<T, SIGN>(tile, P.ax, 1, ny, P.pitch, 1, 0);
        fft_axis<T, SIGN>(tile, P.ay, P.pitch, nx, 1, 1, 0);
    } else {
        fft_axis<T, SIGN>(tile, P.ay, P.pitch, nx, 1, 1, 0);
        fft_axis<T, SIGN>(tile, P.ax, 1, ny, P.pitch, 1, 0);
    }
    for (int e = threadIdx.x; e < elems; e += blockDim.x) {
        const int y = e / nx, x = e - y * nx;
        st_cx(base + e, tile[x + y * P.pitch]);
    }
}

// K3: forward z, forward t, scale mode k by p2max/(V p2(k)) (zero mode -> 0), inverse t, inverse z.
template <typename T>
__global__ void __launch_bounds__(FftBounds<T>::kMaxThreads, 1)
fft_zt_kernel(Cx<T>* __restrict__ D, const ZtPass P, long long V, const int* done) {
    pdl_entry();
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (done && *reinterpret_cast<const volatile int*>(done)) return;
    Cx<T>* tile = reinterpret_cast<Cx<T>*>(smem_raw);
    const int comp = blockIdx.x / P.tiles_per_comp;
    const int tidx = blockIdx.x - comp * P.tiles_per_comp;
    const long long tile_off = (long long)tidx * P.cx;          // first (x,y)-plane site of the tile
    Cx<T>* base = D + (size_t)comp * V + tile_off;
    const int nz = P.az.N, nt = P.at.N, cx = P.cx;
    const int n01 = cx * nz;
    const int elems = n01 * nt;
    for (int e = threadIdx.x; e < elems; e += blockDim.x) {
        const int it = e / n01, r = e - it * n01;
        const int iz = r / cx, i0 = r - iz * cx;
        tile[i0 + iz * P.pz + it * P.pt] = ld_cx(base + i0 + iz * P.gz + it * P.gt);
    }
    __syncthreads();
    fft_axis<T, -1>(tile, P.az, P.pz, cx, 1, nt, P.pt);
    fft_axis<T, -1>(tile, P.at, P.pt, cx, 1, nz, P.pz);
    {
        const T* p0 = reinterpret_cast<const T*>(P.psq_x);
        const T* p1 = reinterpret_cast<const T*>(P.psq_y);
        const T* p2 = reinterpret_cast<const T*>(P.az.psq);
        const T* p3 = reinterpret_cast<const T*>(P.at.psq);
        const T num = (T)P.scale_num;
        for (int e = threadIdx.x; e < elems; e += blockDim.x) {
            const int it = e / n01, r = e - it * n01;
            const int iz = r / cx, i0 = r - iz * cx;
            const long long sxy = tile_off + i0;
            const int ky = int(sxy / P.Lx), kx = int(sxy - (long long)ky * P.Lx);
            const T psq = p0[kx] + p1[ky] + p2[iz] + p3[it];
            const T sc = ((kx | ky | iz | it) == 0) ? T(0) : num / psq;
            Cx<T>* q = tile + i0 + iz * P.pz + it * P.pt;
            *q = sc * (*q);
        }
        __syncthreads();
    }
    fft_axis<T, +1>(tile, P.at, P.pt, cx, 1, nz, P.pz);
    fft_axis<T, +1>(tile, P.az, P.pz, cx, 1, nt, P.pt);
    for (int e = threadIdx.x; e < elems; e += blockDim.x) {
        const int it = e / n01, r = e - it * n01;
        const int iz = r / cx, i0 = r - iz * cx;
        st_cx(base + i0 + iz * P.gz + it * P.gt, tile[i0 + iz * P.pz + it * P.pt]);
    }
}

}  // namespace lgf
