// lgf_static.cu -- lgf_measure_static: step 1 of the path (theta and F of a link field, north_star step 1; SURVEY.md
// §8(a) row K1) for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  It is a variant of K1's reduction (lgf_site.cuh: k1_delta_theta_F + k1_finish) that reads the
// links in the BOUNDARY layout of lgf.h (links[s][mu][row][col][re,im], device memory), needs no context and no
// workspace, and keeps its only scratch -- the per-CTA (theta, F) partial sums -- in a file-scope __device__ array.
//
// The array costs kStaticScratchBytes (1 MiB) of device memory on EVERY GPU that loads this library, until the process
// exits, and bounds the lattice to LGF_STATIC_MAX_SITES = 64^4 sites (the largest configuration of BASELINE.json).
// All calls share it: two calls whose kernels overlap on the GPU (different streams, or graph branches) RACE on it;
// calls on one stream are ordered and safe.  Nothing in it has to start at zero: every partial a call reads has been
// written by that call's own first kernel, so the previous call's contents are dead.
//
// In host code `g_static_partials` is a host-side stand-in for the symbol, not a device address; the address the
// kernels get comes from cudaGetSymbolAddress, resolved once per device with that device current (static_scratch()).
// This file calls no cudaMalloc / cudaFree and no library routine that allocates.
// Product code (sm_100a); shares nothing with oracle/.
#include "../../include/lgf.h"

#include <cstdio>
#include <mutex>

#include "lgf_math.cuh"

using namespace lgf;

namespace {

constexpr int kStaticThreads = 256;                                                  // sites per CTA
constexpr long long kStaticMaxSites = LGF_STATIC_MAX_SITES;
constexpr int kStaticMaxBlocks = (int)((kStaticMaxSites + kStaticThreads - 1) / kStaticThreads);
constexpr size_t kStaticScratchBytes = (size_t)kStaticMaxBlocks * sizeof(double2);   // 65536 * 16 B = 1 MiB

static __device__ __align__(256) double2 g_static_partials[kStaticMaxBlocks];

thread_local char g_static_error[256] = "";

int static_fail(cudaError_t e, const char* what) {
    snprintf(g_static_error, sizeof(g_static_error), "%s: %s", what, cudaGetErrorString(e));
    return LGF_ECUDA;
}

// Device address of the scratch array on the CURRENT device (resolved on first use per device, then cached).
constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
double2* g_static_ptr[kMaxDevices] = {};

int static_scratch(double2** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return static_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) {
        snprintf(g_static_error, sizeof(g_static_error), "device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
        return LGF_EUNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        double2* p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_partials);
        if (e != cudaSuccess) return static_fail(e, "cudaGetSymbolAddress(g_static_partials)");
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return LGF_OK;
}

constexpr int kStaticFinishThreads = 1024;

// Sum of (a, b) over the CTA's NT threads, valid in thread 0 (warp shuffles, then one shared-memory hop); the same
// tree as lgf_site.cuh's block_sum2, restated here because that header also DEFINES non-template kernels.
template <int NT>
__device__ __forceinline__ void static_block_sum2(double& a, double& b) {
    __shared__ double sa[NT / 32], sb[NT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sa[w] = a; sb[w] = b; }
    __syncthreads();
    if (w == 0) {
        a = (l < NT / 32) ? sa[l] : 0.0;
        b = (l < NT / 32) ? sb[l] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, o);
            b += __shfl_down_sync(0xffffffffu, b, o);
        }
    }
}

struct StaticGeom {
    int L[4];
    long long V;
};

// One full 3x3 link of the boundary layout: 9 consecutive complex numbers.
template <typename T>
__device__ __forceinline__ void load_link_aos(Su3<T>& u, const Cx<T>* __restrict__ links, long long s, int mu) {
    const Cx<T>* p = links + ((size_t)s * 4 + mu) * 9;
#pragma unroll
    for (int c = 0; c < 9; ++c) u.m[c] = ld_cx(p + c);
}

// First half: thread per site, the per-site arithmetic of k1_delta_theta_F in the same order (so a site contributes
// bit-identical terms), the CTA's sums into partials[blockIdx.x].
template <typename T>
__global__ void __launch_bounds__(kStaticThreads)
k1_static_partials(const Cx<T>* __restrict__ links, double2* __restrict__ partials, const StaticGeom g) {
    const long long s = (long long)blockIdx.x * kStaticThreads + threadIdx.x;
    double th = 0.0, fn = 0.0;
    if (s < g.V) {
        int x[4];
        long long r = s;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            x[mu] = (int)(r % g.L[mu]);
            r /= g.L[mu];
        }
        Cx<T> c0(0, 0), c1(0, 0), c2(0, 0);
        T a0 = 0, a1 = 0, a2 = 0, retr = 0;
        long long stride = 1;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const long long sb = (x[mu] == 0) ? s + stride * (g.L[mu] - 1) : s - stride;
            {
                Su3<T> a;
                load_link_aos<T>(a, links, s, mu);
                c0 = c0 - (a.m[1] - conj(a.m[3]));
                c1 = c1 - (a.m[2] - conj(a.m[6]));
                c2 = c2 - (a.m[5] - conj(a.m[7]));
                a0 -= a.m[0].im; a1 -= a.m[4].im; a2 -= a.m[8].im;
                retr += a.m[0].re + a.m[4].re + a.m[8].re;
            }
            {
                Su3<T> b;
                load_link_aos<T>(b, links, sb, mu);
                c0 = c0 + (b.m[1] - conj(b.m[3]));
                c1 = c1 + (b.m[2] - conj(b.m[6]));
                c2 = c2 + (b.m[5] - conj(b.m[7]));
                a0 += b.m[0].im; a1 += b.m[4].im; a2 += b.m[8].im;
            }
            stride *= g.L[mu];
        }
        a0 *= T(2); a1 *= T(2); a2 *= T(2);
        const T tr3 = (a0 + a1 + a2) / T(3);
        const T d0 = a0 - tr3, d1 = a1 - tr3, d2 = a2 - tr3;
        th = 2.0 * ((double)norm2(c0) + (double)norm2(c1) + (double)norm2(c2)) + (double)d0 * d0 + (double)d1 * d1 +
             (double)d2 * d2;
        fn = (double)retr;
    }
    static_block_sum2<kStaticThreads>(th, fn);
    if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(th, fn);
}

// Second half: one CTA folds the n partials in a fixed order (run-to-run identical) into out = {theta, F}.
__global__ void __launch_bounds__(kStaticFinishThreads)
k1_static_finish(const double2* __restrict__ partials, int n, double V, double* __restrict__ out) {
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < n; i += kStaticFinishThreads) {
        const double2 p = partials[i];
        a += p.x;
        b += p.y;
    }
    static_block_sum2<kStaticFinishThreads>(a, b);
    if (threadIdx.x == 0) {
        out[0] = a / (3.0 * V);
        out[1] = b / (12.0 * V);
    }
}

}  // namespace

extern "C" {

size_t lgf_static_scratch_bytes(void) { return kStaticScratchBytes; }

const char* lgf_static_last_error(void) { return g_static_error; }

int lgf_static_init(void) {
    double2* p = nullptr;
    return static_scratch(&p);
}

int lgf_measure_static(const int32_t L[4], int precision, const void* links_dev, void* cuda_stream, double* theta_F_dev) {
    if (!L || !links_dev || !theta_F_dev || (precision != LGF_F32 && precision != LGF_F64)) {
        snprintf(g_static_error, sizeof(g_static_error), "lgf_measure_static: null pointer or bad precision");
        return LGF_EINVAL;
    }
    StaticGeom g;
    long long V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (L[mu] < 2 || L[mu] > (1 << 20)) {
            snprintf(g_static_error, sizeof(g_static_error), "lgf_measure_static: L[%d] = %d outside 2..2^20", mu, (int)L[mu]);
            return LGF_EINVAL;
        }
        g.L[mu] = L[mu];
        V *= L[mu];
        if (V > kStaticMaxSites) {
            snprintf(g_static_error, sizeof(g_static_error),
                     "lgf_measure_static: lattice exceeds LGF_STATIC_MAX_SITES = %lld sites (the static scratch array holds one "
                     "partial per %d sites); use a context (lgf_create + lgf_measure) for larger lattices",
                     kStaticMaxSites, kStaticThreads);
            return LGF_EINVAL;
        }
    }
    g.V = V;
    double2* partials = nullptr;
    if (int rc = static_scratch(&partials)) return rc;
    cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    const int nblocks = (int)((V + kStaticThreads - 1) / kStaticThreads);
    if (precision == LGF_F64)
        k1_static_partials<double><<<nblocks, kStaticThreads, 0, stream>>>(reinterpret_cast<const Cx<double>*>(links_dev), partials, g);
    else
        k1_static_partials<float><<<nblocks, kStaticThreads, 0, stream>>>(reinterpret_cast<const Cx<float>*>(links_dev), partials, g);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(e, "k1_static_partials launch");
    k1_static_finish<<<1, kStaticFinishThreads, 0, stream>>>(partials, nblocks, (double)V, theta_F_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return static_fail(e, "k1_static_finish launch");
    return LGF_OK;
}

}  // extern "C"
