// lgf_math.cuh -- complex and SU(3) register arithmetic for the CUDA path (sm_100a).
// Product code; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lgf {

template <typename T> struct Vec2;
template <> struct Vec2<float> { typedef float2 type; };
template <> struct Vec2<double> { typedef double2 type; };

// complex number, layout-compatible with float2 / double2 (re, im interleaved)
template <typename T>
struct __align__(2 * sizeof(T)) Cx {
    T re, im;
    Cx() = default;
    __host__ __device__ Cx(T r, T i) : re(r), im(i) {}
};

template <typename T> __device__ __forceinline__ Cx<T> operator+(Cx<T> a, Cx<T> b) { return Cx<T>(a.re + b.re, a.im + b.im); }
template <typename T> __device__ __forceinline__ Cx<T> operator-(Cx<T> a, Cx<T> b) { return Cx<T>(a.re - b.re, a.im - b.im); }
template <typename T> __device__ __forceinline__ Cx<T> operator*(Cx<T> a, Cx<T> b) {
    return Cx<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename T> __device__ __forceinline__ Cx<T> operator*(T s, Cx<T> a) { return Cx<T>(s * a.re, s * a.im); }
template <typename T> __device__ __forceinline__ Cx<T> conj(Cx<T> a) { return Cx<T>(a.re, -a.im); }
// a * conj(b)
template <typename T> __device__ __forceinline__ Cx<T> mulc(Cx<T> a, Cx<T> b) {
    return Cx<T>(a.re * b.re + a.im * b.im, a.im * b.re - a.re * b.im);
}
// conj(a) * conj(b)
template <typename T> __device__ __forceinline__ Cx<T> cmulc(Cx<T> a, Cx<T> b) {
    return Cx<T>(a.re * b.re - a.im * b.im, -(a.re * b.im + a.im * b.re));
}
// acc += a*b
template <typename T> __device__ __forceinline__ void fma_cx(Cx<T>& acc, Cx<T> a, Cx<T> b) {
    acc.re += a.re * b.re; acc.re -= a.im * b.im;
    acc.im += a.re * b.im; acc.im += a.im * b.re;
}
// acc += a*conj(b)
template <typename T> __device__ __forceinline__ void fma_cxc(Cx<T>& acc, Cx<T> a, Cx<T> b) {
    acc.re += a.re * b.re; acc.re += a.im * b.im;
    acc.im += a.im * b.re; acc.im -= a.re * b.im;
}
template <typename T> __device__ __forceinline__ T norm2(Cx<T> a) { return a.re * a.re + a.im * a.im; }
// multiply by +i / -i
template <typename T> __device__ __forceinline__ Cx<T> mul_i(Cx<T> a) { return Cx<T>(-a.im, a.re); }
template <typename T> __device__ __forceinline__ Cx<T> mul_mi(Cx<T> a) { return Cx<T>(a.im, -a.re); }

// fp32: MUFU.RSQ + one Newton step (~1 ulp) instead of sqrt and divide with their slow-path branches (~25 instructions
// each, 7 per site in K5, which is issue-bound in fp32); fp64 keeps the correctly rounded 1/sqrt.
__device__ __forceinline__ float rsqrt_t(float x) {
    const float y = rsqrtf(x);
    return y * fmaf(-0.5f * x * y, y, 1.5f);
}
__device__ __forceinline__ double rsqrt_t(double x) { return 1.0 / sqrt(x); }

// Streaming 16-byte / 8-byte global accesses of one complex number.
template <typename T> __device__ __forceinline__ Cx<T> ldg_cx(const Cx<T>* p) {
    typedef typename Vec2<T>::type V;
    V v = __ldg(reinterpret_cast<const V*>(p));
    return Cx<T>(v.x, v.y);
}
template <typename T> __device__ __forceinline__ Cx<T> ld_cx(const Cx<T>* p) {
    typedef typename Vec2<T>::type V;
    V v = *reinterpret_cast<const V*>(p);
    return Cx<T>(v.x, v.y);
}
template <typename T> __device__ __forceinline__ void st_cx(Cx<T>* p, Cx<T> a) {
    typedef typename Vec2<T>::type V;
    V v; v.x = a.re; v.y = a.im;
    *reinterpret_cast<V*>(p) = v;
}

// Link traffic is streamed (each link is touched once per kernel): an L2 evict-first policy keeps the
// 126 MB L2 for the Delta field, which K1 -> K2 -> K3 -> K4 -> K5 hand to each other.
// LGF_STREAM_LINKS (compile-time, default 1) switches the hint off for A/B runs.
#ifndef LGF_STREAM_LINKS
#define LGF_STREAM_LINKS 1
#endif
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ Cx<double> ld_cx_stream(const Cx<double>* p, uint64_t pol) {
#if LGF_STREAM_LINKS
    double x, y;
    asm("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(x), "=d"(y) : "l"(p), "l"(pol));
    return Cx<double>(x, y);
#else
    return ld_cx(p);
#endif
}
__device__ __forceinline__ Cx<float> ld_cx_stream(const Cx<float>* p, uint64_t pol) {
#if LGF_STREAM_LINKS
    float x, y;
    asm("ld.global.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(x), "=f"(y) : "l"(p), "l"(pol));
    return Cx<float>(x, y);
#else
    return ld_cx(p);
#endif
}
__device__ __forceinline__ void st_cx_stream(Cx<double>* p, Cx<double> a, uint64_t pol) {
#if LGF_STREAM_LINKS
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(a.re), "d"(a.im), "l"(pol) : "memory");
#else
    st_cx(p, a);
#endif
}
__device__ __forceinline__ void st_cx_stream(Cx<float>* p, Cx<float> a, uint64_t pol) {
#if LGF_STREAM_LINKS
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(a.re), "f"(a.im), "l"(pol) : "memory");
#else
    st_cx(p, a);
#endif
}

// Programmatic dependent launch (sm_90+), first statement of every kernel of the iteration: wait until the kernel
// this one depends on has completed and its writes are visible, then let the NEXT kernel of the chain be
// scheduled as soon as every CTA of this one has started (its CTAs fill SMs as ours retire and block in their
// own wait).  Every kernel of the chain waits, so completion is transitive.  Both instructions are no-ops
// when the launch carries no programmatic dependency.
__device__ __forceinline__ void pdl_entry() {
    asm volatile("griddepcontrol.wait;" ::: "memory");
#ifndef LGF_PDL_NOTRIGGER
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}

// Stores of a field the NEXT kernel reads in full and that fits the L2 (Delta out of K1, Delta~ out of K4):
// evict-last, so that the links streaming through the same L2 do not push it out before it is consumed.
#ifndef LGF_KEEP_DELTA
#define LGF_KEEP_DELTA 1
#endif
__device__ __forceinline__ uint64_t l2_evict_last_policy() {
    uint64_t p;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
template <typename T> __device__ __forceinline__ void st_cx_keep(Cx<T>* p, Cx<T> a, uint64_t pol) {
#if LGF_KEEP_DELTA
    st_cx_stream(p, a, pol);      // same instruction, different policy operand
#else
    st_cx(p, a);
#endif
}

// 3x3 complex matrix in registers, row-major m[3*row + col]
template <typename T> struct Su3 { Cx<T> m[9]; };

// row 2 = conj(row0 x row1)   (third row rebuilt on the fly from the first two)
template <typename T> __device__ __forceinline__ void rebuild_row2(Su3<T>& u) {
    u.m[6] = cmulc(u.m[1], u.m[5]) - cmulc(u.m[2], u.m[4]);
    u.m[7] = cmulc(u.m[2], u.m[3]) - cmulc(u.m[0], u.m[5]);
    u.m[8] = cmulc(u.m[0], u.m[4]) - cmulc(u.m[1], u.m[3]);
}

// Row Gram-Schmidt on rows 0,1 in place, then row 2 = conj(row0 x row1)
// (north_star step 4 "reunitarise"; SURVEY.md §8(c) reading #9).
template <typename T> __device__ __forceinline__ void reunitarise(Su3<T>& g) {
    T n0 = norm2(g.m[0]) + norm2(g.m[1]) + norm2(g.m[2]);
    T i0 = rsqrt_t(n0);
#pragma unroll
    for (int j = 0; j < 3; ++j) g.m[j] = i0 * g.m[j];
    Cx<T> dot(0, 0);  // conj(r0) . r1
#pragma unroll
    for (int j = 0; j < 3; ++j) fma_cxc(dot, g.m[3 + j], g.m[j]);
#pragma unroll
    for (int j = 0; j < 3; ++j) g.m[3 + j] = g.m[3 + j] - dot * g.m[j];
    T n1 = norm2(g.m[3]) + norm2(g.m[4]) + norm2(g.m[5]);
    T i1 = rsqrt_t(n1);
#pragma unroll
    for (int j = 0; j < 3; ++j) g.m[3 + j] = i1 * g.m[3 + j];
    rebuild_row2(g);
}

// g = reunitarise(1 + (alpha/2) Dt) from the packed anti-Hermitian traceless field
// (c0 = D01, c1 = D02, c2 = D12, c3 = Im D00 + i Im D11); ha = alpha/2.
template <typename T>
__device__ __forceinline__ void build_g(Su3<T>& g, Cx<T> c0, Cx<T> c1, Cx<T> c2, Cx<T> c3, T ha) {
    const T d0 = c3.re, d1 = c3.im, d2 = -(c3.re + c3.im);
    g.m[0] = Cx<T>(T(1), ha * d0);
    g.m[1] = ha * c0;
    g.m[2] = ha * c1;
    g.m[3] = Cx<T>(-ha * c0.re, ha * c0.im);   // D10 = -conj(D01)
    g.m[4] = Cx<T>(T(1), ha * d1);
    g.m[5] = ha * c2;
    g.m[6] = Cx<T>(-ha * c1.re, ha * c1.im);
    g.m[7] = Cx<T>(-ha * c2.re, ha * c2.im);
    g.m[8] = Cx<T>(T(1), ha * d2);
    reunitarise(g);   // rows 0,1 orthonormalised; row 2 of the input is not used (rebuilt)
}

}  // namespace lgf
