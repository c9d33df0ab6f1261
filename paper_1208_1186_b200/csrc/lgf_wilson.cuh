// lgf_wilson.cuh -- the step after the path: temporal Wilson lines and the singlet
// correlator of eq. (1), on the links the context holds (normally the gauge-fixed ones):
//     W(x) = U_t(x,0) U_t(x,1) ... U_t(x,Lt-1)          (ordered product of the t-links at spatial site x)
//     C(r) = (1/(3 Vs)) sum_x Tr[ W(x + r) W(x)^+ ]      (average over the spatial lattice, Vs = Lx Ly Lz)
// C is a sum of nine autocorrelations (one per matrix element), evaluated through the correlation theorem:
//     sum_x f(x + r) conj f(x) = (1/Vs) sum_k |F(k)|^2 exp(+2 pi i k.r/L),   F = unnormalised forward DFT of f,
// with the (x,y) transforms done by the runtime-radix plane kernel of lgf_fft.cuh (any 2^a 3^b extents) and the z
// transforms as direct sums over the line (Lz <= 4096 terms from the exact root table): this runs once per
// configuration, after hundreds of gauge-fixing iterations, so it is written for clarity, not for the roofline.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include "lgf_site.cuh"

namespace lgf {

// W[c][xs], c = 0..8 row-major matrix element, xs = x + Lx (y + Ly z): one thread per spatial site walks along t.
template <typename T, int NC>
__global__ void __launch_bounds__(128)
k_wilson_lines(const Cx<T>* __restrict__ U, Cx<T>* __restrict__ W, long long V, long long Vs, int Lt) {
    const long long xs = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (xs >= Vs) return;
    Su3<T> w;
    load_link<T, NC>(w, U, V, 3, xs);
    for (int t = 1; t < Lt; ++t) {
        Su3<T> u, p;
        load_link<T, NC>(u, U, V, 3, xs + Vs * t);
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                Cx<T> acc = w.m[3 * i] * u.m[j];
                fma_cx(acc, w.m[3 * i + 1], u.m[3 + j]);
                fma_cx(acc, w.m[3 * i + 2], u.m[6 + j]);
                p.m[3 * i + j] = acc;
            }
        w = p;
    }
#pragma unroll
    for (int c = 0; c < 9; ++c) st_cx(W + (size_t)c * Vs + xs, w.m[c]);
}

// P(kx, ky, kz) = sum_c | sum_z F_c(kx, ky, z) exp(-2 pi i kz z / Lz) |^2 : thread per (kxy, kz); F_c are the nine fields
// after the forward (x,y) transform.  tw[j] = exp(-2 pi i j / Lz).  Stored as a complex field with zero imaginary part.
template <typename T>
__global__ void __launch_bounds__(128)
k_z_power(const Cx<T>* __restrict__ F, Cx<T>* __restrict__ P, const Cx<T>* __restrict__ tw, long long LxLy, int Lz) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= LxLy * Lz) return;
    const int kz = (int)(i / LxLy);
    const long long q = i - (long long)kz * LxLy;
    const long long Vs = LxLy * Lz;
    T pw = 0;
    for (int c = 0; c < 9; ++c) {
        Cx<T> acc(0, 0);
        int j = 0;                                             // (kz * z) mod Lz, kept by addition
        for (int z = 0; z < Lz; ++z) {
            fma_cx(acc, ld_cx(F + (size_t)c * Vs + (size_t)z * LxLy + q), ldg_cx(tw + j));
            j += kz;
            if (j >= Lz) j -= Lz;
        }
        pw += norm2(acc);
    }
    st_cx(P + i, Cx<T>(pw, T(0)));
}

// G(kx, ky, z) = sum_kz P(kx, ky, kz) exp(+2 pi i kz z / Lz); twi[j] = exp(+2 pi i j / Lz).
template <typename T>
__global__ void __launch_bounds__(128)
k_z_inverse(const Cx<T>* __restrict__ P, Cx<T>* __restrict__ G, const Cx<T>* __restrict__ twi, long long LxLy, int Lz) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= LxLy * Lz) return;
    const int z = (int)(i / LxLy);
    const long long q = i - (long long)z * LxLy;
    Cx<T> acc(0, 0);
    int j = 0;
    for (int kz = 0; kz < Lz; ++kz) {
        const T p = ld_cx(P + (size_t)kz * LxLy + q).re;
        const Cx<T> w = ldg_cx(twi + j);
        acc.re += p * w.re;
        acc.im += p * w.im;
        j += z;
        if (j >= Lz) j -= Lz;
    }
    st_cx(G + i, acc);
}

// C(r) = G(r) / (3 Vs^2) after the inverse (x,y) transform of G
template <typename T>
__global__ void k_corr_scale(const Cx<T>* __restrict__ G, Cx<T>* __restrict__ C, long long Vs, T scale) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vs) return;
    const Cx<T> g = ld_cx(G + i);
    st_cx(C + i, Cx<T>(scale * g.re, scale * g.im));
}

// W[c][xs] -> [xs][3][3] (the boundary layout of lgf_wilson_lines)
template <typename T>
__global__ void k_lines_to_aos(const Cx<T>* __restrict__ W, Cx<T>* __restrict__ out, long long Vs) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Vs * 9) return;
    const long long xs = i / 9;
    const int c = (int)(i - xs * 9);
    out[i] = W[(size_t)c * Vs + xs];
}

}  // namespace lgf
