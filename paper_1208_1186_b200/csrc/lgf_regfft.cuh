// lgf_regfft.cuh -- small DFTs done entirely in registers with compile-time twiddles.
// RegFft<R, SIGN, T>::run(v): in-place DFT of v[0..R-1], natural order in and out,
//   out[k] = sum_n v[n] exp(SIGN * 2 pi i n k / R),   R = 2^a 3^b (R <= 64).
// Built by compile-time Cooley-Tukey recursion (radix 4, 2, 3); every twiddle is a literal folded
// into the instruction stream, trivial ones (1, +-i, (+-1 +- i)/sqrt 2) cost no multiplies.
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <type_traits>

#include "lgf_math.cuh"

namespace lgf {

// ---- compile-time cos/sin of 2 pi k / n (exact integer octant reduction + Taylor on [0, pi/4]) ----
namespace ct {
constexpr double kPi = 3.14159265358979323846264338327950288;
__host__ __device__ constexpr double taylor_sin(double x) {
    const double x2 = x * x;
    double term = x, sum = x;
    for (int i = 1; i <= 12; ++i) { term *= -x2 / double((2 * i) * (2 * i + 1)); sum += term; }
    return sum;
}
__host__ __device__ constexpr double taylor_cos(double x) {
    const double x2 = x * x;
    double term = 1.0, sum = 1.0;
    for (int i = 1; i <= 12; ++i) { term *= -x2 / double((2 * i - 1) * (2 * i)); sum += term; }
    return sum;
}
// angle = 2 pi k / n with 0 <= k < n; work in units of 1/(8n) turns to split octants exactly
__host__ __device__ constexpr double cos2pi(long long k, long long n) {
    k %= n; if (k < 0) k += n;
    // symmetry: cos(2pi k/n) = cos(2pi (n-k)/n)
    if (2 * k > n) k = n - k;                 // now 0 <= angle <= pi
    if (4 * k > n) return -cos2pi(n - 2 * k, 2 * n) ;   // cos(a) = -cos(pi - a): pi - a = 2pi (n-2k)/(2n)
    // 0 <= angle <= pi/2
    if (8 * k > n) {                           // pi/4 < a <= pi/2: cos(a) = sin(pi/2 - a), pi/2 - a = 2pi (n-4k)/(4n)
        return taylor_sin(2.0 * kPi * double(n - 4 * k) / double(4 * n));
    }
    return taylor_cos(2.0 * kPi * double(k) / double(n));
}
__host__ __device__ constexpr double sin2pi(long long k, long long n) {
    // sin(a) = cos(a - pi/2) = cos(2pi (4k - n) / (4n))
    return cos2pi(4 * k - n, 4 * n);
}
}  // namespace ct

template <int I, int N, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// a *= exp(SIGN * 2 pi i K / R)
template <int K, int R, int SIGN, typename T>
__device__ __forceinline__ Cx<T> mul_tw(Cx<T> a) {
    constexpr int k = ((K % R) + R) % R;
    if constexpr (k == 0) {
        return a;
    } else if constexpr (2 * k == R) {
        return Cx<T>(-a.re, -a.im);
    } else if constexpr (4 * k == R) {           // exp(SIGN i pi/2) = SIGN * i
        return SIGN > 0 ? mul_i(a) : mul_mi(a);
    } else if constexpr (4 * k == 3 * R) {       // exp(SIGN i 3pi/2) = -SIGN * i
        return SIGN > 0 ? mul_mi(a) : mul_i(a);
    } else if constexpr ((8 * k) % R == 0) {     // odd multiples of pi/4: (+-1 +- i)/sqrt2
        constexpr double c = ct::cos2pi(k, R), s = SIGN * ct::sin2pi(k, R);
        const T h = T(0.70710678118654752440084436210485);
        // (c + i s)(re + i im), |c| = |s| = h
        const T p = (c > 0 ? a.re : -a.re), q = (s > 0 ? a.im : -a.im);   // c*re/h, s*im/h
        const T u = (c > 0 ? a.im : -a.im), w = (s > 0 ? a.re : -a.re);   // c*im/h, s*re/h
        return Cx<T>(h * (p - q), h * (u + w));
    } else {
        constexpr double c = ct::cos2pi(k, R), s = SIGN * ct::sin2pi(k, R);
        return Cx<T>(a.re * T(c) - a.im * T(s), a.re * T(s) + a.im * T(c));
    }
}

template <int R, int SIGN, typename T> struct RegFft;

template <int SIGN, typename T> struct RegFft<1, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>*) {}
};
template <int SIGN, typename T> struct RegFft<2, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const Cx<T> a = v[0] + v[1], b = v[0] - v[1];
        v[0] = a; v[1] = b;
    }
};
template <int SIGN, typename T> struct RegFft<3, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const T h = T(0.86602540378443864676372317075294);  // sqrt(3)/2
        const Cx<T> t = v[1] + v[2];
        const Cx<T> m(v[0].re - T(0.5) * t.re, v[0].im - T(0.5) * t.im);
        const Cx<T> d = h * (v[1] - v[2]);
        const Cx<T> s = SIGN > 0 ? mul_i(d) : mul_mi(d);
        v[0] = v[0] + t; v[1] = m + s; v[2] = m - s;
    }
};
template <int SIGN, typename T> struct RegFft<4, SIGN, T> {
    __device__ static __forceinline__ void run(Cx<T>* v) {
        const Cx<T> b0 = v[0] + v[2], b1 = v[0] - v[2], b2 = v[1] + v[3];
        const Cx<T> d = v[1] - v[3];
        const Cx<T> b3 = SIGN > 0 ? mul_i(d) : mul_mi(d);
        v[0] = b0 + b2; v[2] = b0 - b2; v[1] = b1 + b3; v[3] = b1 - b3;
    }
};

// generic R = P * M, P = radix (4, 2 or 3): decimation in time
//   sub_r[j] = v[r + P j] (j < M) -> DFT_M -> S_r[kb];  out[kb + M ka] = DFT_P over r of (w_R^{r kb} S_r[kb]) at ka
template <int R, int SIGN, typename T> struct RegFft {
    static constexpr int P = (R % 4 == 0) ? 4 : ((R % 2 == 0) ? 2 : 3);
    static constexpr int M = R / P;
    static_assert(R % P == 0 && R > 4, "RegFft: R must be 2^a 3^b");
    __device__ static __forceinline__ void run(Cx<T>* v) {
        Cx<T> sub[P][M];
        static_for<0, P>([&](auto r) {
            static_for<0, M>([&](auto j) { sub[r.value][j.value] = v[r.value + P * j.value]; });
            RegFft<M, SIGN, T>::run(sub[r.value]);
        });
        static_for<0, M>([&](auto kb) {
            Cx<T> t[P];
            static_for<0, P>([&](auto r) { t[r.value] = mul_tw<r.value * kb.value, R, SIGN>(sub[r.value][kb.value]); });
            RegFft<P, SIGN, T>::run(t);
            static_for<0, P>([&](auto ka) { v[kb.value + M * ka.value] = t[ka.value]; });
        });
    }
};

}  // namespace lgf
