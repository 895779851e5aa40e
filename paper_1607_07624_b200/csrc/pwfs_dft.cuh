// pwfs_dft.cuh -- small complex-FP32 DFTs held entirely in registers.
//
// Dft<N, DIR>::run(x) replaces x[0..N) (natural order) by its unnormalised DFT
// X[k] = sum_n x[n] exp(DIR 2 pi i n k / N), DIR = -1 forward / +1 inverse, for
// any 2/3/5-smooth N.  Everything is resolved at compile time: the recursion
// (decimation in time, radix 4 where possible, else 2, 3, 5), every array index
// and every twiddle factor, so after inlining the arrays live in registers and
// twiddles are FMA immediates.  Trivial twiddles (1, -1, +-i, (+-1+-i)/sqrt2)
// cost no multiply.  These are the butterflies of steps a3/a5.
#pragma once
#include <cuda_runtime.h>
#include <utility>

namespace pwk {

// ------------------------------------------------------------ static loops --
template <typename F, int... Is>
__device__ __forceinline__ void sfor_impl(F &&f, std::integer_sequence<int, Is...>) {
    (f(std::integral_constant<int, Is>{}), ...);
}
template <int N, typename F>
__device__ __forceinline__ void sfor(F &&f) {
    sfor_impl(f, std::make_integer_sequence<int, N>{});
}

// ------------------------------------------------- compile-time cos / sin ---
// cos(2 pi num/den), sin(2 pi num/den) in double by quadrant reduction (exact in
// integers) and Taylor series on |a| <= pi/4.
namespace ct {
constexpr double kPi = 3.141592653589793238462643383279502884;
__host__ __device__ constexpr double sin_poly(double a) {
    double a2 = a * a, term = a, sum = a;
    for (int i = 1; i < 14; ++i) { term *= -a2 / ((2.0 * i) * (2.0 * i + 1.0)); sum += term; }
    return sum;
}
__host__ __device__ constexpr double cos_poly(double a) {
    double a2 = a * a, term = 1.0, sum = 1.0;
    for (int i = 1; i < 14; ++i) { term *= -a2 / ((2.0 * i - 1.0) * (2.0 * i)); sum += term; }
    return sum;
}
__host__ __device__ constexpr long long pmod(long long a, long long m) { return ((a % m) + m) % m; }
struct cs { double c, s; };
__host__ __device__ constexpr cs cossin2pi(long long num, long long den) {
    num = pmod(num, den);
    // quadrant q = round(4 num/den); remainder r = num/den - q/4 in turns, |r| <= 1/8
    long long q = (8 * num + den) / (2 * den);
    double r = (double)(4 * num - q * den) / (double)(4 * den);
    double a = 2.0 * kPi * r;
    double c = (4 * num == q * den) ? 1.0 : cos_poly(a);
    double s = (4 * num == q * den) ? 0.0 : sin_poly(a);
    switch (q & 3) {
        case 0: return {c, s};
        case 1: return {-s, c};
        case 2: return {-c, -s};
        default: return {s, -c};
    }
}
}  // namespace ct

// ----------------------------------------------------- complex primitives ---
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    return make_float2(fmaf(-a.y, w.y, a.x * w.x), fmaf(a.y, w.x, a.x * w.y));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {  // a * conj(w)
    return make_float2(fmaf(a.y, w.y, a.x * w.x), fmaf(a.y, w.x, -a.x * w.y));
}
// multiply by DIR*i
template <int DIR>
__device__ __forceinline__ float2 mul_i(float2 a) {
    if constexpr (DIR > 0) return make_float2(-a.y, a.x);
    else return make_float2(a.y, -a.x);
}

// a * exp(DIR 2 pi i NUM/DEN) with the constant folded at compile time.
template <int NUM, int DEN, int DIR>
__device__ __forceinline__ float2 mul_w(float2 a) {
    constexpr ct::cs w = ct::cossin2pi((long long)DIR * NUM, DEN);
    constexpr float c = (float)w.c;
    constexpr float s = (float)w.s;
    constexpr int num = (int)ct::pmod((long long)DIR * NUM, DEN);
    if constexpr (num == 0) {
        return a;
    } else if constexpr (2 * num == DEN) {
        return make_float2(-a.x, -a.y);
    } else if constexpr (4 * num == DEN) {            // +i
        return make_float2(-a.y, a.x);
    } else if constexpr (4 * num == 3 * DEN) {        // -i
        return make_float2(a.y, -a.x);
    } else if constexpr ((8 * num) % DEN == 0) {      // (+-1 +- i)/sqrt2
        constexpr float h = 0.70710678118654752440f;
        if constexpr (c > 0 && s > 0) return make_float2((a.x - a.y) * h, (a.x + a.y) * h);
        else if constexpr (c < 0 && s > 0) return make_float2((-a.x - a.y) * h, (a.x - a.y) * h);
        else if constexpr (c < 0 && s < 0) return make_float2((a.y - a.x) * h, (-a.x - a.y) * h);
        else return make_float2((a.x + a.y) * h, (a.y - a.x) * h);
    } else {
        return make_float2(fmaf(-s, a.y, c * a.x), fmaf(s, a.x, c * a.y));
    }
}

// ------------------------------------------------------------- butterflies --
template <int N, int DIR>
struct Dft;

template <int DIR>
struct Dft<1, DIR> {
    __device__ __forceinline__ static void run(float2 (&)[1]) {}
};

template <int DIR>
struct Dft<2, DIR> {
    __device__ __forceinline__ static void run(float2 (&x)[2]) {
        float2 a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
};

template <int DIR>
struct Dft<3, DIR> {
    __device__ __forceinline__ static void run(float2 (&x)[3]) {
        constexpr float s60 = 0.86602540378443864676f * (float)DIR;
        float2 a = x[0], b = x[1], c = x[2];
        float2 t = cadd(b, c), u = csub(b, c);
        x[0] = cadd(a, t);
        float2 m = make_float2(fmaf(-0.5f, t.x, a.x), fmaf(-0.5f, t.y, a.y));
        // X1 = m + i*DIR*s*u,  X2 = m - i*DIR*s*u
        x[1] = make_float2(fmaf(-s60, u.y, m.x), fmaf(s60, u.x, m.y));
        x[2] = make_float2(fmaf(s60, u.y, m.x), fmaf(-s60, u.x, m.y));
    }
};

template <int DIR>
struct Dft<4, DIR> {
    __device__ __forceinline__ static void run(float2 (&x)[4]) {
        float2 t0 = cadd(x[0], x[2]), t1 = csub(x[0], x[2]);
        float2 t2 = cadd(x[1], x[3]), t3 = mul_i<DIR>(csub(x[1], x[3]));
        x[0] = cadd(t0, t2);
        x[1] = cadd(t1, t3);
        x[2] = csub(t0, t2);
        x[3] = csub(t1, t3);
    }
};

template <int DIR>
struct Dft<5, DIR> {
    __device__ __forceinline__ static void run(float2 (&x)[5]) {
        constexpr float c1 = 0.30901699437494742410f;    // cos 72
        constexpr float c2 = -0.80901699437494742410f;   // cos 144
        constexpr float s1 = 0.95105651629515357212f * (float)DIR;   // sin 72
        constexpr float s2 = 0.58778525229247312917f * (float)DIR;   // sin 144
        float2 a = x[0];
        float2 t1 = cadd(x[1], x[4]), t2 = cadd(x[2], x[3]);
        float2 t3 = csub(x[1], x[4]), t4 = csub(x[2], x[3]);
        x[0] = cadd(a, cadd(t1, t2));
        float2 m1 = make_float2(fmaf(c2, t2.x, fmaf(c1, t1.x, a.x)), fmaf(c2, t2.y, fmaf(c1, t1.y, a.y)));
        float2 m2 = make_float2(fmaf(c1, t2.x, fmaf(c2, t1.x, a.x)), fmaf(c1, t2.y, fmaf(c2, t1.y, a.y)));
        float2 n1 = make_float2(fmaf(s2, t4.x, s1 * t3.x), fmaf(s2, t4.y, s1 * t3.y));
        float2 n2 = make_float2(fmaf(-s1, t4.x, s2 * t3.x), fmaf(-s1, t4.y, s2 * t3.y));
        // X1 = m1 + i n1, X4 = m1 - i n1, X2 = m2 + i n2, X3 = m2 - i n2  (DIR folded in s1, s2)
        x[1] = make_float2(m1.x - n1.y, m1.y + n1.x);
        x[4] = make_float2(m1.x + n1.y, m1.y - n1.x);
        x[2] = make_float2(m2.x - n2.y, m2.y + n2.x);
        x[3] = make_float2(m2.x + n2.y, m2.y - n2.x);
    }
};

// Composite N = P*Q, decimation in time:
//   Y_p = DFT_Q( x[P q' + p] ),  X[q + Q j] = sum_p W_P^{p j} ( W_N^{p q} Y_p[q] ).
template <int N, int DIR>
struct Dft {
    static constexpr int P = (N % 4 == 0) ? 4 : (N % 2 == 0) ? 2 : (N % 3 == 0) ? 3 : 5;
    static constexpr int Q = N / P;
    static_assert(N % P == 0 && Q >= 1, "Dft: length must be 2/3/5-smooth");
    __device__ __forceinline__ static void run(float2 (&x)[N]) {
        float2 y[P][Q];
        sfor<P>([&](auto pc) {
            constexpr int p = decltype(pc)::value;
            float2 sub[Q];
            sfor<Q>([&](auto qc) { constexpr int q = decltype(qc)::value; sub[q] = x[P * q + p]; });
            Dft<Q, DIR>::run(sub);
            sfor<Q>([&](auto qc) { constexpr int q = decltype(qc)::value; y[p][q] = sub[q]; });
        });
        sfor<Q>([&](auto qc) {
            constexpr int q = decltype(qc)::value;
            float2 t[P];
            sfor<P>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                t[p] = mul_w<p * q, N, DIR>(y[p][q]);
            });
            Dft<P, DIR>::run(t);
            sfor<P>([&](auto jc) { constexpr int j = decltype(jc)::value; x[q + Q * j] = t[j]; });
        });
    }
};

}  // namespace pwk
