// pwfs_dft.cuh -- small complex-FP32 DFTs held entirely in registers, written
// with Blackwell's packed FP32x2 instructions (FADD2 / FMUL2 / FFMA2).
//
// Dft<N, DIR>::run(x) replaces x[0..N) (natural order) by its unnormalised DFT
// X[k] = sum_n x[n] exp(DIR 2 pi i n k / N), DIR = -1 forward / +1 inverse, for
// any 2/3/5-smooth N.  DftP<N, DIR, NZ> is the same transform when x[NZ..N) is
// known to be zero at compile time (zero-padded input: those butterflies and
// twiddles are never emitted, and x[NZ..N) is never read).
//
// Everything is resolved at compile time: the recursion (decimation in time,
// radix 4 where possible, else 2, 3, 5), every array index and every twiddle, so
// after inlining the arrays live in registers and twiddles are immediates.
//
// A complex number is a float2 = one 64-bit register pair, so on sm_100a
//   complex add / sub / add of +-i*b          = 1 FADD2 (operand swap/negate modifiers)
//   complex * compile-time or run-time twiddle = 1 FMUL2 + 1 FFMA2
// i.e. half the issue slots of scalar code for the same FP32 pipe time.  These
// are the butterflies of steps a3/a5.
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
    if constexpr (N > 0) sfor_impl(f, std::make_integer_sequence<int, N>{});
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
__host__ __device__ constexpr int cdiv(int a, int b) { return (a + b - 1) / b; }
__host__ __device__ constexpr int imin(int a, int b) { return a < b ? a : b; }
__host__ __device__ constexpr int imax(int a, int b) { return a > b ? a : b; }
}  // namespace ct

// ----------------------------------------------------- complex primitives ---
__device__ __forceinline__ float2 bc(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// a + DIR*i*b  and  a - DIR*i*b   (one FADD2 each: swapped halves, one negated)
template <int DIR>
__device__ __forceinline__ float2 cadd_i(float2 a, float2 b) {
    if constexpr (DIR > 0) return __fadd2_rn(a, make_float2(-b.y, b.x));
    else return __fadd2_rn(a, make_float2(b.y, -b.x));
}
template <int DIR>
__device__ __forceinline__ float2 csub_i(float2 a, float2 b) { return cadd_i<-DIR>(a, b); }
// a * w, run-time w:  t = a.y*(w.y, w.x);  r = a.x*w + (-t.x, t.y)      (FMUL2 + FFMA2)
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    const float2 t = __fmul2_rn(bc(a.y), make_float2(w.y, w.x));
    return __ffma2_rn(bc(a.x), w, make_float2(-t.x, t.y));
}
// a * conj(w) = w.x*a + w.y*(a.y, -a.x):  t = w.y*(a.y, a.x);  r = w.x*a + (t.x, -t.y)
__device__ __forceinline__ float2 cmulc(float2 a, float2 w) {
    const float2 t = __fmul2_rn(bc(w.y), make_float2(a.y, a.x));
    return __ffma2_rn(bc(w.x), a, make_float2(t.x, -t.y));
}
// a * (c + i s) with compile-time c, s:  c*a + s*(-a.y, a.x)             (FMUL2 + FFMA2, immediates)
__device__ __forceinline__ float2 cmul_const(float2 a, float c, float s) {
    return __ffma2_rn(bc(c), a, __fmul2_rn(bc(s), make_float2(-a.y, a.x)));
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
    } else if constexpr ((8 * num) % DEN == 0) {      // (+-1 +- i)/sqrt2: one FADD2 + one FMUL2
        constexpr float h = 0.70710678118654752440f;
        // (1+i)a = a + i a ; (-1+i)a = -(a - i a) ; (-1-i)a = -(a + i a) ; (1-i)a = a - i a
        if constexpr (c > 0 && s > 0) return __fmul2_rn(__fadd2_rn(a, make_float2(-a.y, a.x)), bc(h));
        else if constexpr (c < 0 && s > 0) return __fmul2_rn(__fadd2_rn(a, make_float2(a.y, -a.x)), bc(-h));
        else if constexpr (c < 0 && s < 0) return __fmul2_rn(__fadd2_rn(a, make_float2(-a.y, a.x)), bc(-h));
        else return __fmul2_rn(__fadd2_rn(a, make_float2(a.y, -a.x)), bc(h));
    } else {
        return cmul_const(a, c, s);
    }
}

// ------------------------------------------ twiddles in "1 + i tau" form -----
// A twiddle multiply followed by the butterfly's add/sub costs FMUL2 + FFMA2 + FADD2.
// Writing w = sigma * i^rot * (1 + i tau), |tau| <= 1 (rot = nearest quadrant, sigma = cos,
// tau = tan of the remainder), the product splits into
//     u = y + i tau y          one FFMA2 (none for tau = 0, one FADD2 for tau = +-1),
//     i^rot                    operand swap/negate modifiers, no instruction,
//     sigma                    a real scale that the NEXT add absorbs: a + sigma*u is one FFMA2
// (Linzer-Feig style scaling).  So a non-trivial twiddle costs one packed instruction
// instead of two; the butterflies below take the pending scales of their inputs as a
// compile-time set S (S::s(p) = scale of input p, S::s(0) = 1).
namespace ct {
struct lf { double sigma; int rot; double tau; };
__host__ __device__ constexpr lf lf_of(long long num, long long den) {
    num = pmod(num, den);
    long long q = (8 * num + den) / (2 * den);
    double r = (double)(4 * num - q * den) / (double)(4 * den);
    double a = 2.0 * kPi * r;
    bool exact = (4 * num == q * den);
    double c = exact ? 1.0 : cos_poly(a);
    double s = exact ? 0.0 : sin_poly(a);
    return {c, (int)(q & 3), s / c};
}
}  // namespace ct

struct OneS { __host__ __device__ static constexpr float s(int) { return 1.f; } };
// scales of the inputs t[p] = W_N^{DIR p q} y[p] of combine step q
template <int N, int Q_, int DIR>
struct TwS {
    __host__ __device__ static constexpr float s(int p) { return (float)ct::lf_of((long long)DIR * p * Q_, N).sigma; }
};

template <int E>
__device__ __forceinline__ float2 rot_i(float2 a) {      // a * i^E
    if constexpr ((E & 3) == 0) return a;
    else if constexpr ((E & 3) == 1) return make_float2(-a.y, a.x);
    else if constexpr ((E & 3) == 2) return make_float2(-a.x, -a.y);
    else return make_float2(a.y, -a.x);
}
// i^rot (y + i tau y) for w = exp(DIR 2 pi i NUM/DEN); the factor sigma stays pending
template <int NUM, int DEN, int DIR>
__device__ __forceinline__ float2 lf_pre(float2 y) {
    constexpr ct::lf w = ct::lf_of((long long)DIR * NUM, DEN);
    constexpr float tau = (float)w.tau;
    float2 u;
    if constexpr (tau == 0.f) u = y;
    else if constexpr (tau == 1.f) u = __fadd2_rn(y, make_float2(-y.y, y.x));
    else if constexpr (tau == -1.f) u = __fadd2_rn(y, make_float2(y.y, -y.x));
    else u = __ffma2_rn(bc(tau), make_float2(-y.y, y.x), y);
    return rot_i<w.rot>(u);
}
// a + c*b, compile-time real c
#define PWK_AXPY(c, b, a) (((c) == 1.f) ? __fadd2_rn((a), (b)) : ((c) == -1.f) ? __fadd2_rn((a), make_float2(-(b).x, -(b).y)) : __ffma2_rn(bc(c), (b), (a)))

// ------------------------------------------------- prime-size butterflies ---
// Bfly<P, DIR, PZ>::run<S>: DFT of size P of the inputs S::s(p) * x[p]; x[PZ..P) are zero
// (never read).
template <int P, int DIR, int PZ>
struct Bfly;

template <int DIR, int PZ>
struct Bfly<2, DIR, PZ> {
    template <class S = OneS>
    __device__ __forceinline__ static void run(float2 (&x)[2]) {
        constexpr float s1 = S::s(1);
        if constexpr (PZ >= 2) {
            const float2 a = x[0], b = x[1];
            x[0] = PWK_AXPY(s1, b, a);
            x[1] = PWK_AXPY(-s1, b, a);
        } else {
            x[1] = x[0];
        }
    }
};

template <int DIR, int PZ>
struct Bfly<3, DIR, PZ> {
    template <class S = OneS>
    __device__ __forceinline__ static void run(float2 (&x)[3]) {
        constexpr float s60 = 0.86602540378443864676f * (float)DIR;
        constexpr float s1 = S::s(1);
        if constexpr (PZ == 1) {
            x[1] = x[0]; x[2] = x[0];
        } else {
            const float2 a = x[0];
            float2 t = x[1], u = x[1];                 // true values carry s1
            if constexpr (PZ >= 3) {
                constexpr float r = S::s(2) / s1;
                t = PWK_AXPY(r, x[2], x[1]);
                u = PWK_AXPY(-r, x[2], x[1]);
            }
            x[0] = PWK_AXPY(s1, t, a);
            const float2 m = __ffma2_rn(bc(-0.5f * s1), t, a);
            const float2 iu = make_float2(-u.y, u.x);
            x[1] = __ffma2_rn(bc(s60 * s1), iu, m);      // m + i DIR s u
            x[2] = __ffma2_rn(bc(-s60 * s1), iu, m);     // m - i DIR s u
        }
    }
};

template <int DIR, int PZ>
struct Bfly<4, DIR, PZ> {
    template <class S = OneS>
    __device__ __forceinline__ static void run(float2 (&x)[4]) {
        constexpr float s1 = S::s(1);
        if constexpr (PZ == 1) {
            x[1] = x[0]; x[2] = x[0]; x[3] = x[0];
        } else if constexpr (PZ == 2) {             // X_j = a + w^j s1 b, w = DIR i
            const float2 a = x[0], b = x[1], ib = rot_i<DIR>(x[1]);
            x[0] = PWK_AXPY(s1, b, a);
            x[1] = PWK_AXPY(s1, ib, a);
            x[2] = PWK_AXPY(-s1, b, a);
            x[3] = PWK_AXPY(-s1, ib, a);
        } else {
            constexpr float s2 = S::s(2);
            const float2 t0 = PWK_AXPY(s2, x[2], x[0]), t1 = PWK_AXPY(-s2, x[2], x[0]);
            float2 t2 = x[1], t3 = x[1];                // true values carry s1
            if constexpr (PZ >= 4) {
                constexpr float r = S::s(3) / s1;
                t2 = PWK_AXPY(r, x[3], x[1]);
                t3 = PWK_AXPY(-r, x[3], x[1]);
            }
            const float2 it3 = rot_i<DIR>(t3);
            x[0] = PWK_AXPY(s1, t2, t0);
            x[1] = PWK_AXPY(s1, it3, t1);
            x[2] = PWK_AXPY(-s1, t2, t0);
            x[3] = PWK_AXPY(-s1, it3, t1);
        }
    }
};

template <int DIR, int PZ>
struct Bfly<5, DIR, PZ> {
    template <class S = OneS>
    __device__ __forceinline__ static void run(float2 (&x)[5]) {
        constexpr float c1 = 0.30901699437494742410f;    // cos 72
        constexpr float c2 = -0.80901699437494742410f;   // cos 144
        constexpr float s1 = 0.95105651629515357212f * (float)DIR;   // sin 72
        constexpr float s2 = 0.58778525229247312917f * (float)DIR;   // sin 144
        constexpr float g1 = S::s(1);                    // pending scale of x[1] (and of t1, t3)
        if constexpr (PZ == 1) {
            x[1] = x[0]; x[2] = x[0]; x[3] = x[0]; x[4] = x[0];
        } else {
            const float2 a = x[0];
            float2 t1 = x[1], t3 = x[1];
            if constexpr (PZ >= 5) {
                constexpr float r = S::s(4) / g1;
                t1 = PWK_AXPY(r, x[4], x[1]);
                t3 = PWK_AXPY(-r, x[4], x[1]);
            }
            float2 m1 = __ffma2_rn(bc(c1 * g1), t1, a), m2 = __ffma2_rn(bc(c2 * g1), t1, a);
            float2 n1 = __fmul2_rn(bc(s1 * g1), t3), n2 = __fmul2_rn(bc(s2 * g1), t3);
            float2 x0 = PWK_AXPY(g1, t1, a);
            if constexpr (PZ >= 3) {
                constexpr float g2 = S::s(2);            // pending scale of x[2] (and of t2, t4)
                float2 t2 = x[2], t4 = x[2];
                if constexpr (PZ >= 4) {
                    constexpr float r = S::s(3) / g2;
                    t2 = PWK_AXPY(r, x[3], x[2]);
                    t4 = PWK_AXPY(-r, x[3], x[2]);
                }
                x0 = PWK_AXPY(g2, t2, x0);
                m1 = __ffma2_rn(bc(c2 * g2), t2, m1);
                m2 = __ffma2_rn(bc(c1 * g2), t2, m2);
                n1 = __ffma2_rn(bc(s2 * g2), t4, n1);
                n2 = __ffma2_rn(bc(-s1 * g2), t4, n2);
            }
            // X1 = m1 + i n1, X4 = m1 - i n1, X2 = m2 + i n2, X3 = m2 - i n2  (DIR folded in s1, s2)
            x[0] = x0;
            x[1] = cadd_i<1>(m1, n1);
            x[4] = csub_i<1>(m1, n1);
            x[2] = cadd_i<1>(m2, n2);
            x[3] = csub_i<1>(m2, n2);
        }
    }
};

// ------------------------------------------------------ composite lengths ---
// N = P*Q, decimation in time:
//   Y_p = DFT_Q( x[P q' + p] ),  X[q + Q j] = sum_p W_P^{p j} ( W_N^{p q} Y_p[q] ).
// With x[NZ..N) = 0 sub-sequence p has ceil((NZ-p)/P) leading non-zeros and only
// the first min(P, NZ) sub-sequences are non-zero at all.
template <int N, int DIR, int NZ>
struct DftP {
    static_assert(NZ >= 1 && NZ <= N, "DftP: 1 <= NZ <= N");
    static constexpr int P = (N % 4 == 0) ? 4 : (N % 2 == 0) ? 2 : (N % 3 == 0) ? 3 : 5;
    static constexpr int Q = N / P;
    static_assert(N == 1 || N % P == 0, "DftP: length must be 2/3/5-smooth");
    static constexpr int PZ = ct::imin(P, NZ);

    __device__ __forceinline__ static void run(float2 (&x)[N]) {
        if constexpr (N == 1) {
        } else if constexpr (NZ == 1) {              // DFT of a delta at 0 is constant
            sfor<N - 1>([&](auto ic) { x[decltype(ic)::value + 1] = x[0]; });
        } else if constexpr (Q == 1) {
            Bfly<P, DIR, PZ>::template run<OneS>(x);
        } else {
            float2 y[P][Q];
            sfor<PZ>([&](auto pc) {
                constexpr int p = decltype(pc)::value;
                constexpr int NZp = ct::cdiv(NZ - p, P);
                float2 sub[Q];
                sfor<NZp>([&](auto qc) { constexpr int q = decltype(qc)::value; sub[q] = x[P * q + p]; });
                DftP<Q, DIR, NZp>::run(sub);
                sfor<Q>([&](auto qc) { constexpr int q = decltype(qc)::value; y[p][q] = sub[q]; });
            });
            sfor<Q>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                float2 t[P];
                sfor<PZ>([&](auto pc) {
                    constexpr int p = decltype(pc)::value;
                    t[p] = lf_pre<p * q, N, DIR>(y[p][q]);
                });
                Bfly<P, DIR, PZ>::template run<TwS<N, q, DIR>>(t);
                sfor<P>([&](auto jc) { constexpr int j = decltype(jc)::value; x[q + Q * j] = t[j]; });
            });
        }
    }
};

template <int N, int DIR>
struct Dft {
    __device__ __forceinline__ static void run(float2 (&x)[N]) { DftP<N, DIR, N>::run(x); }
};

}  // namespace pwk
