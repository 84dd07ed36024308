// lgf_cplx.cuh -- complex scalar type, compile-time loops and compile-time twiddle factors.
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <type_traits>

namespace lgf {

// Complex number, 2*sizeof(R) aligned so that one element is one 8-byte (fp32) or 16-byte (fp64)
// vector load/store.
template <class R>
struct alignas(2 * sizeof(R)) C {
    R x, y;
};

template <class R> __host__ __device__ __forceinline__ C<R> mk(R x, R y) { C<R> r; r.x = x; r.y = y; return r; }
template <class R> __host__ __device__ __forceinline__ C<R> operator+(C<R> a, C<R> b) { return mk<R>(a.x + b.x, a.y + b.y); }
template <class R> __host__ __device__ __forceinline__ C<R> operator-(C<R> a, C<R> b) { return mk<R>(a.x - b.x, a.y - b.y); }
// Single precision on sm_100: complex add / subtract as ONE packed instruction (FADD2 / FFMA2, add.f32x2 / fma.rn.f32x2) --
// the real and imaginary parts already sit in adjacent registers.  Each lane rounds to nearest like the scalar
// instruction, so the results are the scalar ones bit for bit; what it buys is issue slots: the fp32 FFT sweeps are
// issue-bound (ncu: 47-61 % of the issue slots, FMA pipe 33-41 %), and 27 % of their instructions were scalar adds.
// (Non-template overloads: preferred over the templates above for C<float>.)
__host__ __device__ __forceinline__ C<float> operator+(C<float> a, C<float> b) {
#ifdef __CUDA_ARCH__
    const float2 r = __fadd2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
    return mk<float>(r.x, r.y);
#else
    return mk<float>(a.x + b.x, a.y + b.y);
#endif
}
__host__ __device__ __forceinline__ C<float> operator-(C<float> a, C<float> b) {
#ifdef __CUDA_ARCH__
    const float2 r = __ffma2_rn(make_float2(b.x, b.y), make_float2(-1.0f, -1.0f), make_float2(a.x, a.y));   // a - b, exact product
    return mk<float>(r.x, r.y);
#else
    return mk<float>(a.x - b.x, a.y - b.y);
#endif
}
// s * v + o with a real s (the radix-2 stage of the split line transforms); one packed FFMA2 in single precision
template <class R> __host__ __device__ __forceinline__ C<R> fma_rc(R s, C<R> v, C<R> o) { return mk<R>(fma(s, v.x, o.x), fma(s, v.y, o.y)); }
__host__ __device__ __forceinline__ C<float> fma_rc(float s, C<float> v, C<float> o) {
#ifdef __CUDA_ARCH__
    const float2 r = __ffma2_rn(make_float2(s, s), make_float2(v.x, v.y), make_float2(o.x, o.y));
    return mk<float>(r.x, r.y);
#else
    return mk<float>(fmaf(s, v.x, o.x), fmaf(s, v.y, o.y));
#endif
}
template <class R> __host__ __device__ __forceinline__ C<R> operator-(C<R> a) { return mk<R>(-a.x, -a.y); }
template <class R> __host__ __device__ __forceinline__ C<R> operator*(C<R> a, C<R> b) { return mk<R>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <class R> __host__ __device__ __forceinline__ C<R> operator*(R s, C<R> a) { return mk<R>(s * a.x, s * a.y); }
template <class R> __host__ __device__ __forceinline__ C<R> conj(C<R> a) { return mk<R>(a.x, -a.y); }
// a * conj(b)
template <class R> __host__ __device__ __forceinline__ C<R> mulc(C<R> a, C<R> b) { return mk<R>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
// acc += a * b
template <class R> __host__ __device__ __forceinline__ void mad(C<R> &acc, C<R> a, C<R> b) {
    acc.x += a.x * b.x; acc.x -= a.y * b.y; acc.y += a.x * b.y; acc.y += a.y * b.x;
}
// acc += a * conj(b)
template <class R> __host__ __device__ __forceinline__ void madc(C<R> &acc, C<R> a, C<R> b) {
    acc.x += a.x * b.x; acc.x += a.y * b.y; acc.y += a.y * b.x; acc.y -= a.x * b.y;
}
template <class R> __host__ __device__ __forceinline__ R norm2(C<R> a) { return a.x * a.x + a.y * a.y; }


// 1 / x and 1 / sqrt(x) for positive normal x.  In double precision the IEEE-exact `a / b` and `1 / sqrt(x)` each
// expand to a hardware seed plus a dozen instructions with slow-path branches; the hot kernels call them 16 times per
// thread (the p2max / p2 factors of the t lines) and twice per g(x).  Here: the 20-bit hardware seed and three Newton
// steps (error below 2 ulp of double, no branches) -- inside every parity tolerance.  Single
// precision keeps the compiler's correctly rounded division and square root.
__device__ __forceinline__ double inv_pos(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
#pragma unroll
    for (int k = 0; k < 3; k++) r = fma(r, fma(-x, r, 1.0), r);
    return r;
}
__device__ __forceinline__ float inv_pos(float x) { return 1.0f / x; }
// s / x with x > 0: the branch-free reciprocal in double, the plain division in single precision
__device__ __forceinline__ double div_pos(double s, double x) { return s * inv_pos(x); }
__device__ __forceinline__ float div_pos(float s, float x) { return s / x; }
__device__ __forceinline__ double inv_sqrt_pos(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double h = 0.5 * x;
#pragma unroll
    for (int k = 0; k < 3; k++) y = fma(y, fma(-h * y, y, 0.5), y);
    return y;
}
__device__ __forceinline__ float inv_sqrt_pos(float x) { return 1.0f / sqrtf(x); }   // (rsqrtf, 2 ulp, let the fp32 links drift: plaquette 1.5e-6 after 20 updates)

// compile-time loop: f(std::integral_constant<int, i>) for i in [B, E)
template <int B, int E, class F>
__host__ __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// ---- compile-time cos / sin of 2*pi*m/L --------------------------------------------------------
// Exact integer octant reduction, then a Taylor polynomial on [0, pi/4] (error below 1 ulp of double).
namespace ct {
constexpr double PI = 3.14159265358979323846264338327950288;
constexpr double sin_small(double x) {   // 0 <= x <= pi/4
    const double x2 = x * x;
    double t = 1.0 / 355687428096000.0;                       // 1/17!
    t = -1.0 / 1307674368000.0 + x2 * t;                      // 1/15!
    t = 1.0 / 6227020800.0 + x2 * t;                          // 1/13!
    t = -1.0 / 39916800.0 + x2 * t;
    t = 1.0 / 362880.0 + x2 * t;
    t = -1.0 / 5040.0 + x2 * t;
    t = 1.0 / 120.0 + x2 * t;
    t = -1.0 / 6.0 + x2 * t;
    return x + x * x2 * t;
}
constexpr double cos_small(double x) {
    const double x2 = x * x;
    double t = 1.0 / 6402373705728000.0;                      // 1/18!
    t = -1.0 / 20922789888000.0 + x2 * t;                     // 1/16!
    t = 1.0 / 87178291200.0 + x2 * t;                         // 1/14!
    t = -1.0 / 479001600.0 + x2 * t;
    t = 1.0 / 3628800.0 + x2 * t;
    t = -1.0 / 40320.0 + x2 * t;
    t = 1.0 / 720.0 + x2 * t;
    t = -1.0 / 24.0 + x2 * t;
    t = 0.5 + x2 * t;
    return 1.0 - x2 * t;
}
struct CS { double c, s; };
// cos, sin of 2*pi*m/L for integers 0 <= m < L
constexpr CS cossin(int m, int L) {
    long num = 8L * m, den = 8L * L;            // t = num/den in [0, 1)
    double sc = 1.0, ss = 1.0;
    bool swap = false;
    if (2 * num > den) { num = den - num; ss = -ss; }                   // t -> 1 - t
    if (4 * num > den) { num = den / 2 - num; sc = -sc; }               // t -> 1/2 - t
    if (8 * num > den) { num = den / 4 - num; swap = true; }            // t -> 1/4 - t
    const double x = 2.0 * PI * (double)num / (double)den;
    double c = cos_small(x), s = sin_small(x);
    if (8 * num == den) { c = 0.70710678118654752440; s = c; }
    if (num == 0) { c = 1.0; s = 0.0; }
    if (swap) { const double t = c; c = s; s = t; }
    return CS{sc * c, ss * s};
}
}  // namespace ct

// z * exp(SIGN * 2 pi i M / L), M and L compile-time; trivial factors cost no multiplications.
template <int L, int M, int SIGN, class R>
__host__ __device__ __forceinline__ C<R> twiddle_mul(C<R> z) {
    constexpr int m = ((M % L) + L) % L;
    if constexpr (m == 0) {
        return z;
    } else if constexpr (2 * m == L) {
        return mk<R>(-z.x, -z.y);
    } else if constexpr (4 * m == L) {          // * (SIGN i)
        if constexpr (SIGN > 0) return mk<R>(-z.y, z.x); else return mk<R>(z.y, -z.x);
    } else if constexpr (4 * m == 3 * L) {      // * (-SIGN i)
        if constexpr (SIGN > 0) return mk<R>(z.y, -z.x); else return mk<R>(-z.y, z.x);
    } else {
        constexpr ct::CS cs = ct::cossin(m, L);
        constexpr R wr = (R)cs.c;
        constexpr R wi = (R)(SIGN * cs.s);
        if constexpr ((8 * m) % L == 0) {       // |wr| == |wi| == sqrt(1/2)
            constexpr R h = (R)0.70710678118654752440;
            constexpr bool cpos = cs.c > 0, spos = (SIGN * cs.s) > 0;
            const R a = cpos ? z.x : -z.x, b = cpos ? z.y : -z.y;      // sign(wr) * z
            const R c = spos ? z.y : -z.y, d = spos ? z.x : -z.x;      // sign(wi) * (y, x)
            return mk<R>(h * (a - c), h * (b + d));
        } else {
            return mk<R>(z.x * wr - z.y * wi, z.x * wi + z.y * wr);
        }
    }
}

// ---- in-register DFT of compile-time length N (natural order in, natural order out) ------------
// X[k] = sum_n v[n] exp(SIGN 2 pi i n k / N).  Composite N by Cooley-Tukey N = N1*N2.
template <int N, int SIGN, class R>
struct Dft {
    static constexpr int N1 = (N % 4 == 0) ? 4 : ((N % 2 == 0) ? 2 : 3);
    static constexpr int N2 = N / N1;
    static_assert(N1 * N2 == N && N > 4, "unsupported DFT length");
    static __host__ __device__ __forceinline__ void run(C<R> (&v)[N]) {
        C<R> t[N];
        static_for<0, N2>([&](auto n2c) {
            constexpr int n2 = decltype(n2c)::value;
            C<R> u[N1];
            static_for<0, N1>([&](auto n1c) { constexpr int n1 = decltype(n1c)::value; u[n1] = v[N2 * n1 + n2]; });
            Dft<N1, SIGN, R>::run(u);
            static_for<0, N1>([&](auto k1c) {
                constexpr int k1 = decltype(k1c)::value;
                t[k1 * N2 + n2] = twiddle_mul<N, n2 * k1, SIGN, R>(u[k1]);
            });
        });
        static_for<0, N1>([&](auto k1c) {
            constexpr int k1 = decltype(k1c)::value;
            C<R> u[N2];
            static_for<0, N2>([&](auto n2c) { constexpr int n2 = decltype(n2c)::value; u[n2] = t[k1 * N2 + n2]; });
            Dft<N2, SIGN, R>::run(u);
            static_for<0, N2>([&](auto k2c) { constexpr int k2 = decltype(k2c)::value; v[k1 + N1 * k2] = u[k2]; });
        });
    }
};
template <int SIGN, class R>
struct Dft<1, SIGN, R> {
    static __host__ __device__ __forceinline__ void run(C<R> (&)[1]) {}
};
template <int SIGN, class R>
struct Dft<2, SIGN, R> {
    static __host__ __device__ __forceinline__ void run(C<R> (&v)[2]) {
        const C<R> a = v[0], b = v[1];
        v[0] = a + b;
        v[1] = a - b;
    }
};
template <int SIGN, class R>
struct Dft<3, SIGN, R> {
    static __host__ __device__ __forceinline__ void run(C<R> (&v)[3]) {
        constexpr R h = (R)0.86602540378443864676;   // sqrt(3)/2
        const C<R> a = v[0], s = v[1] + v[2], d = v[1] - v[2];
        const C<R> m = mk<R>(a.x - (R)0.5 * s.x, a.y - (R)0.5 * s.y);
        // SIGN * i * h * d
        const C<R> r = (SIGN > 0) ? mk<R>(-h * d.y, h * d.x) : mk<R>(h * d.y, -h * d.x);
        v[0] = a + s;
        v[1] = m + r;
        v[2] = m - r;
    }
};
template <int SIGN, class R>
struct Dft<4, SIGN, R> {
    static __host__ __device__ __forceinline__ void run(C<R> (&v)[4]) {
        const C<R> t0 = v[0] + v[2], t1 = v[0] - v[2], t2 = v[1] + v[3], d = v[1] - v[3];
        const C<R> t3 = (SIGN > 0) ? mk<R>(-d.y, d.x) : mk<R>(d.y, -d.x);   // SIGN * i * d
        v[0] = t0 + t2;
        v[1] = t1 + t3;
        v[2] = t0 - t2;
        v[3] = t1 - t3;
    }
};

// Line-FFT factorisation L = N1 * N2 used by the shared-memory passes: the N1-point step runs on
// values taken straight from global memory, the N2-point step on values exchanged through shared memory.
template <int L> struct LineFactor {
    static constexpr int N1 = (L <= 8) ? L : ((L % 8 == 0) ? 8 : ((L % 4 == 0) ? 4 : ((L % 6 == 0) ? 6 : 3)));
    static constexpr int N2 = L / N1;
    static_assert(N1 * N2 == L && N2 <= 8, "unsupported FFT line length");
};

}  // namespace lgf
