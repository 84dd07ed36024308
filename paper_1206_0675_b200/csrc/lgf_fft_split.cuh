// lgf_fft_split.cuh -- a line transform of length L = 2 M shared by TWO threads of one warp (lanes l and
// l ^ PMASK): each holds M elements in registers, one radix-2 stage crosses the pair with warp shuffles, the
// M-point DFT is done in registers (Dft<M>, compile-time twiddles).  Halves the registers a line costs per
// thread (more warps in flight) and makes 64-point fp64 lines possible at all.
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
//
//   forward (decimation in frequency), thread h = 0 / 1 of the pair:
//     in : v[m] = x[m + M h]
//     u[m] = h == 0 ?  x[m] + x[m + M]  :  (x[m] - x[m + M]) w_L^m ,   w_L = exp(-2 pi i / L)
//     out: v[j] = X[2 j + h] = DFT_M(u)[j]
//   inverse (decimation in time), conjugate twiddles, unnormalised:
//     in : v[j] = X[2 j + h]
//     y = IDFT_M(v);  thread 1: y[m] *= conj(w_L)^m
//     out: v[m] = x[m + M h] = h == 0 ?  y0[m] + y1[m]  :  y0[m] - y1[m]
#pragma once
#include "lgf_cplx.cuh"

namespace lgf {

__device__ __forceinline__ C<double> shfl_xor_c(C<double> z, int mask) {
    return mk<double>(__shfl_xor_sync(0xffffffffu, z.x, mask), __shfl_xor_sync(0xffffffffu, z.y, mask));
}
__device__ __forceinline__ C<float> shfl_xor_c(C<float> z, int mask) {
    return mk<float>(__shfl_xor_sync(0xffffffffu, z.x, mask), __shfl_xor_sync(0xffffffffu, z.y, mask));
}

template <int L, int PMASK, class R>
struct SplitDft {
    static constexpr int M = L / 2;
    static_assert(L % 2 == 0 && M >= 2, "split transform needs an even length");

    // all 32 lanes of the warp must call (shuffles); h = this thread's half (0 / 1)
    static __device__ __forceinline__ void forward(C<R> (&v)[M], int h) {
        // one fused multiply-add per real makes both halves' butterfly, o + s v with s = +1 (thread 0: x[m] +
        // x[m + M]) or -1 (thread 1: x[m] - x[m + M], o being the partner's x[m]); exact, since s v is.  Computing
        // sum and difference in both threads and selecting cost 4 double-precision adds per element instead of 2.
        const R s = h ? (R)-1 : (R)1;
        static_for<0, M>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            const C<R> o = shfl_xor_c(v[m], PMASK);
            const C<R> t = fma_rc(s, v[m], o);
            if constexpr (m == 0) v[m] = t;
            else v[m] = h ? twiddle_mul<L, m, -1, R>(t) : t;             // thread 1: (x[m] - x[m + M]) w^m
        });
        Dft<M, -1, R>::run(v);
    }
    static __device__ __forceinline__ void inverse(C<R> (&v)[M], int h) {
        Dft<M, +1, R>::run(v);
        const R s = h ? (R)-1 : (R)1;
        static_for<0, M>([&](auto mc) {
            constexpr int m = decltype(mc)::value;
            C<R> y = v[m];
            if constexpr (m != 0) y = h ? twiddle_mul<L, m, +1, R>(v[m]) : v[m];   // thread 1: y1[m] conj(w)^m
            const C<R> o = shfl_xor_c(y, PMASK);
            v[m] = fma_rc(s, y, o);                                     // y0 + y1  /  y0 - y1
        });
    }
};

}  // namespace lgf
