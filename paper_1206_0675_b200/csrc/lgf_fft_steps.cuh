// lgf_fft_steps.cuh -- the shared-memory line-transform steps used by the FFT passes (see the header of
// lgf_fft.cu for the factorisation L = N1*N2 and the permuted frequency order they leave behind).
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#pragma once
#include "lgf_state.cuh"

namespace lgf {

// elements of a tile live at tile[hi*sHi + n*sN + lo], n = 0..L-1 along the transformed axis
struct TileShape {
    int nlo, nhi, sN, sHi;
};

template <class R, int L, int SIGN>
__device__ __forceinline__ void line_step_outer(C<R> *tile, const C<R> *tw, const TileShape ts) {
    // the N1-point butterflies (forward: first step, inverse: last step)
    constexpr int N1 = LineFactor<L>::N1, N2 = LineFactor<L>::N2;
    const int ntask = N2 * ts.nhi * ts.nlo;
    for (int task = threadIdx.x; task < ntask; task += blockDim.x) {
        const int lo = task % ts.nlo, r = task / ts.nlo, hi = r % ts.nhi, j = r / ts.nhi;
        C<R> *p = tile + hi * ts.sHi + lo + j * ts.sN;
        C<R> v[N1];
#pragma unroll
        for (int n1 = 0; n1 < N1; n1++) v[n1] = p[(N2 * n1) * ts.sN];
        Dft<N1, SIGN, R>::run(v);
        if constexpr (SIGN < 0 && N2 > 1) {            // forward: twiddle after the butterfly
#pragma unroll
            for (int k1 = 1; k1 < N1; k1++) v[k1] = v[k1] * tw[j * k1];
        }
#pragma unroll
        for (int k1 = 0; k1 < N1; k1++) p[(N2 * k1) * ts.sN] = v[k1];
    }
}

template <class R, int L, int SIGN>
__device__ __forceinline__ void line_step_inner(C<R> *tile, const C<R> *tw, const TileShape ts) {
    // the N2-point butterflies (forward: second step, inverse: first step, followed by conj twiddles)
    constexpr int N1 = LineFactor<L>::N1, N2 = LineFactor<L>::N2;
    if constexpr (N2 > 1) {
        const int ntask = N1 * ts.nhi * ts.nlo;
        for (int task = threadIdx.x; task < ntask; task += blockDim.x) {
            const int lo = task % ts.nlo, r = task / ts.nlo, hi = r % ts.nhi, k1 = r / ts.nhi;
            C<R> *p = tile + hi * ts.sHi + lo + (N2 * k1) * ts.sN;
            C<R> v[N2];
#pragma unroll
            for (int n2 = 0; n2 < N2; n2++) v[n2] = p[n2 * ts.sN];
            Dft<N2, SIGN, R>::run(v);
            if constexpr (SIGN > 0) {                  // inverse: conj twiddle w_L^-(n2 k1)
#pragma unroll
                for (int n2 = 1; n2 < N2; n2++) v[n2] = mulc(v[n2], tw[n2 * k1]);
            }
#pragma unroll
            for (int n2 = 0; n2 < N2; n2++) p[n2 * ts.sN] = v[n2];
        }
    }
}

template <class R, int L>
__device__ __forceinline__ void line_fft_forward(C<R> *tile, const C<R> *tw, const TileShape ts) {
    line_step_outer<R, L, -1>(tile, tw, ts);
    __syncthreads();
    line_step_inner<R, L, -1>(tile, tw, ts);
    __syncthreads();
}
template <class R, int L>
__device__ __forceinline__ void line_fft_inverse(C<R> *tile, const C<R> *tw, const TileShape ts) {
    line_step_inner<R, L, +1>(tile, tw, ts);
    __syncthreads();
    line_step_outer<R, L, +1>(tile, tw, ts);
    __syncthreads();
}

}  // namespace lgf
