// lgf_fft.cu -- hand-written batched 4-D complex FFT over the packed components of Delta
// (Alg. 1 lines 3-8), one lattice axis per pass, in place, with the p2max/p2
// multiplication (line 5) and the 1/V normalisation (line 7) fused between the forward and the
// inverse transform of the last axis.  No cuFFT.  Part of liblgf; shares nothing with oracle/.
//
// Line transform of length L = N1*N2 (N1, N2 <= 8, LineFactor<L>), decimation in frequency on the way
// in and decimation in time on the way back, both in place in a shared-memory tile:
//   forward  step 1: for fixed n2:  v[n1] = x[N2 n1 + n2];  N1-point DFT;  y[N2 k1 + n2] = w_L^(n2 k1) v[k1]
//            step 2: for fixed k1:  v[n2] = y[N2 k1 + n2];  N2-point DFT;  z[N2 k1 + k2] = v[k2]
//   so position p = N2 k1 + k2 of the line holds frequency k(p) = k1 + N1 k2.  The k-space field is
//   only ever multiplied point-wise by a function of k and transformed back, so it is left in this
//   permuted order (the p2 table is stored in the same order) and the inverse runs the two steps
//   backwards with conjugate twiddles; no reordering pass, no second buffer (the paper's k3 kernel and
//   reorder array, are not needed).
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

// One pass over one axis.  grid = (tiles, 4 components).  Global element (hi, n, lo) of tile
// (lob, hib) of component c:  W[c*V + (lob*nlo + lo) + S*(n + L*(hib*nhi + hi))].
template <class R, int L, int MODE>
__global__ void __launch_bounds__(256) k_fft_axis(C<R> *__restrict__ W, Geom g, long long S, int nlo, int nhi,
                                                   int lo_blocks, const C<R> *__restrict__ twiddle,
                                                   const R *__restrict__ p2tab, R scale,
                                                   const DevState *__restrict__ st) {
    if (st->done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tw = reinterpret_cast<C<R> *>(smem_raw);          // [L] forward twiddles exp(-2 pi i m / L)
    C<R> *tile = tw + 64;
    TileShape ts;
    ts.nlo = nlo;
    ts.nhi = nhi;
    if (S == 1) { ts.sN = 1; ts.sHi = L | 1; }              // x axis: lines contiguous, odd pitch
    else { ts.sN = nlo; ts.sHi = L * nlo; }
    const long long lo0 = (long long)(blockIdx.x % lo_blocks) * nlo;
    const long long hi0 = (long long)(blockIdx.x / lo_blocks) * nhi;
    C<R> *Wc = W + (long long)blockIdx.y * g.V;

    for (int m = threadIdx.x; m < L; m += blockDim.x) tw[m] = twiddle[m];
    const int nelem = nhi * L * nlo;
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int lo = idx % nlo, r = idx / nlo, n = r % L, hi = r / L;
        tile[hi * ts.sHi + n * ts.sN + lo] = Wc[lo0 + lo + S * (n + (long long)L * (hi0 + hi))];
    }
    __syncthreads();

    if constexpr (MODE == FFT_FWD || MODE == FFT_FWD_SCALE_INV) line_fft_forward<R, L>(tile, tw, ts);
    if constexpr (MODE == FFT_FWD_SCALE_INV) {
        // Alg. 1 lines 5 and 7: times p2max / p2(k) and 1/V; zero mode -> 0 (R5-R7).
        // p2tab[mu*64 + p] = 4 sin^2(pi k_mu(p) / L_mu) in the permuted order of axis mu.
        for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
            const int lo = idx % nlo, r = idx / nlo, n = r % L, hi = r / L;
            const long long s = lo0 + lo + S * (n + (long long)L * (hi0 + hi));
            int c[4];
            site_coords(g, s, c);
            const R p2 = p2tab[c[0]] + p2tab[64 + c[1]] + p2tab[128 + c[2]] + p2tab[192 + c[3]];
            const R f = (s == 0) ? (R)0 : scale / p2;
            C<R> *e = tile + hi * ts.sHi + n * ts.sN + lo;
            *e = f * (*e);
        }
        __syncthreads();
    }
    if constexpr (MODE == FFT_INV || MODE == FFT_FWD_SCALE_INV) line_fft_inverse<R, L>(tile, tw, ts);

    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int lo = idx % nlo, r = idx / nlo, n = r % L, hi = r / L;
        Wc[lo0 + lo + S * (n + (long long)L * (hi0 + hi))] = tile[hi * ts.sHi + n * ts.sN + lo];
    }
}

template <class R, int L>
static cudaError_t launch_L(const AxisPass &p, C<R> *W, const Geom &g, const R *twiddle, const R *p2tab, R scale,
                            const DevState *st, cudaStream_t stream) {
    const int lo_blocks = (int)(p.S / p.nlo);
    const long long tiles = (long long)lo_blocks * (p.H / p.nhi);
    dim3 grid((unsigned)tiles, 4);
    const C<R> *tw = reinterpret_cast<const C<R> *>(twiddle);
    auto go = [&](auto kern) {
        cudaError_t e = cudaSuccess;
        if (p.smem > 48 * 1024)
            e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem);
        if (e != cudaSuccess) return e;
        kern<<<grid, p.threads, p.smem, stream>>>(W, g, p.S, p.nlo, p.nhi, lo_blocks, tw, p2tab, scale, st);
        return cudaGetLastError();
    };
    switch (p.mode) {
        case FFT_FWD: return go(k_fft_axis<R, L, FFT_FWD>);
        case FFT_INV: return go(k_fft_axis<R, L, FFT_INV>);
        default: return go(k_fft_axis<R, L, FFT_FWD_SCALE_INV>);
    }
}

template <class R>
cudaError_t launch_fft_pass(const AxisPass &p, C<R> *W, const Geom &g, const R *twiddle, const R *p2tab, R scale,
                            const DevState *st, cudaStream_t stream) {
    switch (p.L) {
#define LGF_CASE(LEN) case LEN: return launch_L<R, LEN>(p, W, g, twiddle, p2tab, scale, st, stream);
        LGF_CASE(2) LGF_CASE(3) LGF_CASE(4) LGF_CASE(6) LGF_CASE(8) LGF_CASE(12) LGF_CASE(16) LGF_CASE(24)
        LGF_CASE(32) LGF_CASE(48) LGF_CASE(64)
#undef LGF_CASE
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_fft_pass<float>(const AxisPass &, C<float> *, const Geom &, const float *, const float *,
                                            float, const DevState *, cudaStream_t);
template cudaError_t launch_fft_pass<double>(const AxisPass &, C<double> *, const Geom &, const double *,
                                             const double *, double, const DevState *, cudaStream_t);

}  // namespace lgf
