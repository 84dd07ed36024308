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
#include "lgf_fft_steps.cuh"
#include "lgf_pdl.cuh"

namespace lgf {

// One pass over one axis.  grid = (tiles, 4 components).  Global element (hi, n, lo) of tile
// (lob, hib) of component c:  W[c*V + (lob*nlo + lo) + S*(n + L*(hib*nhi + hi))].
template <class R, int L, int MODE>
__global__ void __launch_bounds__(256) k_fft_axis(C<R> *__restrict__ W, Geom g, long long S, int nlo, int nhi,
                                                   int lo_blocks, const C<R> *__restrict__ twiddle,
                                                   const R *__restrict__ p2tab, R scale,
                                                   const DevState *__restrict__ st) {
    pdl_enter();
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
            const R f = (p2 == (R)0) ? (R)0 : scale / p2;            // p2 = 0 only at k = 0 (R6); also right for a
                                                                     // z-slab of k space (lgf_slab.cu), where s = 0 is not k = 0
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

// ---- two axes per pass ----------------------------------------------------------------------------
// PASS_XY: the (x, y) planes of all four components are contiguous in W (plane q = c*Lz*Lt + z + Lz*t
// starts at q*Lx*Ly), so a CTA takes P consecutive planes with fully coalesced loads, keeps them in
// shared memory with an odd row pitch, and transforms both axes there: x steps with lanes running over
// rows (conflict-free because of the odd pitch), y steps with lanes running over x.
template <class R, int LX, int LY, int MODE>
__global__ void __launch_bounds__(256) k_fft_xy(C<R> *__restrict__ W, int P, const C<R> *__restrict__ twx_g,
                                                 const C<R> *__restrict__ twy_g, const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    constexpr int PX = LX | 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *twx = reinterpret_cast<C<R> *>(smem_raw);
    C<R> *twy = twx + 64;
    C<R> *tile = twy + 64;
    for (int m = threadIdx.x; m < LX; m += blockDim.x) twx[m] = twx_g[m];
    for (int m = threadIdx.x; m < LY; m += blockDim.x) twy[m] = twy_g[m];
    C<R> *base = W + (long long)blockIdx.x * P * (LX * LY);
    const int nelem = P * LY * LX;
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int x = idx % LX, r = idx / LX;
        tile[r * PX + x] = base[idx];
    }
    __syncthreads();
    TileShape tsx, tsy;
    tsx.nlo = 1; tsx.nhi = P * LY; tsx.sN = 1; tsx.sHi = PX;
    tsy.nlo = LX; tsy.nhi = P; tsy.sN = PX; tsy.sHi = PX * LY;
    if constexpr (MODE == FFT_FWD) {
        line_fft_forward<R, LX>(tile, twx, tsx);
        line_fft_forward<R, LY>(tile, twy, tsy);
    } else {
        line_fft_inverse<R, LY>(tile, twy, tsy);
        line_fft_inverse<R, LX>(tile, twx, tsx);
    }
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int x = idx % LX, r = idx / LX;
        base[idx] = tile[r * PX + x];
    }
}

// PASS_ZT: for XC consecutive (x, y) indices of one component, the whole (z, t) plane: forward z,
// forward t, times p2max / (V p2(k)) (Alg. 1 lines 5, 7), inverse t, inverse z -- one read and one
// write of the field for four line transforms.  Shared-memory element (xc, z, t) lives at
// xc + XC*z + pitch*t; pitch = XC*Lz + padding chosen so that the z steps (lanes over xc, then t)
// are bank-conflict free; the t steps run lanes over the contiguous (xc, z) index.
template <class R, int LZ, int LT>
__global__ void __launch_bounds__(256) k_fft_zt(C<R> *__restrict__ W, Geom g, int XC, int pitch,
                                                 const C<R> *__restrict__ twz_g, const C<R> *__restrict__ twt_g,
                                                 const R *__restrict__ p2tab, R scale,
                                                 const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *twz = reinterpret_cast<C<R> *>(smem_raw);
    C<R> *twt = twz + 64;
    C<R> *tile = twt + 64;
    for (int m = threadIdx.x; m < LZ; m += blockDim.x) twz[m] = twz_g[m];
    for (int m = threadIdx.x; m < LT; m += blockDim.x) twt[m] = twt_g[m];
    const long long plane = g.S[2];
    const long long lo0 = (long long)blockIdx.x * XC;
    C<R> *Wc = W + (long long)blockIdx.y * g.V + lo0;
    const int nelem = LT * LZ * XC;
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int xc = idx % XC, r = idx / XC, z = r % LZ, t = r / LZ;
        tile[t * pitch + z * XC + xc] = Wc[xc + plane * (z + LZ * t)];
    }
    __syncthreads();
    TileShape tsz, tst;
    tsz.nlo = XC; tsz.nhi = LT; tsz.sN = XC; tsz.sHi = pitch;
    tst.nlo = XC * LZ; tst.nhi = 1; tst.sN = pitch; tst.sHi = 0;
    line_fft_forward<R, LZ>(tile, twz, tsz);
    line_fft_forward<R, LT>(tile, twt, tst);
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int xc = idx % XC, r = idx / XC, z = r % LZ, t = r / LZ;
        const int lo = (int)lo0 + xc, x = lo % g.L[0], y = lo / g.L[0];
        const R p2 = p2tab[x] + p2tab[64 + y] + p2tab[128 + z] + p2tab[192 + t];
        const R f = (p2 == (R)0) ? (R)0 : scale / p2;            // p2 = 0 only at k = 0 (R6)
        C<R> *e = tile + t * pitch + z * XC + xc;
        *e = f * (*e);
    }
    __syncthreads();
    line_fft_inverse<R, LT>(tile, twt, tst);
    line_fft_inverse<R, LZ>(tile, twz, tsz);
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int xc = idx % XC, r = idx / XC, z = r % LZ, t = r / LZ;
        Wc[xc + plane * (z + LZ * t)] = tile[t * pitch + z * XC + xc];
    }
}

// ---- launchers ------------------------------------------------------------------------------------
template <class K>
static cudaError_t set_smem(K kern, size_t smem) {
    return ensure_dynamic_smem(kern, smem);
}

template <class R, int L>
static cudaError_t launch_L(const AxisPass &p, C<R> *W, const Geom &g, const R *twiddle, const R *p2tab, R scale,
                            const DevState *st, LaunchStream stream) {
    const int lo_blocks = (int)(p.S / p.nlo);
    const long long tiles = (long long)lo_blocks * (p.H / p.nhi);
    dim3 grid((unsigned)tiles, 4);
    const C<R> *tw = reinterpret_cast<const C<R> *>(twiddle);
    auto go = [&](auto kern) {
        cudaError_t e = set_smem(kern, p.smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(kern, grid, dim3(p.threads), p.smem, stream, W, g, p.S, p.nlo, p.nhi, lo_blocks, tw, p2tab, scale, st);
    };
    switch (p.mode) {
        case FFT_FWD: return go(k_fft_axis<R, L, FFT_FWD>);
        case FFT_INV: return go(k_fft_axis<R, L, FFT_INV>);
        default: return go(k_fft_axis<R, L, FFT_FWD_SCALE_INV>);
    }
}

template <class R, int LX, int LY>
static cudaError_t launch_xy(const AxisPass &p, C<R> *W, const Geom &g, const R *const twiddle[4], const DevState *st,
                             LaunchStream stream) {
    const long long planes = 4LL * g.L[2] * g.L[3];
    const unsigned grid = (unsigned)(planes / p.nhi);
    const C<R> *twx = reinterpret_cast<const C<R> *>(twiddle[0]), *twy = reinterpret_cast<const C<R> *>(twiddle[1]);
    auto go = [&](auto kern) {
        cudaError_t e = set_smem(kern, p.smem);
        if (e != cudaSuccess) return e;
        return launch_pdl(kern, dim3(grid), dim3(p.threads), p.smem, stream, W, p.nhi, twx, twy, st);
    };
    return p.mode == FFT_FWD ? go(k_fft_xy<R, LX, LY, FFT_FWD>) : go(k_fft_xy<R, LX, LY, FFT_INV>);
}

template <class R, int LZ, int LT>
static cudaError_t launch_zt(const AxisPass &p, C<R> *W, const Geom &g, const R *const twiddle[4], const R *p2tab,
                             R scale, const DevState *st, LaunchStream stream) {
    dim3 grid((unsigned)(g.S[2] / p.nlo), 4);
    const C<R> *twz = reinterpret_cast<const C<R> *>(twiddle[2]), *twt = reinterpret_cast<const C<R> *>(twiddle[3]);
    auto kern = k_fft_zt<R, LZ, LT>;
    cudaError_t e = set_smem(kern, p.smem);
    if (e != cudaSuccess) return e;
    return launch_pdl(kern, grid, dim3(p.threads), p.smem, stream, W, g, p.nlo, p.pitch, twz, twt, p2tab, scale, st);
}

// the (La, Lb) pairs for which two-axis kernels are instantiated: BASELINE.json's lattices
#define LGF_XY_PAIRS(X) X(8, 8) X(16, 16) X(24, 24) X(32, 32) X(64, 64)
#define LGF_ZT_PAIRS(X) X(8, 8) X(16, 16) X(24, 48) X(32, 32) X(64, 64)

bool fft_pair_supported(int kind, int La, int Lb) {
#define LGF_CHECK(A, B) if (La == A && Lb == B) return true;
    if (kind == PASS_XY) { LGF_XY_PAIRS(LGF_CHECK) }
    if (kind == PASS_ZT) { LGF_ZT_PAIRS(LGF_CHECK) }
#undef LGF_CHECK
    return false;
}

template <class R>
cudaError_t launch_fft_pass(const AxisPass &p, C<R> *W, const Geom &g, const R *const twiddle[4], const R *p2tab,
                            R scale, const DevState *st, LaunchStream stream) {
    if (p.kind == PASS_XY) {
#define LGF_GO(A, B) if (p.L == A && p.L2 == B) return launch_xy<R, A, B>(p, W, g, twiddle, st, stream);
        LGF_XY_PAIRS(LGF_GO)
#undef LGF_GO
        return cudaErrorInvalidValue;
    }
    if (p.kind == PASS_ZT) {
#define LGF_GO(A, B) if (p.L == A && p.L2 == B) return launch_zt<R, A, B>(p, W, g, twiddle, p2tab, scale, st, stream);
        LGF_ZT_PAIRS(LGF_GO)
#undef LGF_GO
        return cudaErrorInvalidValue;
    }
    switch (p.L) {
#define LGF_CASE(LEN) case LEN: return launch_L<R, LEN>(p, W, g, twiddle[p.axis], p2tab, scale, st, stream);
        LGF_CASE(2) LGF_CASE(3) LGF_CASE(4) LGF_CASE(6) LGF_CASE(8) LGF_CASE(12) LGF_CASE(16) LGF_CASE(24)
        LGF_CASE(32) LGF_CASE(48) LGF_CASE(64)
#undef LGF_CASE
        default: return cudaErrorInvalidValue;
    }
}

template cudaError_t launch_fft_pass<float>(const AxisPass &, C<float> *, const Geom &, const float *const[4],
                                            const float *, float, const DevState *, LaunchStream);
template cudaError_t launch_fft_pass<double>(const AxisPass &, C<double> *, const Geom &, const double *const[4],
                                             const double *, double, const DevState *, LaunchStream);

}  // namespace lgf
