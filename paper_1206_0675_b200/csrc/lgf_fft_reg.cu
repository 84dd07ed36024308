// lgf_fft_reg.cu -- register-resident line transforms: the fast path of the batched 4-D FFT
// (Alg. 1 lines 3-8) for lattices whose lines fit in one thread's registers.
// Part of liblgf (CUDA path); no cuFFT; shares nothing with oracle/.
//
// Every thread owns one whole line of the transformed axis: it loads the L elements straight from
// global memory (L independent 16-byte / 8-byte loads in flight per thread, lanes running over the
// contiguous index so every request is coalesced), does the length-L DFT in registers with
// compile-time twiddles (Dft<L>, natural order in and out), and hands the result to the thread that
// owns the crossing line through shared memory.  Three sweeps of the field per iteration:
//
//   k_fftr_xy<FWD>   (x, y) planes: y lines from global -> smem transpose -> x lines -> global.  The
//                    k-space plane is written TRANSPOSED, element (kx, ky) at kx*Ly + ky, so that the
//                    stores (lanes over ky) are coalesced too.
//   k_fftr_zt        XC consecutive (kx, ky) indices x the whole (z, t) plane: z lines from global ->
//                    smem -> t lines: forward, times p2max / (V p2(k)) (Alg. 1 lines 5, 7), inverse ->
//                    smem -> z lines inverse -> global.
//   k_fftr_xy<INV>   kx lines from global (transposed layout) -> smem -> ky lines -> global, natural
//                    (x, y) layout again; inside an iteration the GOUT variant ends with the g-build (a5)
//                    and writes g(x) instead of w(x).
//
// One shared-memory round trip per sweep in (x, y), two in (z, t), against five and ten for the
// in-place two-step passes of lgf_fft.cu, which remain the path for lines that do not fit in registers.
#include "lgf_fft_steps.cuh"
#include "lgf_pdl.cuh"

namespace lgf {

// ---- (x, y) planes --------------------------------------------------------------------------------
// P planes per CTA, L threads per plane.  Plane q (q = c*Lz*Lt + z + Lz*t) starts at W + q*L*L.
// GOUT (inverse sweep only): the CTA's P planes are the four packed components of P/4 (z, t) slices, so
// all of w(x) is on chip when the sweep ends; instead of storing w it builds g(x) = GS(1 + i (alpha/2) w(x))
// (a5, Alg. 1 line 10) and stores rows 0, 1 of g to G -- the separate g-build pass over the field disappears.
template <class R, int L, int MODE, int P, bool GOUT>
__global__ void __launch_bounds__(P *L) k_fftr_xy(C<R> *__restrict__ W, const DevState *__restrict__ st,
                                                  C<R> *__restrict__ G, long long V, int nzt, R half_alpha) {
    pdl_enter();
    if (st->done) return;
    static_assert(!GOUT || (MODE == FFT_INV && P % 4 == 0 && L % 4 == 0), "g output needs all four components on chip");
    constexpr int PX = L | 1;                    // odd row pitch: lanes over rows hit distinct banks
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tile_all = reinterpret_cast<C<R> *>(smem_raw);
    const int p = threadIdx.x / L, i = threadIdx.x % L;
    // plane number: GOUT: component p % 4 of slice blockIdx.x * (P/4) + p / 4; otherwise consecutive planes
    const long long q = GOUT ? (long long)(p % 4) * nzt + (long long)blockIdx.x * (P / 4) + p / 4
                             : (long long)blockIdx.x * P + p;
    C<R> *base = W + q * (L * L);
    C<R> *tile = tile_all + p * (L * PX);
    C<R> v[L];
#pragma unroll
    for (int n = 0; n < L; n++) v[n] = base[n * L + i];                 // line n = 0..L-1 at fixed i, coalesced over i
    if constexpr (MODE == FFT_FWD) {
        Dft<L, -1, R>::run(v);                                          // over y at x = i  ->  ky = n
#pragma unroll
        for (int n = 0; n < L; n++) tile[n * PX + i] = v[n];            // tile[ky][x]
        __syncthreads();
#pragma unroll
        for (int n = 0; n < L; n++) v[n] = tile[i * PX + n];            // row ky = i, x = n
        Dft<L, -1, R>::run(v);                                          // over x  ->  kx = n
    } else {
        Dft<L, +1, R>::run(v);                                          // over kx at ky = i  ->  x = n
#pragma unroll
        for (int n = 0; n < L; n++) tile[i * PX + n] = v[n];            // tile[ky][x]
        __syncthreads();
#pragma unroll
        for (int n = 0; n < L; n++) v[n] = tile[n * PX + i];            // column x = i, ky = n
        Dft<L, +1, R>::run(v);                                          // over ky  ->  y = n
    }
    if constexpr (!GOUT) {
#pragma unroll
        for (int n = 0; n < L; n++) base[n * L + i] = v[n];             // FWD: (kx = n, ky = i); INV: (y = n, x = i)
    } else {
        __syncthreads();                                                // everyone has read its column
#pragma unroll
        for (int n = 0; n < L; n++) tile[n * PX + i] = v[n];            // tile[y][x] of component p % 4
        __syncthreads();
        const C<R> *t4 = tile_all + (p / 4) * 4 * (L * PX);             // the four component tiles of this slice
        const long long s0 = ((long long)blockIdx.x * (P / 4) + p / 4) * (L * L);
#pragma unroll
        for (int m = 0; m < L / 4; m++) {
            const int y = (p % 4) + 4 * m;
            Herm<R> w;
            w.m01 = t4[y * PX + i];
            w.m02 = t4[L * PX + y * PX + i];
            w.m12 = t4[2 * L * PX + y * PX + i];
            const C<R> dg = t4[3 * L * PX + y * PX + i];
            w.m00 = dg.x;
            w.m11 = dg.y;
            C<R> gx[9];
            build_g(w, half_alpha, gx);
            const long long s = s0 + y * L + i;
#pragma unroll
            for (int e = 0; e < 6; e++) G[(long long)e * V + s] = gx[e];
        }
    }
}

// ---- (z, t) planes --------------------------------------------------------------------------------
// grid = ((Lx*Ly)/XC, 4 components); threads = XC * max(LZ, LT).  Shared-memory element (xc, z, t) at
// xc + XC*z + PITCH*t, PITCH = XC*LZ + padding (lanes (xc, t) of the z-line steps on distinct banks).
// TREG: the t lines are transformed in registers (natural k order); otherwise with the in-place
// two-step shared-memory transform of lgf_fft_steps.cuh (permuted k order along t; the p2 table of
// axis t is stored in the matching order by the planner).
template <class R, int LZ, int LT, int XC, bool TREG>
struct ZtShape {
    static constexpr int PHASE = 128 / (int)sizeof(C<R>);
    static constexpr int PITCH = XC * LZ + ((XC < PHASE && (XC * LZ) % PHASE == 0) ? XC : 0);
    static constexpr int THREADS = XC * (LZ > LT ? LZ : LT);
    static constexpr size_t SMEM = sizeof(C<R>) * ((size_t)PITCH * LT + (TREG ? 0 : 64));
    // resident CTAs per SM the register allocation is asked to allow.  Asking for 3 at 32 x 32 fp64 (168
    // registers, 280 B of spills) made the sweep slower (50 -> 65 us on B200), so the compiler is left alone.
    static constexpr int MINB = 1;
};

template <class R, int LZ, int LT, int XC, bool TREG>
__global__ void __launch_bounds__((ZtShape<R, LZ, LT, XC, TREG>::THREADS), (ZtShape<R, LZ, LT, XC, TREG>::MINB))
    k_fftr_zt(C<R> *__restrict__ W, Geom g, const C<R> *__restrict__ twt_g, const R *__restrict__ p2tab, R scale,
              const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    using S = ZtShape<R, LZ, LT, XC, TREG>;
    constexpr int PITCH = S::PITCH;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tile = reinterpret_cast<C<R> *>(smem_raw);
    const long long plane = g.S[2];
    const int lo0 = blockIdx.x * XC;
    C<R> *Wc = W + (long long)blockIdx.y * g.V + lo0;
    const int tid = threadIdx.x;
    const int xc = tid % XC, r = tid / XC;

    if (r < LT) {                                                       // z line at (xc, t = r)
        C<R> v[LZ];
        const C<R> *src = Wc + xc + plane * ((long long)LZ * r);
#pragma unroll
        for (int z = 0; z < LZ; z++) v[z] = src[plane * z];
        Dft<LZ, -1, R>::run(v);
#pragma unroll
        for (int z = 0; z < LZ; z++) tile[r * PITCH + z * XC + xc] = v[z];
    }
    __syncthreads();
    // k-space (x, y) index of this thread's column: the forward (x, y) sweep wrote the plane transposed
    const int lo = lo0 + xc, kx = lo / g.L[1], ky = lo % g.L[1];
    if constexpr (TREG) {
        if (r < LZ) {                                                   // t line at (xc, kz = r)
            C<R> v[LT];
#pragma unroll
            for (int t = 0; t < LT; t++) v[t] = tile[t * PITCH + tid];
            Dft<LT, -1, R>::run(v);
            const R p2xyz = p2tab[kx] + p2tab[64 + ky] + p2tab[128 + r];
#pragma unroll
            for (int t = 0; t < LT; t++) {
                const R p2 = p2xyz + p2tab[192 + t];
                const R f = (p2 == (R)0) ? (R)0 : scale / p2;           // Alg. 1 lines 5, 7; zero mode -> 0 (R6)
                v[t] = f * v[t];
            }
            Dft<LT, +1, R>::run(v);
#pragma unroll
            for (int t = 0; t < LT; t++) tile[t * PITCH + tid] = v[t];
        }
        __syncthreads();
    } else {
        C<R> *twt = tile + PITCH * LT;
        for (int m = tid; m < LT; m += blockDim.x) twt[m] = twt_g[m];
        TileShape tst;
        tst.nlo = XC * LZ; tst.nhi = 1; tst.sN = PITCH; tst.sHi = 0;
        __syncthreads();
        line_fft_forward<R, LT>(tile, twt, tst);
        for (int idx = tid; idx < XC * LZ * LT; idx += blockDim.x) {
            const int j = idx % (XC * LZ), t = idx / (XC * LZ), jx = j % XC, kz = j / XC;
            const int l2 = lo0 + jx;
            const R p2 = p2tab[l2 / g.L[1]] + p2tab[64 + l2 % g.L[1]] + p2tab[128 + kz] + p2tab[192 + t];
            const R f = (p2 == (R)0) ? (R)0 : scale / p2;
            C<R> *e = tile + t * PITCH + j;
            *e = f * (*e);
        }
        __syncthreads();
        line_fft_inverse<R, LT>(tile, twt, tst);
    }
    if (r < LT) {
        C<R> v[LZ];
#pragma unroll
        for (int z = 0; z < LZ; z++) v[z] = tile[r * PITCH + z * XC + xc];
        Dft<LZ, +1, R>::run(v);
        C<R> *dst = Wc + xc + plane * ((long long)LZ * r);
#pragma unroll
        for (int z = 0; z < LZ; z++) dst[plane * z] = v[z];
    }
    (void)kx; (void)ky;
}

// ---- launchers ------------------------------------------------------------------------------------
template <class R> struct RegCfg;
// planes per CTA of the (x, y) sweep and consecutive (kx, ky) indices per CTA of the (z, t) sweep
template <> struct RegCfg<double> { static constexpr int XC = 4; };
template <> struct RegCfg<float> { static constexpr int XC = 8; };
template <int L> struct XyPlanes { static constexpr int P = (L >= 32) ? 4 : ((L >= 24) ? 4 : ((L >= 16) ? 8 : 16)); };

#define LGF_REG_XY(X) X(8) X(16) X(24) X(32)
#define LGF_REG_ZT(X) X(8, 8, true) X(16, 16, true) X(32, 32, true) X(24, 48, false)

bool fft_reg_supported(const Geom &g) {
    bool xy = false, zt = false;
#define LGF_C1(LEN) if (g.L[0] == LEN && g.L[1] == LEN && (4LL * g.L[2] * g.L[3]) % XyPlanes<LEN>::P == 0) xy = true;
    LGF_REG_XY(LGF_C1)
#undef LGF_C1
#define LGF_C2(A, B, T) if (g.L[2] == A && g.L[3] == B) zt = true;
    LGF_REG_ZT(LGF_C2)
#undef LGF_C2
    return xy && zt && (g.S[2] % 8 == 0);
}
bool fft_reg_t_natural(const Geom &g) {
#define LGF_C3(A, B, T) if (g.L[2] == A && g.L[3] == B) return T;
    LGF_REG_ZT(LGF_C3)
#undef LGF_C3
    return false;
}

template <class R>
cudaError_t launch_fft_reg(int which, const Geom &g, C<R> *W, const R *twiddle_t, const R *p2tab, R scale,
                           const DevState *st, LaunchStream stream, C<R> *G, R half_alpha) {
    if (which == 0 || which == 2 || which == 3) {                       // (x, y) forward / inverse / inverse + g
        const long long planes = 4LL * g.L[2] * g.L[3];
        const int nzt = g.L[2] * g.L[3];
#define LGF_GO(LEN)                                                                                       \
    if (g.L[0] == LEN) {                                                                                   \
        constexpr int P = XyPlanes<LEN>::P;                                                                \
        constexpr size_t SM = sizeof(C<R>) * P * LEN * (LEN | 1);                                            \
        auto kf = k_fftr_xy<R, LEN, FFT_FWD, P, false>;                                                    \
        auto ki = k_fftr_xy<R, LEN, FFT_INV, P, false>;                                                    \
        auto kg = k_fftr_xy<R, LEN, FFT_INV, P, true>;                                                     \
        auto kern = which == 0 ? kf : (which == 2 ? ki : kg);                                              \
        {                                                                                                \
            cudaError_t e = ensure_dynamic_smem(kern, SM);                                               \
            if (e != cudaSuccess) return e;                                                              \
        }                                                                                                \
        return launch_pdl(kern, dim3((unsigned)(planes / P)), dim3(P * LEN), SM, stream, W, st, G, g.V, nzt, half_alpha); \
    }
        LGF_REG_XY(LGF_GO)
#undef LGF_GO
        return cudaErrorInvalidValue;
    }
    constexpr int XC = RegCfg<R>::XC;
#define LGF_GO(A, B, T)                                                                                       \
    if (g.L[2] == A && g.L[3] == B) {                                                                         \
        using S = ZtShape<R, A, B, XC, T>;                                                                    \
        auto kern = k_fftr_zt<R, A, B, XC, T>;                                                                \
        {                                                                                                     \
            cudaError_t e = ensure_dynamic_smem(kern, S::SMEM);                                               \
            if (e != cudaSuccess) return e;                                                                   \
        }                                                                                                     \
        dim3 grid((unsigned)(g.S[2] / XC), 4);                                                                \
        return launch_pdl(kern, grid, dim3(S::THREADS), S::SMEM, stream, W, g, reinterpret_cast<const C<R> *>(twiddle_t), \
                          p2tab, scale, st);                                                                  \
    }
    LGF_REG_ZT(LGF_GO)
#undef LGF_GO
    return cudaErrorInvalidValue;
}

template cudaError_t launch_fft_reg<float>(int, const Geom &, C<float> *, const float *, const float *, float,
                                           const DevState *, LaunchStream, C<float> *, float);
template cudaError_t launch_fft_reg<double>(int, const Geom &, C<double> *, const double *, const double *, double,
                                            const DevState *, LaunchStream, C<double> *, double);

}  // namespace lgf
