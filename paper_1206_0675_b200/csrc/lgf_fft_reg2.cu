// lgf_fft_reg2.cu -- register-line sweeps of the batched 4-D FFT (Alg. 1 lines 3-8) with
// TWO threads per line (lgf_fft_split.cuh): the same three sweeps as lgf_fft_reg.cu,
//   k_fftr2_xy<FWD>, k_fftr2_zt (forward z, t; times p2max / (V p2(k)); inverse t, z), k_fftr2_xy<INV[, GOUT]>,
// but each thread holds half a line, so a 32-point fp64 line costs 64 data registers per thread instead of
// 128 (more warps in flight) and 64-point lines fit at all.  All four axes end up in natural k order.
// Part of liblgf (CUDA path); no cuFFT; shares nothing with oracle/.
//
// Thread layout: a warp owns 16 lines; lane = q + 16 h, q = line within the warp, h = which half of the
// line.  The pair (q, 0), (q, 1) exchanges with __shfl_xor(.., 16).  Lanes q run over the contiguous
// index of every global and shared-memory access.
#include <cstdio>
#include <string>

#include "lgf_fft_split.cuh"
#include "lgf_state.cuh"
#include "lgf_pdl.cuh"
#include "lgf_tma.cuh"

namespace lgf {

constexpr int PAIR_MASK = 16;

// ---- (x, y) planes --------------------------------------------------------------------------------
// P planes per CTA, 2 L threads per plane (L / 16 warps).  Plane q starts at W + q L^2.  The k-space plane
// is stored transposed, element (kx, ky) at kx L + ky, as in lgf_fft_reg.cu.
// GOUT (inverse only): the P planes are the four packed components of P / 4 (z, t) slices; the sweep ends
// with a5, g = GS(1 + i (alpha/2) w), and stores rows 0, 1 of g instead of w.
template <class R, int L, int MODE, int P, bool GOUT>
__global__ void __launch_bounds__(2 * P * L) k_fftr2_xy(C<R> *__restrict__ W, const DevState *__restrict__ st,
                                                        C<R> *__restrict__ G, long long V, int nzt, R half_alpha) {
    pdl_enter();
    if (st->done) return;
    static_assert(L % 16 == 0, "16 lines per warp");
    static_assert(!GOUT || (MODE == FFT_INV && P % 4 == 0), "g output needs all four components on chip");
    constexpr int M = L / 2;
    constexpr int PX = L | 1;                    // odd row pitch
    using S = SplitDft<L, PAIR_MASK, R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tile_all = reinterpret_cast<C<R> *>(smem_raw);
    const int tid = threadIdx.x;
    const int p = tid / (2 * L), tp = tid % (2 * L);          // plane, thread within the plane
    const int h = (tp >> 4) & 1;                               // lane = q + 16 h
    const int i = (tp >> 5) * 16 + (tp & 15);                  // line number 0 .. L-1
    const long long q = GOUT ? (long long)(p % 4) * nzt + (long long)blockIdx.x * (P / 4) + p / 4
                             : (long long)blockIdx.x * P + p;
    C<R> *base = W + q * (L * L);
    C<R> *tile = tile_all + p * (L * PX);
    C<R> v[M];
    if constexpr (MODE == FFT_FWD) {
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = base[(m + M * h) * L + i];        // y = m + M h at x = i
        S::forward(v, h);                                                    // -> ky = 2 j + h
#pragma unroll
        for (int j = 0; j < M; j++) tile[(2 * j + h) * PX + i] = v[j];       // tile[ky][x]
        __syncthreads();
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = tile[i * PX + m + M * h];         // row ky = i, x = m + M h
        S::forward(v, h);                                                    // -> kx = 2 j + h
#pragma unroll
        for (int j = 0; j < M; j++) base[(2 * j + h) * L + i] = v[j];        // (kx, ky = i), transposed plane
    } else {
#pragma unroll
        for (int j = 0; j < M; j++) v[j] = base[(2 * j + h) * L + i];        // kx = 2 j + h at ky = i
        S::inverse(v, h);                                                    // -> x = m + M h
#pragma unroll
        for (int m = 0; m < M; m++) tile[i * PX + m + M * h] = v[m];         // tile[ky][x]
        __syncthreads();
#pragma unroll
        for (int j = 0; j < M; j++) v[j] = tile[(2 * j + h) * PX + i];       // column x = i, ky = 2 j + h
        S::inverse(v, h);                                                    // -> y = m + M h
        if constexpr (!GOUT) {
#pragma unroll
            for (int m = 0; m < M; m++) base[(m + M * h) * L + i] = v[m];    // (y, x = i)
        } else {
            __syncthreads();                                                 // everyone has read its column
#pragma unroll
            for (int m = 0; m < M; m++) tile[(m + M * h) * PX + i] = v[m];   // tile[y][x] of component p % 4
            __syncthreads();
            const C<R> *t4 = tile_all + (p / 4) * 4 * (L * PX);
            const long long s0 = ((long long)blockIdx.x * (P / 4) + p / 4) * (L * L);
            // the 8 L threads of a slice share its L^2 sites: thread (p % 4, h, i) takes rows y = (p%4) + 4 h' ...
            const int sub = (p % 4) * 2 + h;                                 // 0 .. 7
#pragma unroll
            for (int mm = 0; mm < L / 8; mm++) {
                const int y = sub + 8 * mm;
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
}

// ---- (x, y) planes through the bulk-copy engine (lgf_tune "fft_bulk") ---------------------------------
// The same sweep with the plane brought on chip by ONE cp.async.bulk per plane (1-D TMA, SASS UBLKCP; an (x, y)
// plane is a contiguous 16 KB block at 32^4 fp64) signalled by an mbarrier, and -- where the result goes back to W
// -- taken off chip by one bulk store (UBLKCP.G.S).  The plane lands in the transposition tile's own storage
// (dense L x L inside the L x (L | 1) tile), so the shared-memory footprint and the CTAs per SM are those of
// k_fftr2_xy; what it costs is one more pass through shared memory and two more barriers per plane.  Measured on
// B200 (32^4, FFT time per iteration, default / bulk): see DESIGN.md section 6 -- it is an ablation, off by default.
template <class R, int L, int MODE, int P, bool GOUT>
__global__ void __launch_bounds__(2 * P * L) k_fftr2_xy_bulk(C<R> *__restrict__ W, const DevState *__restrict__ st,
                                                             C<R> *__restrict__ G, long long V, int nzt, R half_alpha) {
    pdl_enter();
    if (st->done) return;
    static_assert(L % 16 == 0, "16 lines per warp");
    constexpr int M = L / 2;
    constexpr int PX = L | 1;
    constexpr unsigned PLANE_BYTES = L * L * sizeof(C<R>);
    using S = SplitDft<L, PAIR_MASK, R>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C<R> *tile_all = reinterpret_cast<C<R> *>(smem_raw);
    __shared__ uint64_t bar;
    const int tid = threadIdx.x;
    const int p = tid / (2 * L), tp = tid % (2 * L);
    const int h = (tp >> 4) & 1;
    const int i = (tp >> 5) * 16 + (tp & 15);
    auto plane_of = [&](int pp) {
        return GOUT ? (long long)(pp % 4) * nzt + (long long)blockIdx.x * (P / 4) + pp / 4 : (long long)blockIdx.x * P + pp;
    };
    C<R> *base = W + plane_of(p) * (L * L);
    C<R> *tile = tile_all + p * (L * PX);
    if (tid == 0) {
        mbar_init(&bar, 1);
        mbar_init_fence();
        mbar_arrive_expect_tx(&bar, P * PLANE_BYTES);
        for (int pp = 0; pp < P; pp++) bulk_g2s(tile_all + pp * (L * PX), W + plane_of(pp) * (L * L), PLANE_BYTES, &bar);
    }
    __syncthreads();                                         // the barrier's initialisation is visible to every waiter
    mbar_wait(&bar, 0);
    C<R> v[M];
    if constexpr (MODE == FFT_FWD) {
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = tile[(m + M * h) * L + i];        // dense plane: y = m + M h at x = i
        __syncthreads();                                                     // everyone has its line: the tile may be overwritten
        S::forward(v, h);
#pragma unroll
        for (int j = 0; j < M; j++) tile[(2 * j + h) * PX + i] = v[j];       // tile[ky][x]
        __syncthreads();
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = tile[i * PX + m + M * h];
        S::forward(v, h);
        __syncthreads();
#pragma unroll
        for (int j = 0; j < M; j++) tile[(2 * j + h) * L + i] = v[j];        // dense again: (kx, ky = i), transposed plane
    } else {
#pragma unroll
        for (int j = 0; j < M; j++) v[j] = tile[(2 * j + h) * L + i];
        __syncthreads();
        S::inverse(v, h);
#pragma unroll
        for (int m = 0; m < M; m++) tile[i * PX + m + M * h] = v[m];
        __syncthreads();
#pragma unroll
        for (int j = 0; j < M; j++) v[j] = tile[(2 * j + h) * PX + i];
        S::inverse(v, h);
        __syncthreads();
        if constexpr (!GOUT) {
#pragma unroll
            for (int m = 0; m < M; m++) tile[(m + M * h) * L + i] = v[m];    // dense (y, x = i)
        } else {
#pragma unroll
            for (int m = 0; m < M; m++) tile[(m + M * h) * PX + i] = v[m];
            __syncthreads();
            const C<R> *t4 = tile_all + (p / 4) * 4 * (L * PX);
            const long long s0 = ((long long)blockIdx.x * (P / 4) + p / 4) * (L * L);
            const int sub = (p % 4) * 2 + h;
#pragma unroll
            for (int mm = 0; mm < L / 8; mm++) {
                const int y = sub + 8 * mm;
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
            return;
        }
    }
    // the dense result planes back to W: ordinary shared-memory stores, made visible to the copy engine, one bulk store each
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (tid == 0) {
        for (int pp = 0; pp < P; pp++)
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(W + plane_of(pp) * (L * L)),
                         "r"(smem_u32(tile_all + pp * (L * PX))), "r"(PLANE_BYTES)
                         : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // shared memory must outlive the reads
    }
    (void)base;
}

// ---- (z, t) planes --------------------------------------------------------------------------------
// grid = ((Lx Ly) / XC, 4 components).  Shared-memory element (xc, z, t) at xc + XC z + PITCH t, PITCH =
// XC LZ + padding (the 8-lane phases of the z-line stores, lanes (xc, t), land on distinct banks).
// z lines: line l -> (xc = l % XC, t = l / XC); t lines: line l = xc + XC kz.  Two threads per line.
template <class R, int LZ, int LT, int XC>
struct Zt2Shape {
    static constexpr int PHASE = 128 / (int)sizeof(C<R>);
    static constexpr int PITCH = XC * LZ + ((XC < PHASE && (XC * LZ) % PHASE == 0) ? XC : 0);
    static constexpr int LINES = XC * (LZ > LT ? LZ : LT);
    static constexpr int THREADS = 2 * LINES;
    static constexpr size_t SMEM = sizeof(C<R>) * (size_t)PITCH * LT;
    // at least two CTAs per SM where the tile allows it: caps the registers at 128 for 256 threads (the compiler
    // otherwise spends 134 on overlapping the 16 reciprocals of the scale step, which halves the occupancy)
    // (fp64 lines of up to 32 points only; 0 = no request, which is NOT the same as asking for 1: with "1" the fp32
    // 64 x 64 sweep took 168 registers instead of 128 and lost its second CTA -- 64^4 fp32 FFT 1.17 -> 1.35 ms)
    static constexpr int MINB = (sizeof(R) == 8 && SMEM <= 110 * 1024 && LZ <= 32 && LT <= 32) ? 2 : 0;
    static_assert((XC * LZ) % 16 == 0 && (XC * LT) % 16 == 0, "16 lines per warp");
};

template <class R, int LZ, int LT, int XC>
__global__ void __launch_bounds__((Zt2Shape<R, LZ, LT, XC>::THREADS), (Zt2Shape<R, LZ, LT, XC>::MINB))
    k_fftr2_zt(C<R> *__restrict__ W, Geom g, const R *__restrict__ p2tab, R scale, const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    using Sh = Zt2Shape<R, LZ, LT, XC>;
    constexpr int PITCH = Sh::PITCH, MZ = LZ / 2, MT = LT / 2;
    using SZ = SplitDft<LZ, PAIR_MASK, R>;
    using ST = SplitDft<LT, PAIR_MASK, R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tile = reinterpret_cast<C<R> *>(smem_raw);
    const long long plane = g.S[2];
    const int lo0 = blockIdx.x * XC;
    C<R> *Wc = W + (long long)blockIdx.y * g.V + lo0;
    const int tid = threadIdx.x;
    const int h = (tid >> 4) & 1;
    const int l = (tid >> 5) * 16 + (tid & 15);               // line number
    const int xc = l % XC, r = l / XC;                        // z-line steps: t = r; t-line step: kz = r

    // whole warps take each branch (the line counts are multiples of 16), so the shuffles inside are safe
    if (l < XC * LT) {                                        // forward z at (xc, t = r)
        C<R> v[MZ];
        const C<R> *src = Wc + xc + plane * ((long long)LZ * r);
#pragma unroll
        for (int m = 0; m < MZ; m++) v[m] = src[plane * (m + MZ * h)];
        SZ::forward(v, h);                                    // -> kz = 2 j + h
#pragma unroll
        for (int j = 0; j < MZ; j++) tile[r * PITCH + (2 * j + h) * XC + xc] = v[j];
    }
    __syncthreads();
    if (l < XC * LZ) {                                        // t line at (xc, kz = r): forward, scale, inverse
        C<R> v[MT];
#pragma unroll
        for (int m = 0; m < MT; m++) v[m] = tile[(m + MT * h) * PITCH + l];
        ST::forward(v, h);                                    // -> kt = 2 j + h
        // k-space (x, y) index of this column: the forward (x, y) sweep wrote the plane transposed
        const int lo = lo0 + xc, kx = lo / g.L[1], ky = lo % g.L[1];
        const R p2xyz = p2tab[kx] + p2tab[64 + ky] + p2tab[128 + r];
#pragma unroll
        for (int j = 0; j < MT; j++) {
            const R p2 = p2xyz + p2tab[192 + 2 * j + h];
            const R f = (p2 == (R)0) ? (R)0 : div_pos(scale, p2);     // Alg. 1 lines 5, 7; zero mode -> 0 (R6)
            v[j] = f * v[j];
        }
        ST::inverse(v, h);                                    // -> t = m + MT h
#pragma unroll
        for (int m = 0; m < MT; m++) tile[(m + MT * h) * PITCH + l] = v[m];
    }
    __syncthreads();
    if (l < XC * LT) {                                        // inverse z at (xc, t = r)
        C<R> v[MZ];
#pragma unroll
        for (int j = 0; j < MZ; j++) v[j] = tile[r * PITCH + (2 * j + h) * XC + xc];
        SZ::inverse(v, h);                                    // -> z = m + MZ h
        C<R> *dst = Wc + xc + plane * ((long long)LZ * r);
#pragma unroll
        for (int m = 0; m < MZ; m++) dst[plane * (m + MZ * h)] = v[m];
    }
}

// ---- configuration and launchers --------------------------------------------------------------------
// planes per CTA of the inverse (P; a multiple of 4 allows the g output) and of the forward (PF) (x, y) sweep,
// and consecutive (kx, ky) indices per CTA of the (z, t) sweep.  Measured at 32^4 on B200 (FFT time per
// iteration): PF = 4 -> 2: fp64 0.1129 -> 0.1091 ms, fp32 0.0643 -> 0.0628 ms (smaller CTAs, shorter last
// wave; PF = 1 the same as 2); XC = 4 against 2 / 1 / 8: fp64 0.1129 against 0.1189 / 0.1438 / 0.1226 ms.
template <class R, int L> struct Xy2Cfg;
template <> struct Xy2Cfg<double, 16> { static constexpr int P = 8, PF = 8; };
template <> struct Xy2Cfg<double, 32> { static constexpr int P = 4, PF = 2; };
template <> struct Xy2Cfg<double, 64> { static constexpr int P = 1, PF = 1; };   // 4 planes of 64 x 64 fp64 exceed shared memory
template <> struct Xy2Cfg<float, 16> { static constexpr int P = 8, PF = 8; };
template <> struct Xy2Cfg<float, 32> { static constexpr int P = 4, PF = 2; };
template <> struct Xy2Cfg<float, 64> { static constexpr int P = 4, PF = 4; };
// (Lz, Lt) pairs of the (z, t) sweep: Lt = Lz, and Lt = 2 Lz -- the usual shape of a lattice QCD volume (the
// paper tunes on 32^3 x n) -- with the consecutive (kx, ky) indices per CTA
template <class R, int LZ, int LT> struct Zt2Cfg;
template <> struct Zt2Cfg<double, 16, 16> { static constexpr int XC = 4; };
template <> struct Zt2Cfg<double, 32, 32> { static constexpr int XC = 4; };
template <> struct Zt2Cfg<double, 64, 64> { static constexpr int XC = 2; };
template <> struct Zt2Cfg<double, 16, 32> { static constexpr int XC = 4; };
template <> struct Zt2Cfg<double, 32, 64> { static constexpr int XC = 2; };
template <> struct Zt2Cfg<float, 16, 16> { static constexpr int XC = 8; };
template <> struct Zt2Cfg<float, 32, 32> { static constexpr int XC = 4; };
template <> struct Zt2Cfg<float, 64, 64> { static constexpr int XC = 2; };
template <> struct Zt2Cfg<float, 16, 32> { static constexpr int XC = 4; };
template <> struct Zt2Cfg<float, 32, 64> { static constexpr int XC = 2; };
#define LGF_REG2_ZT(X) X(16, 16) X(32, 32) X(64, 64) X(16, 32) X(32, 64)

#define LGF_REG2_LEN(X) X(16) X(32) X(64)

static bool reg2_len(int L) { return L == 16 || L == 32 || L == 64; }

bool fft_reg2_supported(const Geom &g) {
    bool zt = false;
#define LGF_C(A, B) if (g.L[2] == A && g.L[3] == B) zt = true;
    LGF_REG2_ZT(LGF_C)
#undef LGF_C
    if (!(g.L[0] == g.L[1] && reg2_len(g.L[0]) && zt)) return false;
    const long long planes = 4LL * g.L[2] * g.L[3];
    return planes % 8 == 0 && g.S[2] % 8 == 0;
}
// the (x, y) sweeps alone (which = 0, 2, 3) for a geometry whose last two extents are arbitrary -- a t-slab of the
// sharded path (lgf_slab.cu): square planes of a supported length, whole CTAs of planes, and for the g output
// the four components of P / 4 (z, t) slices per CTA
bool fft_reg2_xy_supported(const Geom &g) {
    return g.L[0] == g.L[1] && reg2_len(g.L[0]) && (4LL * g.L[2] * g.L[3]) % 8 == 0 && ((long long)g.L[2] * g.L[3]) % 2 == 0;
}
// can the forward (x, y) sweep run over one component at a time (whole CTAs of that component's planes)?
bool fft_reg2_xy_by_component(const Geom &g, int prec) {
    if (!fft_reg2_xy_supported(g)) return false;
    const long long per = (long long)g.L[2] * g.L[3];
    int pf = 8;
#define LGF_C(LEN) if (g.L[0] == LEN) pf = prec == 8 ? Xy2Cfg<double, LEN>::PF : Xy2Cfg<float, LEN>::PF;
    LGF_REG2_LEN(LGF_C)
#undef LGF_C
    return per % pf == 0;
}
bool fft_reg2_xy_gout(const Geom &g, int prec) { return fft_reg2_xy_supported(g) && !(g.L[0] == 64 && prec == 8); }
// can the inverse (x, y) sweep end with the g-build for this lattice and precision (bytes per real)?
bool fft_reg2_gout(const Geom &g, int prec) {
    if (!fft_reg2_supported(g)) return false;
    if (g.L[0] == 64) return prec == 4;
    return true;
}

static thread_local int t_xy_comp = -1;           // >= 0: the forward (x, y) sweep over ONE packed component only (lgf_slab.cu)
static thread_local bool t_xy_bulk = false;      // set by launch_fft_reg2 for the launch in progress (lgf_tune "fft_bulk")
template <class R, int L, int MODE, int P, bool GOUT>
static cudaError_t launch_xy2_as(const Geom &g, C<R> *W, const DevState *st, LaunchStream stream, C<R> *G, R half_alpha) {
    if (t_xy_bulk) {
        constexpr size_t SMB = sizeof(C<R>) * P * L * (L | 1);
        auto kb = k_fftr2_xy_bulk<R, L, MODE, P, GOUT>;
        if (cudaError_t e = ensure_dynamic_smem(kb, SMB); e != cudaSuccess) return e;
        return launch_pdl(kb, dim3((unsigned)(4LL * g.L[2] * g.L[3] / P)), dim3(2 * P * L), SMB, stream, W, st, G, g.V, g.L[2] * g.L[3],
                          half_alpha);
    }
    constexpr size_t SM = sizeof(C<R>) * P * L * (L | 1);
    long long planes = 4LL * g.L[2] * g.L[3];
    if (!GOUT && t_xy_comp >= 0) {                   // one component: its planes are contiguous in W
        planes /= 4;
        if (planes % P != 0) return cudaErrorInvalidValue;
        W += (long long)t_xy_comp * g.V;
    }
    auto kern = k_fftr2_xy<R, L, MODE, P, GOUT>;
    if (cudaError_t e = ensure_dynamic_smem(kern, SM); e != cudaSuccess) return e;
    return launch_pdl(kern, dim3((unsigned)(planes / P)), dim3(2 * P * L), SM, stream, W, st, G, g.V, g.L[2] * g.L[3],
                      half_alpha);
}
template <class R, int L>
static cudaError_t launch_xy2(int which, const Geom &g, C<R> *W, const DevState *st, LaunchStream stream, C<R> *G,
                              R half_alpha) {
    constexpr int P = Xy2Cfg<R, L>::P, PF = Xy2Cfg<R, L>::PF;
    if (which == 0) return launch_xy2_as<R, L, FFT_FWD, PF, false>(g, W, st, stream, G, half_alpha);
    if (which == 2) return launch_xy2_as<R, L, FFT_INV, P, false>(g, W, st, stream, G, half_alpha);
    if constexpr (P % 4 == 0) return launch_xy2_as<R, L, FFT_INV, P, true>(g, W, st, stream, G, half_alpha);
    return cudaErrorInvalidValue;
}

template <class R, int LZ, int LT>
static cudaError_t launch_zt2(const Geom &g, C<R> *W, const R *p2tab, R scale, const DevState *st, LaunchStream stream) {
    constexpr int XC = Zt2Cfg<R, LZ, LT>::XC;
    using Sh = Zt2Shape<R, LZ, LT, XC>;
    auto kern = k_fftr2_zt<R, LZ, LT, XC>;
    if (cudaError_t e = ensure_dynamic_smem(kern, Sh::SMEM); e != cudaSuccess) return e;
    dim3 grid((unsigned)(g.S[2] / XC), 4);
    return launch_pdl(kern, grid, dim3(Sh::THREADS), Sh::SMEM, stream, W, g, p2tab, scale, st);
}

// which: 0 = (x, y) forward, 1 = (z, t) forward + scale + inverse, 2 = (x, y) inverse, 3 = (x, y) inverse + g
template <class R>
cudaError_t launch_fft_reg2(int which, const Geom &g, C<R> *W, const R *p2tab, R scale, const DevState *st,
                            LaunchStream stream, C<R> *G, R half_alpha, bool bulk, int comp) {
    t_xy_bulk = bulk;
    t_xy_comp = comp;
    if (which == 1) {
#define LGF_GO(A, B) if (g.L[2] == A && g.L[3] == B) return launch_zt2<R, A, B>(g, W, p2tab, scale, st, stream);
        LGF_REG2_ZT(LGF_GO)
#undef LGF_GO
        return cudaErrorInvalidValue;
    }
#define LGF_GO(LEN) if (g.L[0] == LEN) return launch_xy2<R, LEN>(which, g, W, st, stream, G, half_alpha);
    LGF_REG2_LEN(LGF_GO)
#undef LGF_GO
    return cudaErrorInvalidValue;
}

// the instantiation launch_fft_reg2 picks, as a profiler prints it (bench.py matches ncu captures against it)
template <class R>
static std::string reg2_name(int which, const Geom &g) {
    const char *rn = sizeof(R) == 8 ? "double" : "float";
    char buf[96] = "";
    if (which == 1) {
#define LGF_GO(A, B) if (g.L[2] == A && g.L[3] == B) snprintf(buf, sizeof buf, "k_fftr2_zt<%s, %d, %d, %d>", rn, A, B, Zt2Cfg<R, A, B>::XC);
        LGF_REG2_ZT(LGF_GO)
#undef LGF_GO
        return buf;
    }
#define LGF_GO(LEN)                                                                                           \
    if (g.L[0] == LEN) {                                                                                       \
        if (which == 0) snprintf(buf, sizeof buf, "k_fftr2_xy<%s, %d, 0, %d, 0>", rn, LEN, Xy2Cfg<R, LEN>::PF);  \
        else snprintf(buf, sizeof buf, "k_fftr2_xy<%s, %d, 1, %d, %d>", rn, LEN, Xy2Cfg<R, LEN>::P, which == 3 ? 1 : 0); \
    }
    LGF_REG2_LEN(LGF_GO)
#undef LGF_GO
    return buf;
}
std::string fft_reg2_kernel_name(int which, const Geom &g, int prec, bool bulk) {
    std::string s = prec == 8 ? reg2_name<double>(which, g) : reg2_name<float>(which, g);
    if (bulk && which != 1 && s.size() > 10) s.insert(10, "_bulk");      // k_fftr2_xy -> k_fftr2_xy_bulk
    return s;
}

template cudaError_t launch_fft_reg2<float>(int, const Geom &, C<float> *, const float *, float, const DevState *,
                                            LaunchStream, C<float> *, float, bool, int);
template cudaError_t launch_fft_reg2<double>(int, const Geom &, C<double> *, const double *, double, const DevState *,
                                             LaunchStream, C<double> *, double, bool, int);

}  // namespace lgf
