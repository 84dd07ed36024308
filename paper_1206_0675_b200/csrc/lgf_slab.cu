// lgf_slab.cu -- ONE configuration sharded over N ranks (the paper's
// stated future work; its CPU code does the same decomposition with PFFT over MPI, :124).
//
// Rank r of N owns the t-slab  t = r T .. (r+1) T - 1,  T = Lt / N  (all x, y, z), i.e. a contiguous slice of the
// canonical configuration.  One iteration of Algorithm 1 then needs exactly these exchanges:
//   a1    Delta(x) wants U_t(x - t) of the slice below the slab: one 3-D slice of U_t from rank r-1   (halo, LINKS)
//   a2-a4 x, y, z are whole inside the slab: (x, y) planes by the register-line sweeps of lgf_fft_reg2.cu (else one pass
//         per axis, lgf_fft.cu); the t lines are gathered by an ALL-TO-ALL that turns t-slabs into z-slabs (rank r gets
//         z = r Zl .. (r+1) Zl - 1 of every t, Zl = Lz / N).  The passes next to it work straight on its buffers: forward z
//         writes the send buffer, the t pass (forward, times p2max / (V p2(k)), inverse) reads the receive buffer and writes
//         the send buffer of the second all-to-all, inverse z reads its receive buffer -- no pack / unpack pass
//   a6    U_t(x) g(x + t)^dag wants g of the slice above the slab: one slice of g from rank r+1          (halo, G)
//   F, theta: per-rank sums, all-reduced by the caller (two doubles).
// This file holds the kernels and the per-rank context; the exchanges themselves are the caller's (NCCL through
// torch.distributed, paper_1206_0675_b200/slab.py): every entry point here is local to one rank and works on
// buffers the caller hands in, so no kernel ever waits on another rank.  Two forms of a6: k_slab_update transforms
// the links in place (a link transform reads no other link) and leaves a1 to a pass of its own; k_slab_sweep is the
// fused a6 + a1 pass of the iteration loop (second g halo instead of the U_t halo, two link buffers).
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#include <new>
#include <string>
#include <vector>

#include "../../include/lgf.h"
#include "lgf_fft_split.cuh"
#include "lgf_fft_steps.cuh"
#include "lgf_state.cuh"

namespace lgf {
bool host_valid_len(int L);
void host_line_factor(int L, int &N1, int &N2);
void host_cossin_2pi(int m, int L, double &c, double &s);

constexpr int SLAB_THREADS = 256;

template <class R>
__device__ __forceinline__ void slab_load_g(const C<R> *__restrict__ G, long long V, long long s, C<R> (&gx)[9]) {
#pragma unroll
    for (int e = 0; e < 6; e++) gx[e] = G[(long long)e * V + s];
    reconstruct_row2(gx);
}

// fixed-order sum of the per-block partial sums: out[0] = sum Re tr U, out[1] = sum tr(Delta Delta^dag) of the slab
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_sum2(const double *__restrict__ partial, int nb, double *__restrict__ out,
                                                            const int *__restrict__ stop) {
    if (*stop) return;
    __shared__ double scratch[SLAB_THREADS / 32][2];
    double f = 0.0, t = 0.0;
    for (int i = threadIdx.x; i < nb; i += SLAB_THREADS) { f += partial[2 * i]; t += partial[2 * i + 1]; }
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) { out[0] = f; out[1] = t; }
}

// a6 on a slab, in place: U_mu(x) <- g(x) U_mu(x) g(x + mu)^dag (eq. 2, Alg. 1 line 14); g(x + t) of the last local
// slice comes from `ghalo` (rows 0, 1 of g on the slice above, C<R>[6][S3]).
template <class R, int NR>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_update(LinkPair<R> lp, const C<R> *__restrict__ G,
                                                              const C<R> *__restrict__ ghalo, Geom g,
                                                              const DevState *__restrict__ st) {
    if (st->done) return;
    C<R> *__restrict__ links = st->cur ? lp.buf[1] : lp.buf[0];
    const long long s = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x;
    if (s >= g.V) return;
    int c[4];
    site_coords(g, s, c);
    C<R> gx[9];
    slab_load_g(G, g.V, s, gx);
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        C<R> u[9], gn[9], t[9], p[9];
        load_link<R, NR>(links, g.V, mu, s, u);
        if (mu == 3 && c[3] == g.L[3] - 1) slab_load_g(ghalo, g.S[3], s - g.S[3] * (long long)(g.L[3] - 1), gn);
        else slab_load_g(G, g.V, site_fwd(g, s, c, mu), gn);
        mat_mul<NR>(gx, u, t);
        mat_mul_dag<NR>(t, gn, p);
        store_link<R, NR>(links, g.V, mu, s, p);                    // with 12-real storage row 2 is rebuilt on load (eq. 8)
    }
}

// U_t of the slab's last slice, from whichever link buffer is current, into a contiguous send buffer [3 NR][S3]
template <class R>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_pack_ut(LinkPair<R> lp, C<R> *__restrict__ out, long long V, long long S3,
                                                               int nplanes, long long first, const DevState *__restrict__ st) {
    const C<R> *__restrict__ links = st->cur ? lp.buf[1] : lp.buf[0];
    const long long i = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x;
    if (i >= S3 * nplanes) return;
    const long long e = i / S3, sx = i % S3;
    out[i] = links[(3LL * nplanes + e) * V + first + sx];
}

// Where element n of a line lives: base + (n / D) strideQ + (n % D) strideN.  The all-to-all buffers are ordered
// [c][q][tl][zl][xy] (c = packed component of W: four independent exchanges, each a contiguous quarter of the buffer;
// chunk q of a component goes to / came from rank q; tl, zl local to the chunk), so with piece = T Zl Sxy elements
//   a z line in a buffer   (z = q Zl + zl):  D = Zl, strideQ = piece, strideN = Sxy,     base = (c N T + tl) Zl Sxy + xy
//   a t line in a buffer   (t = q T + tl):   D = T,  strideQ = piece, strideN = Zl Sxy,  base = c N piece + zl Sxy + xy
//   a z line in the field W[c][tl][z][xy]:   D = Lz (one piece),      strideN = Sxy,     base = c V + tl Lz Sxy + xy
// (N piece = V elements per component).  blockIdx.y = the "other" local index (tl for z lines, zl for t lines),
// blockIdx.z = c.  The components being separate lets component c's exchange overlap component c + 1's line pass
// (the *_comp entry points below, paper_1206_0675_b200/slab.py).
struct LineAddr {
    long long stride_c, stride_o, strideQ, strideN;
    int D;
    int shift;      // log2(D) when D is a power of two (always, for the lengths the register-line passes take), else -1
};
__device__ __forceinline__ long long line_elem(const LineAddr &a, long long base, int n) {
    return base + (long long)(n / a.D) * a.strideQ + (long long)(n % a.D) * a.strideN;
}

// One line pass of the 4-D FFT (Alg. 1 lines 3-8) that reads with one address map and writes with another, so that
// the passes next to an all-to-all work straight on its buffers and no separate pack / unpack pass exists:
//   z forward   FFT_FWD             src = W (t-slab)        dst = send buffer
//   t           FFT_FWD_SCALE_INV   src = receive buffer    dst = send buffer     (times p2max / (V p2(k)), k = 0 -> 0)
//   z inverse   FFT_INV             src = receive buffer    dst = W
// A CTA takes nlo consecutive (x, y) indices of one line bundle; the transform itself is lgf_fft_steps.cuh's.
template <class R, int L, int MODE>
__global__ void __launch_bounds__(256) k_slab_fft_line(const C<R> *__restrict__ src, C<R> *__restrict__ dst, LineAddr as,
                                                       LineAddr ad, int nlo, int Lx, const C<R> *__restrict__ twiddle,
                                                       const R *__restrict__ p2tab, R scale) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tw = reinterpret_cast<C<R> *>(smem_raw);
    C<R> *tile = tw + 64;
    TileShape ts;
    ts.nlo = nlo; ts.nhi = 1; ts.sN = nlo; ts.sHi = 0;
    const long long xy0 = (long long)blockIdx.x * nlo;
    const long long bs = (long long)blockIdx.z * as.stride_c + (long long)blockIdx.y * as.stride_o + xy0;
    const long long bd = (long long)blockIdx.z * ad.stride_c + (long long)blockIdx.y * ad.stride_o + xy0;
    for (int m = threadIdx.x; m < L; m += blockDim.x) tw[m] = twiddle[m];
    const int nelem = L * nlo;
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int lo = idx % nlo, n = idx / nlo;
        tile[idx] = src[line_elem(as, bs, n) + lo];
    }
    __syncthreads();
    if constexpr (MODE == FFT_FWD || MODE == FFT_FWD_SCALE_INV) line_fft_forward<R, L>(tile, tw, ts);
    if constexpr (MODE == FFT_FWD_SCALE_INV) {
        // t lines: blockIdx.y = zl; p2tab[128 + zl] is this rank's z-slab of the z table (positions, not frequencies)
        for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
            const int lo = idx % nlo, n = idx / nlo;
            const int xy = (int)xy0 + lo, x = xy % Lx, y = xy / Lx;
            const R p2 = p2tab[x] + p2tab[64 + y] + p2tab[128 + blockIdx.y] + p2tab[192 + n];
            const R f = (p2 == (R)0) ? (R)0 : scale / p2;           // p2 = 0 only at k = 0 (R6)
            tile[idx] = f * tile[idx];
        }
        __syncthreads();
    }
    if constexpr (MODE == FFT_INV || MODE == FFT_FWD_SCALE_INV) line_fft_inverse<R, L>(tile, tw, ts);
    for (int idx = threadIdx.x; idx < nelem; idx += blockDim.x) {
        const int lo = idx % nlo, n = idx / nlo;
        dst[line_elem(ad, bd, n) + lo] = tile[idx];
    }
}

// The same three passes with the line in REGISTERS, two threads per line (lgf_fft_split.cuh; lengths 16, 32, 64 with
// whole CTAs of LINE2_LINES consecutive (x, y) indices): no shared memory, every element is loaded once into the register
// that transforms it, and the axis ends in NATURAL frequency order (the p2 table of that axis is stored accordingly).
// Thread layout as in lgf_fft_reg2.cu: a warp owns 16 lines, lane = q + 16 h, q runs over the contiguous index.
constexpr int LINE2_LINES = 64;       // lines per CTA (two threads each); with 128 the 512 CTAs of a 32^4 half lattice leave a 0.73 wave tail (iteration 2 % slower)
__device__ __forceinline__ long long line_elem2(const LineAddr &a, long long base, int n) {
    return base + (long long)(n >> a.shift) * a.strideQ + (long long)(n & (a.D - 1)) * a.strideN;
}
template <class R, int L, int MODE>
__global__ void __launch_bounds__(2 * LINE2_LINES) k_slab_fft_line2(const C<R> *__restrict__ src, C<R> *__restrict__ dst, LineAddr as,
                                                        LineAddr ad, int Lx, const R *__restrict__ p2tab, R scale) {
    constexpr int M = L / 2;
    using S = SplitDft<L, 16, R>;
    const int tid = threadIdx.x;
    const int h = (tid >> 4) & 1;
    const long long xy = (long long)blockIdx.x * LINE2_LINES + (tid >> 5) * 16 + (tid & 15);
    const long long bs = (long long)blockIdx.z * as.stride_c + (long long)blockIdx.y * as.stride_o + xy;
    const long long bd = (long long)blockIdx.z * ad.stride_c + (long long)blockIdx.y * ad.stride_o + xy;
    C<R> v[M];
    if constexpr (MODE == FFT_INV) {
#pragma unroll
        for (int j = 0; j < M; j++) v[j] = src[line_elem2(as, bs, 2 * j + h)];          // frequency k = 2 j + h
    } else {
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = src[line_elem2(as, bs, m + M * h)];
        S::forward(v, h);                                                                // -> k = 2 j + h
    }
    if constexpr (MODE == FFT_FWD_SCALE_INV) {
        // t lines: blockIdx.y = zl (p2tab[128 + zl] = this rank's z-slab of the z table); Alg. 1 lines 5, 7
        const int x = (int)(xy % Lx), y = (int)(xy / Lx);
        const R p2xyz = p2tab[x] + p2tab[64 + y] + p2tab[128 + blockIdx.y];
#pragma unroll
        for (int j = 0; j < M; j++) {
            const R p2 = p2xyz + p2tab[192 + 2 * j + h];
            const R f = (p2 == (R)0) ? (R)0 : scale / p2;                                // p2 = 0 only at k = 0 (R6)
            v[j] = f * v[j];
        }
    }
    if constexpr (MODE == FFT_FWD) {
#pragma unroll
        for (int j = 0; j < M; j++) dst[line_elem2(ad, bd, 2 * j + h)] = v[j];
    } else {
        S::inverse(v, h);                                                                // -> position m + M h
#pragma unroll
        for (int m = 0; m < M; m++) dst[line_elem2(ad, bd, m + M * h)] = v[m];
    }
}
template <class R>
static cudaError_t launch_line2(int L, int mode, const C<R> *src, C<R> *dst, const LineAddr &as, const LineAddr &ad,
                                dim3 grid, int Lx, const R *p2tab, R scale, LaunchStream stream) {
#define LGF_GO(LEN)                                                                                              \
    if (L == LEN) {                                                                                              \
        if (mode == FFT_FWD) k_slab_fft_line2<R, LEN, FFT_FWD><<<grid, 2 * LINE2_LINES, 0, stream>>>(src, dst, as, ad, Lx, p2tab, scale); \
        else if (mode == FFT_INV) k_slab_fft_line2<R, LEN, FFT_INV><<<grid, 2 * LINE2_LINES, 0, stream>>>(src, dst, as, ad, Lx, p2tab, scale); \
        else k_slab_fft_line2<R, LEN, FFT_FWD_SCALE_INV><<<grid, 2 * LINE2_LINES, 0, stream>>>(src, dst, as, ad, Lx, p2tab, scale); \
        return cudaGetLastError();                                                                               \
    }
    LGF_GO(16) LGF_GO(32) LGF_GO(64)
#undef LGF_GO
    return cudaErrorInvalidValue;
}

template <class R, int L>
static cudaError_t launch_line_L(int mode, const C<R> *src, C<R> *dst, const LineAddr &as, const LineAddr &ad, int nlo,
                                 dim3 grid, int Lx, const R *twiddle, const R *p2tab, R scale, LaunchStream stream) {
    const size_t smem = (64 + (size_t)L * nlo) * sizeof(C<R>);
    const C<R> *tw = reinterpret_cast<const C<R> *>(twiddle);
    auto go = [&](auto kern) {
        if (cudaError_t e = ensure_dynamic_smem(kern, smem); e != cudaSuccess) return e;
        kern<<<grid, 256, smem, stream>>>(src, dst, as, ad, nlo, Lx, tw, p2tab, scale);
        return cudaGetLastError();
    };
    if (mode == FFT_FWD) return go(k_slab_fft_line<R, L, FFT_FWD>);
    if (mode == FFT_INV) return go(k_slab_fft_line<R, L, FFT_INV>);
    return go(k_slab_fft_line<R, L, FFT_FWD_SCALE_INV>);
}
template <class R>
static cudaError_t launch_line(int L, int mode, const C<R> *src, C<R> *dst, const LineAddr &as, const LineAddr &ad, int nlo,
                               dim3 grid, int Lx, const R *twiddle, const R *p2tab, R scale, LaunchStream stream) {
    switch (L) {
#define LGF_CASE(LEN) case LEN: return launch_line_L<R, LEN>(mode, src, dst, as, ad, nlo, grid, Lx, twiddle, p2tab, scale, stream);
        LGF_CASE(2) LGF_CASE(3) LGF_CASE(4) LGF_CASE(6) LGF_CASE(8) LGF_CASE(12) LGF_CASE(16) LGF_CASE(24)
        LGF_CASE(32) LGF_CASE(48) LGF_CASE(64)
#undef LGF_CASE
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace lgf

using namespace lgf;

struct lgf_slab {
    int dims[4];
    int rank = 0, N = 1, T = 0, Zl = 0;
    int prec = 0, nr = 3;
    Geom gl{};                   // the slab: (Lx, Ly, Lz, T)
    long long Vglobal = 0;
    cudaStream_t stream = nullptr;
    void *lbuf[2] = {nullptr, nullptr};   // C<R>[4][3 nr][Vl] each: the fused sweep reads one and writes the other;
                                          // which one is current is st->cur, on the device (k_finalize flips it)
    int device = 0;              // the CUDA device the buffers live on
    void *uhalo = nullptr;       // C<R>[3 nr][S3]   U_t of the slice below the slab
    void *W = nullptr;           // C<R>[4][Vl]      packed Delta / w, t-slab order
    void *G = nullptr;           // C<R>[6][Vl]
    void *ghalo = nullptr;       // C<R>[6][S3]      g of the slice above the slab
    void *glo = nullptr;         // C<R>[6][S3]      g of the slice below the slab (fused sweep only)
    bool uhalo_valid = false;    // uhalo holds U_t of the slice below for the CURRENT configuration
    double *partial = nullptr;
    int nb = 0;
    DevState *st = nullptr;      // device-resident control block (lgf_state.cuh): done / nan flags, counters, F, theta, cur
    SweepMaps *sweep_maps = nullptr;   // TMA tensor maps of the staged sweep (lgf_sweep_tma.cu), or null
    DevState *h_poll = nullptr;  // pinned: two slots for the asynchronous looks at the state (lgf_slab_poll)
    cudaEvent_t poll_ev[2] = {nullptr, nullptr};
    int polls_enq = 0, polls_seen = 0;
    double *hist = nullptr;      // (F, theta) pairs, device
    long long hist_cap = 0;
    void *twiddle[4] = {nullptr, nullptr, nullptr, nullptr};
    void *p2tab = nullptr;       // R[4][64], z section shifted to this rank's z-slab
    AxisPass pass_fwd[2], pass_inv[2];   // x, y one axis per pass (any supported length), used unless xy_reg
    bool xy_reg = false;         // (x, y) planes by the register-line sweeps of lgf_fft_reg2.cu (square planes of 16 / 32 / 64)
    bool xy_gout = false;        // ... and the inverse one can end with the g-build (a5)
    int nlo_z = 1, nlo_t = 1;    // consecutive (x, y) indices per CTA of the z / t line passes
    bool by_comp = false;        // the per-component entry points (*_comp) are available: register-line passes on x, y, z and t
    bool z_reg = false, t_reg = false;   // z / t lines in registers (k_slab_fft_line2): natural frequency order on that axis
    LineAddr a_w{}, a_zbuf{}, a_tbuf{};
    bool have_links = false;
    long long launches = 0;
    std::string err;
};

static thread_local std::string g_slab_err;

static int sfail(lgf_slab *ctx, int code, const std::string &msg) {
    if (ctx) ctx->err = msg;
    g_slab_err = msg;
    return code;
}
#define SCK(call)                                                                                     \
    do {                                                                                              \
        cudaError_t e_ = (call);                                                                      \
        if (e_ != cudaSuccess)                                                                        \
            return sfail(ctx, e_ == cudaErrorMemoryAllocation ? LGF_ENOMEM : LGF_ECUDA,               \
                         std::string(#call) + ": " + cudaGetErrorString(e_));                         \
    } while (0)

// every entry point runs on the device the context was created on (the caller may have another one current)
#define SLAB_ENTER(ctx)                                                                               \
    do {                                                                                              \
        cudaError_t e_ = cudaSetDevice((ctx)->device);                                                \
        if (e_ != cudaSuccess) return sfail(ctx, LGF_ECUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e_)); \
    } while (0)

static long long divisor_le(long long n, long long cap) {
    if (cap < 1) cap = 1;
    for (long long d = (cap < n ? cap : n); d >= 1; d--)
        if (n % d == 0) return d;
    return 1;
}

// one in-place shared-memory pass over one axis of geometry g (k_fft_axis of lgf_fft.cu)
static AxisPass slab_axis_pass(const Geom &g, int prec, int axis, int mode) {
    const long long TILE = 2048;
    const size_t cbytes = 2 * (size_t)prec;
    AxisPass p{};
    p.kind = PASS_AXIS;
    p.axis = axis;
    p.L = g.L[axis];
    p.mode = mode;
    p.S = g.S[axis];
    p.H = g.V / (p.S * p.L);
    if (p.S == 1) {
        p.nlo = 1;
        p.nhi = (int)divisor_le(p.H, TILE / p.L);
        p.smem = (64 + (size_t)p.nhi * (p.L | 1)) * cbytes;
    } else {
        p.nlo = (int)divisor_le(p.S, TILE / p.L);
        p.nhi = (int)divisor_le(p.H, TILE / ((long long)p.L * p.nlo));
        p.smem = (64 + (size_t)p.nhi * p.L * p.nlo) * cbytes;
    }
    p.threads = 256;
    return p;
}

template <class R>
static int slab_tables(lgf_slab *ctx) {
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->dims[mu];
        std::vector<R> tw(2 * 64, (R)0);
        for (int m = 0; m < L; m++) {
            double c, s;
            host_cossin_2pi(m, L, c, s);
            tw[2 * m] = (R)c;
            tw[2 * m + 1] = (R)(-s);
        }
        SCK(cudaMalloc(&ctx->twiddle[mu], sizeof(R) * 2 * 64));
        SCK(cudaMemcpy(ctx->twiddle[mu], tw.data(), sizeof(R) * 2 * 64, cudaMemcpyHostToDevice));
    }
    // 4 sin^2(pi k / L) by POSITION along each axis (the per-axis passes leave position p = N2 k1 + k2 holding
    // frequency k = k1 + N1 k2, lgf_fft.cu); the z section holds the positions of this rank's z-slab
    std::vector<R> p2(4 * 64, (R)0);
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->dims[mu];
        int N1, N2;
        host_line_factor(L, N1, N2);
        const int first = mu == 2 ? ctx->rank * ctx->Zl : 0, count = mu == 2 ? ctx->Zl : L;
        const bool natural = mu < 2 ? ctx->xy_reg : (mu == 2 ? ctx->z_reg : ctx->t_reg);   // register-line passes: natural order
        for (int i = 0; i < count; i++) {
            const int p = first + i, k = natural ? p : (p / N2) + N1 * (p % N2);
            double c, s;
            host_cossin_2pi(k, 2 * L, c, s);
            p2[mu * 64 + i] = (R)(4.0 * s * s);
        }
    }
    SCK(cudaMalloc(&ctx->p2tab, sizeof(R) * 4 * 64));
    SCK(cudaMemcpy(ctx->p2tab, p2.data(), sizeof(R) * 4 * 64, cudaMemcpyHostToDevice));
    return LGF_OK;
}

// forward x, y (in place in W), then forward z from W into the send buffer of the first all-to-all
template <class R>
static int slab_fft_forward(lgf_slab *ctx, void *d_send) {
    const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2], (const R *)ctx->twiddle[3]};
    if (ctx->xy_reg) {
        SCK(launch_fft_reg2<R>(0, ctx->gl, (C<R> *)ctx->W, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream, nullptr, (R)0));
        ctx->launches++;
    } else {
        for (int i = 0; i < 2; i++) {
            SCK(launch_fft_pass<R>(ctx->pass_fwd[i], (C<R> *)ctx->W, ctx->gl, tw, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream));
            ctx->launches++;
        }
    }
    if (ctx->z_reg) {
        SCK(launch_line2<R>(ctx->dims[2], FFT_FWD, (const C<R> *)ctx->W, (C<R> *)d_send, ctx->a_w, ctx->a_zbuf,
                            dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->T, 4), ctx->dims[0], (const R *)ctx->p2tab, (R)0, ctx->stream));
        ctx->launches++;
        return LGF_OK;
    }
    const dim3 grid((unsigned)(ctx->gl.S[2] / ctx->nlo_z), ctx->T, 4);
    SCK(launch_line<R>(ctx->dims[2], FFT_FWD, (const C<R> *)ctx->W, (C<R> *)d_send, ctx->a_w, ctx->a_zbuf, ctx->nlo_z, grid,
                       ctx->dims[0], tw[2], (const R *)ctx->p2tab, (R)0, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

// the t lines, from the receive buffer of the first all-to-all into the send buffer of the second
template <class R>
static int slab_fft_t(lgf_slab *ctx, const void *d_recv, void *d_send) {
    const R scale = (R)(16.0 / (double)ctx->Vglobal);              // p2max / V (Alg. 1 lines 5, 7; R5)
    if (ctx->t_reg) {
        SCK(launch_line2<R>(ctx->dims[3], FFT_FWD_SCALE_INV, (const C<R> *)d_recv, (C<R> *)d_send, ctx->a_tbuf, ctx->a_tbuf,
                            dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->Zl, 4), ctx->dims[0], (const R *)ctx->p2tab, scale, ctx->stream));
        ctx->launches++;
        return LGF_OK;
    }
    const dim3 grid((unsigned)(ctx->gl.S[2] / ctx->nlo_t), ctx->Zl, 4);
    SCK(launch_line<R>(ctx->dims[3], FFT_FWD_SCALE_INV, (const C<R> *)d_recv, (C<R> *)d_send, ctx->a_tbuf, ctx->a_tbuf, ctx->nlo_t,
                       grid, ctx->dims[0], (const R *)ctx->twiddle[3], (const R *)ctx->p2tab, scale, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

// inverse z from the receive buffer of the second all-to-all into W, then inverse y, x; with_g: ending in a5
template <class R>
static int slab_fft_inverse(lgf_slab *ctx, const void *d_recv, bool with_g, double alpha) {
    const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2], (const R *)ctx->twiddle[3]};
    if (ctx->z_reg) {
        SCK(launch_line2<R>(ctx->dims[2], FFT_INV, (const C<R> *)d_recv, (C<R> *)ctx->W, ctx->a_zbuf, ctx->a_w,
                            dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->T, 4), ctx->dims[0], (const R *)ctx->p2tab, (R)0, ctx->stream));
    } else {
        const dim3 grid((unsigned)(ctx->gl.S[2] / ctx->nlo_z), ctx->T, 4);
        SCK(launch_line<R>(ctx->dims[2], FFT_INV, (const C<R> *)d_recv, (C<R> *)ctx->W, ctx->a_zbuf, ctx->a_w, ctx->nlo_z, grid,
                           ctx->dims[0], tw[2], (const R *)ctx->p2tab, (R)0, ctx->stream));
    }
    ctx->launches++;
    const R ha = (R)(0.5 * alpha);
    if (ctx->xy_reg) {
        const bool fuse = with_g && ctx->xy_gout;
        SCK(launch_fft_reg2<R>(fuse ? 3 : 2, ctx->gl, (C<R> *)ctx->W, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream,
                               (C<R> *)ctx->G, ha));
        ctx->launches++;
        if (fuse) return LGF_OK;
    } else {
        for (int i = 0; i < 2; i++) {
            SCK(launch_fft_pass<R>(ctx->pass_inv[i], (C<R> *)ctx->W, ctx->gl, tw, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream));
            ctx->launches++;
        }
    }
    if (with_g) {
        SCK(launch_gbuild<R>((const C<R> *)ctx->W, (C<R> *)ctx->G, ctx->gl, ha, ctx->st, ctx->stream));
        ctx->launches++;
    }
    return LGF_OK;
}

// ---- the same passes for ONE packed component c (the four components of W are independent fields): what lets the
// exchange of component c run on another stream while component c + 1 is being transformed (slab.py)
template <class R>
static int slab_fft_forward_comp(lgf_slab *ctx, void *d_send, int c) {
    SCK(launch_fft_reg2<R>(0, ctx->gl, (C<R> *)ctx->W, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream, nullptr, (R)0, false, c));
    SCK(launch_line2<R>(ctx->dims[2], FFT_FWD, (const C<R> *)ctx->W + c * ctx->a_w.stride_c, (C<R> *)d_send + c * ctx->a_zbuf.stride_c,
                        ctx->a_w, ctx->a_zbuf, dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->T, 1), ctx->dims[0],
                        (const R *)ctx->p2tab, (R)0, ctx->stream));
    ctx->launches += 2;
    return LGF_OK;
}
template <class R>
static int slab_fft_t_comp(lgf_slab *ctx, const void *d_recv, void *d_send, int c) {
    const R scale = (R)(16.0 / (double)ctx->Vglobal);              // p2max / V (Alg. 1 lines 5, 7; R5)
    SCK(launch_line2<R>(ctx->dims[3], FFT_FWD_SCALE_INV, (const C<R> *)d_recv + c * ctx->a_tbuf.stride_c,
                        (C<R> *)d_send + c * ctx->a_tbuf.stride_c, ctx->a_tbuf, ctx->a_tbuf,
                        dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->Zl, 1), ctx->dims[0], (const R *)ctx->p2tab, scale, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}
template <class R>
static int slab_fft_zinv_comp(lgf_slab *ctx, const void *d_recv, int c) {
    SCK(launch_line2<R>(ctx->dims[2], FFT_INV, (const C<R> *)d_recv + c * ctx->a_zbuf.stride_c, (C<R> *)ctx->W + c * ctx->a_w.stride_c,
                        ctx->a_zbuf, ctx->a_w, dim3((unsigned)(ctx->gl.S[2] / LINE2_LINES), ctx->T, 1), ctx->dims[0],
                        (const R *)ctx->p2tab, (R)0, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}
// inverse (x, y) sweep of all four components (ending in a5 with_g: the g-build needs all of w(x) on chip)
template <class R>
static int slab_fft_xyinv(lgf_slab *ctx, bool with_g, double alpha) {
    const R ha = (R)(0.5 * alpha);
    const bool fuse = with_g && ctx->xy_gout;
    SCK(launch_fft_reg2<R>(fuse ? 3 : 2, ctx->gl, (C<R> *)ctx->W, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream, (C<R> *)ctx->G, ha));
    ctx->launches++;
    if (with_g && !fuse) {
        SCK(launch_gbuild<R>((const C<R> *)ctx->W, (C<R> *)ctx->G, ctx->gl, ha, ctx->st, ctx->stream));
        ctx->launches++;
    }
    return LGF_OK;
}

template <class R>
static LinkPair<R> slab_links(lgf_slab *ctx) {
    LinkPair<R> lp;
    lp.buf[0] = (C<R> *)ctx->lbuf[0];
    lp.buf[1] = (C<R> *)ctx->lbuf[1];
    return lp;
}
template <class R>
static SweepHalo<R> slab_halo(lgf_slab *ctx) {
    SweepHalo<R> h;
    h.ghi = (const C<R> *)ctx->ghalo;
    h.glo = (const C<R> *)ctx->glo;
    h.uhalo = (C<R> *)ctx->uhalo;
    return h;
}
// a1 on the slab: the one-GPU path's k_delta with the U_t halo (lgf_links.cu); `stop` = the word that makes it return
template <class R>
static int slab_delta(lgf_slab *ctx, double *d_sums, const int *stop) {
    int nb = 0;
    SCK(launch_delta<R>(ctx->nr, slab_links<R>(ctx), (C<R> *)ctx->W, ctx->gl, ctx->partial, &nb, stop, ctx->st, ctx->stream,
                        slab_halo<R>(ctx)));
    k_slab_sum2<<<1, SLAB_THREADS, 0, ctx->stream>>>(ctx->partial, nb, d_sums, stop);
    SCK(cudaGetLastError());
    ctx->launches += 2;
    return LGF_OK;
}

template <class R>
static int slab_update(lgf_slab *ctx) {
    if (ctx->nr == 3)
        k_slab_update<R, 3><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>(slab_links<R>(ctx), (const C<R> *)ctx->G,
                                                                       (const C<R> *)ctx->ghalo, ctx->gl, ctx->st);
    else
        k_slab_update<R, 2><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>(slab_links<R>(ctx), (const C<R> *)ctx->G,
                                                                       (const C<R> *)ctx->ghalo, ctx->gl, ctx->st);
    SCK(cudaGetLastError());
    ctx->launches++;
    return LGF_OK;
}

// a6 + a1 fused: the one-GPU path's k_sweep with the halo policy (g of both neighbouring slices, U_t of the slice
// below read from and stored back into its halo copy); new links into the other buffer -- lgf_slab_finalize flips
template <class R>
static int slab_sweep(lgf_slab *ctx, double *d_sums) {
    int nb = 0;
    if (ctx->sweep_maps && sweep_tma_auto(ctx->gl, ctx->nr, ctx->prec))      // as the one-GPU context: where it measured faster
        SCK(launch_sweep_tma<R>(ctx->sweep_maps, ctx->nr, slab_links<R>(ctx), (const C<R> *)ctx->G, (C<R> *)ctx->W, ctx->gl,
                                ctx->partial, &nb, ctx->st, LaunchStream(ctx->stream, false), 1, false, slab_halo<R>(ctx)));
    else
    SCK(launch_sweep<R>(ctx->nr, slab_links<R>(ctx), (const C<R> *)ctx->G, (C<R> *)ctx->W, ctx->gl, ctx->partial, &nb, ctx->st,
                        LaunchStream(ctx->stream, false), 1, false, -1, 0, 0, slab_halo<R>(ctx)));
    k_slab_sum2<<<1, SLAB_THREADS, 0, ctx->stream>>>(ctx->partial, nb, d_sums, &ctx->st->done);
    SCK(cudaGetLastError());
    ctx->launches += 2;
    return LGF_OK;
}

extern "C" {

const char *lgf_slab_last_error(const lgf_slab *ctx) { return ctx ? ctx->err.c_str() : g_slab_err.c_str(); }

int lgf_slab_destroy(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    void *bufs[] = {ctx->lbuf[0], ctx->lbuf[1], ctx->uhalo, ctx->W, ctx->G, ctx->ghalo, ctx->glo, ctx->partial, ctx->st, ctx->p2tab,
                    ctx->twiddle[0], ctx->twiddle[1], ctx->twiddle[2], ctx->twiddle[3], ctx->hist};
    for (void *b : bufs) cudaFree(b);
    sweep_tma_maps_destroy(ctx->sweep_maps);
    if (ctx->h_poll) cudaFreeHost(ctx->h_poll);
    for (int k = 0; k < 2; k++) if (ctx->poll_ev[k]) cudaEventDestroy(ctx->poll_ev[k]);
    cudaGetLastError();
    delete ctx;
    return LGF_OK;
}

int lgf_slab_create(const int dims[4], int precision, int link_storage, int rank, int nranks, lgf_slab **out) {
    if (!dims || !out) return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: null argument");
    *out = nullptr;
    if (precision != LGF_FP32 && precision != LGF_FP64) return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: bad precision");
    if (link_storage != LGF_LINKS_18 && link_storage != LGF_LINKS_12)
        return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: bad link_storage");
    for (int mu = 0; mu < 4; mu++)
        if (!host_valid_len(dims[mu])) return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: unsupported lattice extent");
    if (nranks < 1 || rank < 0 || rank >= nranks) return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: bad rank / nranks");
    if (dims[3] % nranks != 0 || dims[2] % nranks != 0)
        return sfail(nullptr, LGF_EINVAL, "lgf_slab_create: nranks must divide both Lt (t-slabs) and Lz (z-slabs of the t pass)");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return sfail(nullptr, LGF_ECUDA, "lgf_slab_create: no CUDA device (liblgf has no CPU path)");
    }
    lgf_slab *ctx = new (std::nothrow) lgf_slab();
    if (!ctx) return sfail(nullptr, LGF_ENOMEM, "lgf_slab_create: host allocation failed");
    cudaGetDevice(&ctx->device);                              // every later call runs on this device (slab_enter)
    ctx->prec = precision;
    ctx->nr = link_storage == LGF_LINKS_18 ? 3 : 2;
    ctx->rank = rank;
    ctx->N = nranks;
    ctx->T = dims[3] / nranks;
    ctx->Zl = dims[2] / nranks;
    ctx->Vglobal = 1;
    for (int mu = 0; mu < 4; mu++) { ctx->dims[mu] = dims[mu]; ctx->Vglobal *= dims[mu]; }
    const int Ll[4] = {dims[0], dims[1], dims[2], ctx->T};
    long long Sl = 1;
    for (int mu = 0; mu < 4; mu++) { ctx->gl.L[mu] = Ll[mu]; ctx->gl.S[mu] = Sl; Sl *= Ll[mu]; }
    ctx->gl.V = Sl;
    ctx->xy_reg = fft_reg2_xy_supported(ctx->gl);
    ctx->xy_gout = fft_reg2_xy_gout(ctx->gl, precision);
    {   // address maps of the line passes (LineAddr) and their tiles: about 2048 complex elements per CTA
        const long long Sxy = ctx->gl.S[2], piece = (long long)ctx->T * ctx->Zl * Sxy;
        auto lg2 = [](int d) { int sh = 0; while ((1 << sh) < d) sh++; return (1 << sh) == d ? sh : -1; };
        ctx->a_w = LineAddr{Sl, (long long)dims[2] * Sxy, 0, Sxy, dims[2], lg2(dims[2])};
        ctx->a_zbuf = LineAddr{Sl, (long long)ctx->Zl * Sxy, piece, Sxy, ctx->Zl, lg2(ctx->Zl)};
        ctx->a_tbuf = LineAddr{Sl, Sxy, piece, (long long)ctx->Zl * Sxy, ctx->T, lg2(ctx->T)};
        auto reg_len = [](int L) { return L == 16 || L == 32 || L == 64; };
        ctx->z_reg = reg_len(dims[2]) && Sxy % LINE2_LINES == 0;          // nranks | L then makes Zl, T powers of two
        ctx->t_reg = reg_len(dims[3]) && Sxy % LINE2_LINES == 0;
        ctx->nlo_z = (int)divisor_le(Sxy, 2048 / dims[2]);
        ctx->nlo_t = (int)divisor_le(Sxy, 2048 / dims[3]);
    }
    const size_t V = (size_t)Sl, S3 = (size_t)ctx->gl.S[3], cb = 2 * (size_t)precision;
    ctx->nb = (int)((V + SLAB_THREADS - 1) / SLAB_THREADS);
    int rc = LGF_OK;
    auto alloc = [&](void **p, size_t bytes) {
        if (rc != LGF_OK) return;
        cudaError_t ee = cudaMalloc(p, bytes);
        if (ee != cudaSuccess) rc = sfail(ctx, ee == cudaErrorMemoryAllocation ? LGF_ENOMEM : LGF_ECUDA,
                                          std::string("cudaMalloc: ") + cudaGetErrorString(ee));
    };
    alloc(&ctx->lbuf[0], V * 4 * 3 * ctx->nr * cb);
    alloc(&ctx->lbuf[1], V * 4 * 3 * ctx->nr * cb);
    alloc(&ctx->uhalo, S3 * 3 * ctx->nr * cb);
    alloc(&ctx->W, V * 4 * cb);
    alloc(&ctx->G, V * 6 * cb);
    alloc(&ctx->ghalo, S3 * 6 * cb);
    alloc(&ctx->glo, S3 * 6 * cb);
    alloc((void **)&ctx->partial, sizeof(double) * 2 * (2 * ctx->nb + 1));
    alloc((void **)&ctx->st, sizeof(DevState));
    ctx->hist_cap = 1 << 20;
    alloc((void **)&ctx->hist, sizeof(double) * 2 * ctx->hist_cap);
    if (rc == LGF_OK) {
        cudaError_t ee = cudaMemset(ctx->st, 0, sizeof(DevState));
        if (ee == cudaSuccess) ee = cudaMallocHost((void **)&ctx->h_poll, 2 * sizeof(DevState));
        for (int k = 0; k < 2 && ee == cudaSuccess; k++) ee = cudaEventCreateWithFlags(&ctx->poll_ev[k], cudaEventDisableTiming);
        if (ee != cudaSuccess) rc = sfail(ctx, LGF_ECUDA, std::string("state / poll buffers: ") + cudaGetErrorString(ee));
    }
    if (rc == LGF_OK) rc = precision == LGF_FP64 ? slab_tables<double>(ctx) : slab_tables<float>(ctx);
    if (rc != LGF_OK) {
        g_slab_err = ctx->err;
        lgf_slab_destroy(ctx);
        return rc;
    }
    ctx->by_comp = ctx->xy_reg && ctx->z_reg && ctx->t_reg && fft_reg2_xy_by_component(ctx->gl, precision);
    ctx->sweep_maps = sweep_tma_maps_create(ctx->gl, ctx->nr, precision, ctx->lbuf[0], ctx->lbuf[1], ctx->G);
    for (int a = 0; a < 2; a++) {
        ctx->pass_fwd[a] = slab_axis_pass(ctx->gl, precision, a, FFT_FWD);
        ctx->pass_inv[a] = slab_axis_pass(ctx->gl, precision, 1 - a, FFT_INV);
    }
    *out = ctx;
    return LGF_OK;
}

int lgf_slab_set_stream(lgf_slab *ctx, void *cuda_stream) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    SCK(cudaStreamSynchronize(ctx->stream));             // work enqueued on the old stream is not ordered with the new one
    ctx->stream = (cudaStream_t)cuda_stream;
    return LGF_OK;
}

int lgf_slab_set_links(lgf_slab *ctx, const void *d_links) {
    if (!ctx || !d_links) return sfail(ctx, LGF_EINVAL, "lgf_slab_set_links: null argument");
    SLAB_ENTER(ctx);
    ctx->uhalo_valid = false;
    if (ctx->prec == LGF_FP64) SCK(launch_convert_in<double>(ctx->nr, (const double *)d_links, (C<double> *)ctx->lbuf[0], ctx->gl, ctx->stream));
    else SCK(launch_convert_in<float>(ctx->nr, (const float *)d_links, (C<float> *)ctx->lbuf[0], ctx->gl, ctx->stream));
    SCK(launch_reset_state(ctx->st, ctx->stream));       // buffer 0 current, counters, history and flags cleared
    ctx->launches += 2;
    ctx->have_links = true;
    return LGF_OK;
}

int lgf_slab_get_links(lgf_slab *ctx, void *d_links) {
    if (!ctx || !d_links) return sfail(ctx, LGF_EINVAL, "lgf_slab_get_links: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_get_links: no configuration loaded");
    SLAB_ENTER(ctx);
    if (ctx->prec == LGF_FP64)
        SCK(launch_convert_out<double>(ctx->nr, slab_links<double>(ctx), (double *)d_links, ctx->gl, ctx->st, ctx->stream));
    else
        SCK(launch_convert_out<float>(ctx->nr, slab_links<float>(ctx), (float *)d_links, ctx->gl, ctx->st, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

long long lgf_slab_halo_elems(const lgf_slab *ctx, int which) {
    if (!ctx || (which != LGF_HALO_LINKS && which != LGF_HALO_G && which != LGF_HALO_G_UP)) return LGF_EINVAL;
    return (long long)ctx->gl.S[3] * (which == LGF_HALO_LINKS ? 3 * ctx->nr : 6) * 2;
}

int lgf_slab_halo_pack(lgf_slab *ctx, int which, void *d_send) {
    if (!ctx || !d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_pack: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_halo_pack: no configuration loaded");
    SLAB_ENTER(ctx);
    const size_t cb = 2 * (size_t)ctx->prec, S3 = (size_t)ctx->gl.S[3], V = (size_t)ctx->gl.V;
    if (which == LGF_HALO_LINKS) {          // U_t of the LAST local slice of the current buffer, for the rank above
        const int np = 3 * ctx->nr;
        const int nb = (int)((S3 * np + SLAB_THREADS - 1) / SLAB_THREADS);
        if (ctx->prec == LGF_FP64)
            k_slab_pack_ut<double><<<nb, SLAB_THREADS, 0, ctx->stream>>>(slab_links<double>(ctx), (C<double> *)d_send, (long long)V,
                                                                       (long long)S3, np, (long long)(S3 * (ctx->T - 1)), ctx->st);
        else
            k_slab_pack_ut<float><<<nb, SLAB_THREADS, 0, ctx->stream>>>(slab_links<float>(ctx), (C<float> *)d_send, (long long)V,
                                                                      (long long)S3, np, (long long)(S3 * (ctx->T - 1)), ctx->st);
        SCK(cudaGetLastError());
        ctx->launches++;
    } else if (which == LGF_HALO_G) {       // g of the FIRST local slice, for the rank below
        SCK(cudaMemcpy2DAsync(d_send, S3 * cb, ctx->G, V * cb, S3 * cb, 6, cudaMemcpyDeviceToDevice, ctx->stream));
    } else if (which == LGF_HALO_G_UP) {    // g of the LAST local slice, for the rank above (fused sweep)
        const char *src = (const char *)ctx->G + S3 * (ctx->T - 1) * cb;
        SCK(cudaMemcpy2DAsync(d_send, S3 * cb, src, V * cb, S3 * cb, 6, cudaMemcpyDeviceToDevice, ctx->stream));
    } else return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_pack: bad halo id");
    return LGF_OK;
}

int lgf_slab_halo_unpack(lgf_slab *ctx, int which, const void *d_recv) {
    if (!ctx || !d_recv) return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_unpack: null argument");
    SLAB_ENTER(ctx);
    const size_t cb = 2 * (size_t)ctx->prec, S3 = (size_t)ctx->gl.S[3];
    if (which == LGF_HALO_LINKS) {
        SCK(cudaMemcpyAsync(ctx->uhalo, d_recv, S3 * 3 * ctx->nr * cb, cudaMemcpyDeviceToDevice, ctx->stream));
        ctx->uhalo_valid = true;
    } else if (which == LGF_HALO_G_UP) SCK(cudaMemcpyAsync(ctx->glo, d_recv, S3 * 6 * cb, cudaMemcpyDeviceToDevice, ctx->stream));
    else if (which == LGF_HALO_G) SCK(cudaMemcpyAsync(ctx->ghalo, d_recv, S3 * 6 * cb, cudaMemcpyDeviceToDevice, ctx->stream));
    else return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_unpack: bad halo id");
    return LGF_OK;
}

int lgf_slab_delta(lgf_slab *ctx, double *d_sums) {
    if (!ctx || !d_sums) return sfail(ctx, LGF_EINVAL, "lgf_slab_delta: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_delta: no configuration loaded");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_delta<double>(ctx, d_sums, &ctx->st->zero) : slab_delta<float>(ctx, d_sums, &ctx->st->zero);
}

int lgf_slab_fft_forward(lgf_slab *ctx, void *d_send) {
    if (!ctx || !d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_forward: null argument");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_fft_forward<double>(ctx, d_send) : slab_fft_forward<float>(ctx, d_send);
}

int lgf_slab_fft_t(lgf_slab *ctx, const void *d_recv, void *d_send) {
    if (!ctx || !d_recv || !d_send || d_recv == d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_t: bad argument");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_fft_t<double>(ctx, d_recv, d_send) : slab_fft_t<float>(ctx, d_recv, d_send);
}

int lgf_slab_fft_inverse(lgf_slab *ctx, const void *d_recv) {
    if (!ctx || !d_recv) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_inverse: null argument");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_fft_inverse<double>(ctx, d_recv, false, 0.0) : slab_fft_inverse<float>(ctx, d_recv, false, 0.0);
}

int lgf_slab_fft_inverse_g(lgf_slab *ctx, const void *d_recv, double alpha) {
    if (!ctx || !d_recv) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_inverse_g: null argument");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_fft_inverse<double>(ctx, d_recv, true, alpha) : slab_fft_inverse<float>(ctx, d_recv, true, alpha);
}

int lgf_slab_by_component(const lgf_slab *ctx) { return ctx ? (ctx->by_comp ? 1 : 0) : LGF_EINVAL; }

#define SLAB_COMP_ENTER(name)                                                                         \
    if (!ctx) return LGF_EINVAL;                                                                      \
    if (!ctx->by_comp) return sfail(ctx, LGF_ESTATE, name ": per-component passes are not available for this lattice (lgf_slab_by_component)"); \
    if (comp < 0 || comp > 3) return sfail(ctx, LGF_EINVAL, name ": component must be 0..3");         \
    SLAB_ENTER(ctx)

int lgf_slab_fft_forward_comp(lgf_slab *ctx, void *d_send, int comp) {
    SLAB_COMP_ENTER("lgf_slab_fft_forward_comp");
    if (!d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_forward_comp: null argument");
    return ctx->prec == LGF_FP64 ? slab_fft_forward_comp<double>(ctx, d_send, comp) : slab_fft_forward_comp<float>(ctx, d_send, comp);
}

int lgf_slab_fft_t_comp(lgf_slab *ctx, const void *d_recv, void *d_send, int comp) {
    SLAB_COMP_ENTER("lgf_slab_fft_t_comp");
    if (!d_recv || !d_send || d_recv == d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_t_comp: bad argument");
    return ctx->prec == LGF_FP64 ? slab_fft_t_comp<double>(ctx, d_recv, d_send, comp) : slab_fft_t_comp<float>(ctx, d_recv, d_send, comp);
}

int lgf_slab_fft_zinv_comp(lgf_slab *ctx, const void *d_recv, int comp) {
    SLAB_COMP_ENTER("lgf_slab_fft_zinv_comp");
    if (!d_recv) return sfail(ctx, LGF_EINVAL, "lgf_slab_fft_zinv_comp: null argument");
    return ctx->prec == LGF_FP64 ? slab_fft_zinv_comp<double>(ctx, d_recv, comp) : slab_fft_zinv_comp<float>(ctx, d_recv, comp);
}

int lgf_slab_fft_xyinv(lgf_slab *ctx, int with_g, double alpha) {
    if (!ctx) return LGF_EINVAL;
    if (!ctx->by_comp) return sfail(ctx, LGF_ESTATE, "lgf_slab_fft_xyinv: per-component passes are not available for this lattice");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_fft_xyinv<double>(ctx, with_g != 0, alpha) : slab_fft_xyinv<float>(ctx, with_g != 0, alpha);
}

int lgf_slab_gbuild(lgf_slab *ctx, double alpha) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    if (ctx->prec == LGF_FP64)
        SCK(launch_gbuild<double>((const C<double> *)ctx->W, (C<double> *)ctx->G, ctx->gl, 0.5 * alpha, ctx->st, ctx->stream));
    else
        SCK(launch_gbuild<float>((const C<float> *)ctx->W, (C<float> *)ctx->G, ctx->gl, (float)(0.5 * alpha), ctx->st, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

int lgf_slab_update(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_update: no configuration loaded");
    SLAB_ENTER(ctx);
    ctx->uhalo_valid = false;                // the neighbour's U_t changed too: exchange it again before the next delta
    return ctx->prec == LGF_FP64 ? slab_update<double>(ctx) : slab_update<float>(ctx);
}

int lgf_slab_sweep(lgf_slab *ctx, double *d_sums) {
    if (!ctx || !d_sums) return sfail(ctx, LGF_EINVAL, "lgf_slab_sweep: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_sweep: no configuration loaded");
    if (!ctx->uhalo_valid)
        return sfail(ctx, LGF_ESTATE, "lgf_slab_sweep: the U_t halo is not current (halo_unpack(LGF_HALO_LINKS) after set_links / update)");
    SLAB_ENTER(ctx);
    return ctx->prec == LGF_FP64 ? slab_sweep<double>(ctx, d_sums) : slab_sweep<float>(ctx, d_sums);
}

int lgf_slab_get_field(lgf_slab *ctx, void *d_field) {
    if (!ctx || !d_field) return sfail(ctx, LGF_EINVAL, "lgf_slab_get_field: null argument");
    SLAB_ENTER(ctx);
    if (ctx->prec == LGF_FP64) SCK(launch_field_get<double>((const C<double> *)ctx->W, (double *)d_field, ctx->gl, ctx->stream));
    else SCK(launch_field_get<float>((const C<float> *)ctx->W, (float *)d_field, ctx->gl, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

/* ---- Algorithm 1's control on the device: the slab twin of the one-GPU path's finalize ---- */
int lgf_slab_finalize(lgf_slab *ctx, const double *d_sums, double tol, int after_sweep, int record) {
    if (!ctx || !d_sums) return sfail(ctx, LGF_EINVAL, "lgf_slab_finalize: null argument");
    SLAB_ENTER(ctx);
    // k_finalize (lgf_links.cu) over ONE pair of sums, the all-reduced ones, normalised with the GLOBAL volume
    SCK(launch_finalize(d_sums, 1, ctx->Vglobal, tol, after_sweep, record, ctx->st, ctx->hist, ctx->hist_cap,
                        LaunchStream(ctx->stream, false)));
    ctx->launches++;
    return LGF_OK;
}

int lgf_slab_clear_done(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    SCK(launch_clear_done(ctx->st, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

int lgf_slab_poll(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    if (ctx->polls_enq - ctx->polls_seen >= 2) return sfail(ctx, LGF_ESTATE, "lgf_slab_poll: two looks are already outstanding");
    const int k = ctx->polls_enq & 1;
    SCK(cudaMemcpyAsync(&ctx->h_poll[k], ctx->st, sizeof(DevState), cudaMemcpyDeviceToHost, ctx->stream));
    SCK(cudaEventRecord(ctx->poll_ev[k], ctx->stream));
    ctx->polls_enq++;
    return LGF_OK;
}

int lgf_slab_poll_wait(lgf_slab *ctx, int *done, int *nan, long long *n_updates, double *F, double *theta) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    if (ctx->polls_enq == ctx->polls_seen) return sfail(ctx, LGF_ESTATE, "lgf_slab_poll_wait: no look outstanding");
    const int k = ctx->polls_seen & 1;
    SCK(cudaEventSynchronize(ctx->poll_ev[k]));
    ctx->polls_seen++;
    const DevState &h = ctx->h_poll[k];
    if (done) *done = h.done;
    if (nan) *nan = h.nan;
    if (n_updates) *n_updates = h.n_updates;
    if (F) *F = h.F;
    if (theta) *theta = h.theta;
    return LGF_OK;
}

long long lgf_slab_history_length(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    SLAB_ENTER(ctx);
    DevState h;
    SCK(cudaMemcpyAsync(&h, ctx->st, sizeof(DevState), cudaMemcpyDeviceToHost, ctx->stream));
    SCK(cudaStreamSynchronize(ctx->stream));
    return h.n_hist;
}

int lgf_slab_history(lgf_slab *ctx, long long first, long long count, double *F, double *theta) {
    if (!ctx || first < 0 || count < 0) return sfail(ctx, LGF_EINVAL, "lgf_slab_history: bad argument");
    const long long n = lgf_slab_history_length(ctx);
    if (n < 0) return (int)n;
    const long long have = n < ctx->hist_cap ? n : ctx->hist_cap;
    if (first + count > have) return sfail(ctx, LGF_EINVAL, "lgf_slab_history: range beyond the recorded entries");
    if (count == 0) return LGF_OK;
    std::vector<double> buf(2 * (size_t)count);
    SCK(cudaMemcpyAsync(buf.data(), ctx->hist + 2 * first, sizeof(double) * 2 * count, cudaMemcpyDeviceToHost, ctx->stream));
    SCK(cudaStreamSynchronize(ctx->stream));
    for (long long i = 0; i < count; i++) {
        if (F) F[i] = buf[2 * i];
        if (theta) theta[i] = buf[2 * i + 1];
    }
    return LGF_OK;
}

long long lgf_slab_launch_count(const lgf_slab *ctx) { return ctx ? ctx->launches : LGF_EINVAL; }

}  // extern "C"
