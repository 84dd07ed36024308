// lgf_slab.cu -- ONE configuration sharded over N ranks (the paper's
// stated future work; its CPU code does the same decomposition with PFFT over MPI, :124).
//
// Rank r of N owns the t-slab  t = r T .. (r+1) T - 1,  T = Lt / N  (all x, y, z), i.e. a contiguous slice of the
// canonical configuration.  One iteration of Algorithm 1 then needs exactly these exchanges:
//   a1    Delta(x) wants U_t(x - t) of the slice below the slab: one 3-D slice of U_t from rank r-1   (halo, LINKS)
//   a2-a4 x, y, z are whole inside the slab: transformed locally (lgf_fft.cu, one pass per axis); the t lines are
//         gathered by an ALL-TO-ALL that turns t-slabs into z-slabs (rank r gets z = r Zl .. (r+1) Zl - 1 of every
//         t, Zl = Lz / N), the t pass does forward + p2max / (V p2(k)) + inverse there, a second all-to-all goes back
//   a6    U_t(x) g(x + t)^dag wants g of the slice above the slab: one slice of g from rank r+1          (halo, G)
//   F, theta: per-rank sums, all-reduced by the caller (two doubles).
// This file holds the kernels and the per-rank context; the exchanges themselves are the caller's (NCCL through
// torch.distributed, paper_1206_0675_b200/slab.py): every entry point here is local to one rank and works on
// buffers the caller hands in, so no kernel ever waits on another rank.  The links are updated in place (a link
// transform reads no other link); Delta is recomputed by a pass of its own (the fused sweep of lgf_links.cu needs
// g(x - mu) as well, i.e. a second g halo: left for later).
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#include <new>
#include <string>
#include <vector>

#include "../../include/lgf.h"
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

// a1 on a slab.  g = local geometry (Lx, Ly, Lz, T); the backward t neighbour of the first local slice is read
// from `halo` (U_t of the slice below, C<R>[3 NR][S3]); x, y, z wrap inside the slab.
template <class R, int NR>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_delta(const C<R> *__restrict__ links, const C<R> *__restrict__ halo,
                                                             C<R> *__restrict__ W, Geom g, double *__restrict__ partial) {
    __shared__ double scratch[SLAB_THREADS / 32][2];
    const long long s = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x;
    double f = 0.0, t = 0.0;
    if (s < g.V) {
        int c[4];
        site_coords(g, s, c);
        Herm<R> d = herm_zero<R>();
        R retr = 0;
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            C<R> u[9];
            load_link<R, NR>(links, g.V, mu, s, u);
            retr += u[0].x + u[4].x + u[8].x;                       // eq. 3: Re tr U_mu(x)
            herm_sub(d, algebra_part(u));                           // - A_mu(x)
            if (mu == 3 && c[3] == 0) load_link<R, NR>(halo, g.S[3], 0, s, u);      // s < S3 here: the (x, y, z) index
            else load_link<R, NR>(links, g.V, mu, site_bwd(g, s, c, mu), u);
            herm_add(d, algebra_part(u));                           // + A_mu(x - mu)      (eq. 5)
        }
        store_herm(W, g.V, s, d);
        f = (double)retr;
        t = (double)herm_norm2(d);                                  // eq. 6: tr(Delta Delta^dag)
    }
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) {
        partial[2 * blockIdx.x] = f;
        partial[2 * blockIdx.x + 1] = t;
    }
}

// fixed-order sum of the per-block partial sums: out[0] = sum Re tr U, out[1] = sum tr(Delta Delta^dag) of the slab
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_sum2(const double *__restrict__ partial, int nb, double *__restrict__ out) {
    __shared__ double scratch[SLAB_THREADS / 32][2];
    double f = 0.0, t = 0.0;
    for (int i = threadIdx.x; i < nb; i += SLAB_THREADS) { f += partial[2 * i]; t += partial[2 * i + 1]; }
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) { out[0] = f; out[1] = t; }
}

// a6 on a slab, in place: U_mu(x) <- g(x) U_mu(x) g(x + mu)^dag (eq. 2, Alg. 1 line 14); g(x + t) of the last local
// slice comes from `ghalo` (rows 0, 1 of g on the slice above, C<R>[6][S3]).
template <class R, int NR>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_update(C<R> *__restrict__ links, const C<R> *__restrict__ G,
                                                              const C<R> *__restrict__ ghalo, Geom g) {
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

// The two index maps of the all-to-all.  Buffer element b = (((q 4 + c) T + tl) Zl + zl) Sxy + xy  (chunk q goes to /
// came from rank q; c = packed component of W; tl, zl local to the chunk).
//   side 0 (t-slab field  [c][tl][z][xy],  z = q Zl + zl):    w = c V + (tl Lz + q Zl + zl) Sxy + xy
//   side 1 (z-slab field  [c][t][zl][xy],  t = q T + tl):     w = c V + ((q T + tl) Zl + zl) Sxy + xy
// dir 0: buf[b] = field[w];  dir 1: field[w] = buf[b].
template <class R>
__global__ void __launch_bounds__(SLAB_THREADS) k_slab_transpose(C<R> *__restrict__ field, C<R> *__restrict__ buf, long long V,
                                                                 int Sxy, int T, int Zl, int N, int side, int dir) {
    const long long b = (long long)blockIdx.x * SLAB_THREADS + threadIdx.x;
    if (b >= 4 * V) return;
    long long r = b;
    const int xy = (int)(r % Sxy); r /= Sxy;
    const int zl = (int)(r % Zl); r /= Zl;
    const int tl = (int)(r % T); r /= T;
    const int c = (int)(r % 4);
    const int q = (int)(r / 4);
    const long long w = side == 0 ? (long long)c * V + ((long long)tl * (Zl * N) + q * Zl + zl) * Sxy + xy
                                  : (long long)c * V + (((long long)q * T + tl) * Zl + zl) * Sxy + xy;
    if (dir == 0) buf[b] = field[w];
    else field[w] = buf[b];
}

}  // namespace lgf

using namespace lgf;

struct lgf_slab {
    int dims[4];
    int rank = 0, N = 1, T = 0, Zl = 0;
    int prec = 0, nr = 3;
    Geom gl{};                   // the slab: (Lx, Ly, Lz, T)
    Geom gt{};                   // the z-slab the t pass works on: (Lx, Ly, Zl, Lt); same number of sites
    long long Vglobal = 0;
    cudaStream_t stream = nullptr;
    void *links = nullptr;       // C<R>[4][3 nr][Vl]
    void *uhalo = nullptr;       // C<R>[3 nr][S3]   U_t of the slice below the slab
    void *W = nullptr;           // C<R>[4][Vl]      packed Delta / w, t-slab order
    void *Wt = nullptr;          // C<R>[4][Vl]      the same field in z-slab order
    void *G = nullptr;           // C<R>[6][Vl]
    void *ghalo = nullptr;       // C<R>[6][S3]      g of the slice above the slab
    double *partial = nullptr;
    int nb = 0;
    DevState *st = nullptr;      // all zero: the kernels shared with the one-GPU path look at st->done
    void *twiddle[4] = {nullptr, nullptr, nullptr, nullptr};
    void *p2tab = nullptr;       // R[4][64], z section shifted to this rank's z-slab
    AxisPass pass_fwd[3], pass_inv[3], pass_t;
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
        for (int i = 0; i < count; i++) {
            const int p = first + i, k = (p / N2) + N1 * (p % N2);
            double c, s;
            host_cossin_2pi(k, 2 * L, c, s);
            p2[mu * 64 + i] = (R)(4.0 * s * s);
        }
    }
    SCK(cudaMalloc(&ctx->p2tab, sizeof(R) * 4 * 64));
    SCK(cudaMemcpy(ctx->p2tab, p2.data(), sizeof(R) * 4 * 64, cudaMemcpyHostToDevice));
    return LGF_OK;
}

template <class R>
static int slab_fft_local(lgf_slab *ctx, int inverse) {
    const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2], (const R *)ctx->twiddle[3]};
    for (int i = 0; i < 3; i++) {
        const AxisPass &p = inverse ? ctx->pass_inv[i] : ctx->pass_fwd[i];
        SCK(launch_fft_pass<R>(p, (C<R> *)ctx->W, ctx->gl, tw, (const R *)ctx->p2tab, (R)0, ctx->st, ctx->stream));
        ctx->launches++;
    }
    return LGF_OK;
}

template <class R>
static int slab_fft_t(lgf_slab *ctx) {
    const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2], (const R *)ctx->twiddle[3]};
    const R scale = (R)(16.0 / (double)ctx->Vglobal);              // p2max / V (Alg. 1 lines 5, 7; R5)
    SCK(launch_fft_pass<R>(ctx->pass_t, (C<R> *)ctx->Wt, ctx->gt, tw, (const R *)ctx->p2tab, scale, ctx->st, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

template <class R>
static int slab_delta(lgf_slab *ctx, double *d_sums) {
    if (ctx->nr == 3)
        k_slab_delta<R, 3><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>((const C<R> *)ctx->links, (const C<R> *)ctx->uhalo,
                                                                      (C<R> *)ctx->W, ctx->gl, ctx->partial);
    else
        k_slab_delta<R, 2><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>((const C<R> *)ctx->links, (const C<R> *)ctx->uhalo,
                                                                      (C<R> *)ctx->W, ctx->gl, ctx->partial);
    SCK(cudaGetLastError());
    k_slab_sum2<<<1, SLAB_THREADS, 0, ctx->stream>>>(ctx->partial, ctx->nb, d_sums);
    SCK(cudaGetLastError());
    ctx->launches += 2;
    return LGF_OK;
}

template <class R>
static int slab_update(lgf_slab *ctx) {
    if (ctx->nr == 3)
        k_slab_update<R, 3><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>((C<R> *)ctx->links, (const C<R> *)ctx->G,
                                                                       (const C<R> *)ctx->ghalo, ctx->gl);
    else
        k_slab_update<R, 2><<<ctx->nb, SLAB_THREADS, 0, ctx->stream>>>((C<R> *)ctx->links, (const C<R> *)ctx->G,
                                                                       (const C<R> *)ctx->ghalo, ctx->gl);
    SCK(cudaGetLastError());
    ctx->launches++;
    return LGF_OK;
}

template <class R>
static int slab_transpose(lgf_slab *ctx, int stage, void *d_buf) {
    // stage 0: W (t-slabs) -> send buffer;  1: receive buffer -> Wt (z-slabs);  2: Wt -> send buffer;  3: receive buffer -> W
    const int side = (stage == 0 || stage == 3) ? 0 : 1, dir = (stage == 0 || stage == 2) ? 0 : 1;
    C<R> *field = (C<R> *)(side == 0 ? ctx->W : ctx->Wt);
    const long long n = 4 * ctx->gl.V;
    k_slab_transpose<R><<<(unsigned)((n + SLAB_THREADS - 1) / SLAB_THREADS), SLAB_THREADS, 0, ctx->stream>>>(
        field, (C<R> *)d_buf, ctx->gl.V, (int)ctx->gl.S[2], ctx->T, ctx->Zl, ctx->N, side, dir);
    SCK(cudaGetLastError());
    ctx->launches++;
    return LGF_OK;
}

extern "C" {

const char *lgf_slab_last_error(const lgf_slab *ctx) { return ctx ? ctx->err.c_str() : g_slab_err.c_str(); }

int lgf_slab_destroy(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    cudaStreamSynchronize(ctx->stream);
    void *bufs[] = {ctx->links, ctx->uhalo, ctx->W, ctx->Wt, ctx->G, ctx->ghalo, ctx->partial, ctx->st, ctx->p2tab,
                    ctx->twiddle[0], ctx->twiddle[1], ctx->twiddle[2], ctx->twiddle[3]};
    for (void *b : bufs) cudaFree(b);
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
    ctx->prec = precision;
    ctx->nr = link_storage == LGF_LINKS_18 ? 3 : 2;
    ctx->rank = rank;
    ctx->N = nranks;
    ctx->T = dims[3] / nranks;
    ctx->Zl = dims[2] / nranks;
    ctx->Vglobal = 1;
    for (int mu = 0; mu < 4; mu++) { ctx->dims[mu] = dims[mu]; ctx->Vglobal *= dims[mu]; }
    const int Ll[4] = {dims[0], dims[1], dims[2], ctx->T}, Lt[4] = {dims[0], dims[1], ctx->Zl, dims[3]};
    long long Sl = 1, St = 1;
    for (int mu = 0; mu < 4; mu++) {
        ctx->gl.L[mu] = Ll[mu]; ctx->gl.S[mu] = Sl; Sl *= Ll[mu];
        ctx->gt.L[mu] = Lt[mu]; ctx->gt.S[mu] = St; St *= Lt[mu];
    }
    ctx->gl.V = Sl;
    ctx->gt.V = St;
    const size_t V = (size_t)Sl, S3 = (size_t)ctx->gl.S[3], cb = 2 * (size_t)precision;
    ctx->nb = (int)((V + SLAB_THREADS - 1) / SLAB_THREADS);
    int rc = LGF_OK;
    auto alloc = [&](void **p, size_t bytes) {
        if (rc != LGF_OK) return;
        cudaError_t ee = cudaMalloc(p, bytes);
        if (ee != cudaSuccess) rc = sfail(ctx, ee == cudaErrorMemoryAllocation ? LGF_ENOMEM : LGF_ECUDA,
                                          std::string("cudaMalloc: ") + cudaGetErrorString(ee));
    };
    alloc(&ctx->links, V * 4 * 3 * ctx->nr * cb);
    alloc(&ctx->uhalo, S3 * 3 * ctx->nr * cb);
    alloc(&ctx->W, V * 4 * cb);
    alloc(&ctx->Wt, V * 4 * cb);
    alloc(&ctx->G, V * 6 * cb);
    alloc(&ctx->ghalo, S3 * 6 * cb);
    alloc((void **)&ctx->partial, sizeof(double) * 2 * ctx->nb);
    alloc((void **)&ctx->st, sizeof(DevState));
    if (rc == LGF_OK) {
        cudaError_t ee = cudaMemset(ctx->st, 0, sizeof(DevState));
        if (ee != cudaSuccess) rc = sfail(ctx, LGF_ECUDA, std::string("cudaMemset: ") + cudaGetErrorString(ee));
    }
    if (rc == LGF_OK) rc = precision == LGF_FP64 ? slab_tables<double>(ctx) : slab_tables<float>(ctx);
    if (rc != LGF_OK) {
        g_slab_err = ctx->err;
        lgf_slab_destroy(ctx);
        return rc;
    }
    for (int a = 0; a < 3; a++) {
        ctx->pass_fwd[a] = slab_axis_pass(ctx->gl, precision, a, FFT_FWD);
        ctx->pass_inv[a] = slab_axis_pass(ctx->gl, precision, 2 - a, FFT_INV);
    }
    ctx->pass_t = slab_axis_pass(ctx->gt, precision, 3, FFT_FWD_SCALE_INV);
    *out = ctx;
    return LGF_OK;
}

int lgf_slab_set_stream(lgf_slab *ctx, void *cuda_stream) {
    if (!ctx) return LGF_EINVAL;
    ctx->stream = (cudaStream_t)cuda_stream;
    return LGF_OK;
}

int lgf_slab_set_links(lgf_slab *ctx, const void *d_links) {
    if (!ctx || !d_links) return sfail(ctx, LGF_EINVAL, "lgf_slab_set_links: null argument");
    if (ctx->prec == LGF_FP64) SCK(launch_convert_in<double>(ctx->nr, (const double *)d_links, (C<double> *)ctx->links, ctx->gl, ctx->stream));
    else SCK(launch_convert_in<float>(ctx->nr, (const float *)d_links, (C<float> *)ctx->links, ctx->gl, ctx->stream));
    ctx->launches++;
    ctx->have_links = true;
    return LGF_OK;
}

int lgf_slab_get_links(lgf_slab *ctx, void *d_links) {
    if (!ctx || !d_links) return sfail(ctx, LGF_EINVAL, "lgf_slab_get_links: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_get_links: no configuration loaded");
    if (ctx->prec == LGF_FP64) {
        LinkPair<double> lp{{(C<double> *)ctx->links, (C<double> *)ctx->links}};
        SCK(launch_convert_out<double>(ctx->nr, lp, (double *)d_links, ctx->gl, ctx->st, ctx->stream));
    } else {
        LinkPair<float> lp{{(C<float> *)ctx->links, (C<float> *)ctx->links}};
        SCK(launch_convert_out<float>(ctx->nr, lp, (float *)d_links, ctx->gl, ctx->st, ctx->stream));
    }
    ctx->launches++;
    return LGF_OK;
}

long long lgf_slab_halo_elems(const lgf_slab *ctx, int which) {
    if (!ctx || (which != LGF_HALO_LINKS && which != LGF_HALO_G)) return LGF_EINVAL;
    return (long long)ctx->gl.S[3] * (which == LGF_HALO_LINKS ? 3 * ctx->nr : 6) * 2;
}

int lgf_slab_halo_pack(lgf_slab *ctx, int which, void *d_send) {
    if (!ctx || !d_send) return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_pack: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_halo_pack: no configuration loaded");
    const size_t cb = 2 * (size_t)ctx->prec, S3 = (size_t)ctx->gl.S[3], V = (size_t)ctx->gl.V;
    if (which == LGF_HALO_LINKS) {          // U_t of the LAST local slice, for the rank above
        const char *src = (const char *)ctx->links + ((size_t)3 * 3 * ctx->nr * V + S3 * (ctx->T - 1)) * cb;
        SCK(cudaMemcpy2DAsync(d_send, S3 * cb, src, V * cb, S3 * cb, 3 * ctx->nr, cudaMemcpyDeviceToDevice, ctx->stream));
    } else if (which == LGF_HALO_G) {       // g of the FIRST local slice, for the rank below
        SCK(cudaMemcpy2DAsync(d_send, S3 * cb, ctx->G, V * cb, S3 * cb, 6, cudaMemcpyDeviceToDevice, ctx->stream));
    } else return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_pack: bad halo id");
    return LGF_OK;
}

int lgf_slab_halo_unpack(lgf_slab *ctx, int which, const void *d_recv) {
    if (!ctx || !d_recv) return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_unpack: null argument");
    const size_t cb = 2 * (size_t)ctx->prec, S3 = (size_t)ctx->gl.S[3];
    if (which == LGF_HALO_LINKS) SCK(cudaMemcpyAsync(ctx->uhalo, d_recv, S3 * 3 * ctx->nr * cb, cudaMemcpyDeviceToDevice, ctx->stream));
    else if (which == LGF_HALO_G) SCK(cudaMemcpyAsync(ctx->ghalo, d_recv, S3 * 6 * cb, cudaMemcpyDeviceToDevice, ctx->stream));
    else return sfail(ctx, LGF_EINVAL, "lgf_slab_halo_unpack: bad halo id");
    return LGF_OK;
}

int lgf_slab_delta(lgf_slab *ctx, double *d_sums) {
    if (!ctx || !d_sums) return sfail(ctx, LGF_EINVAL, "lgf_slab_delta: null argument");
    if (!ctx->have_links) return sfail(ctx, LGF_ESTATE, "lgf_slab_delta: no configuration loaded");
    return ctx->prec == LGF_FP64 ? slab_delta<double>(ctx, d_sums) : slab_delta<float>(ctx, d_sums);
}

int lgf_slab_fft_local(lgf_slab *ctx, int inverse) {
    if (!ctx) return LGF_EINVAL;
    return ctx->prec == LGF_FP64 ? slab_fft_local<double>(ctx, inverse) : slab_fft_local<float>(ctx, inverse);
}

int lgf_slab_transpose(lgf_slab *ctx, int stage, void *d_buf) {
    if (!ctx || !d_buf || stage < 0 || stage > 3) return sfail(ctx, LGF_EINVAL, "lgf_slab_transpose: bad argument");
    return ctx->prec == LGF_FP64 ? slab_transpose<double>(ctx, stage, d_buf) : slab_transpose<float>(ctx, stage, d_buf);
}

int lgf_slab_fft_t(lgf_slab *ctx) {
    if (!ctx) return LGF_EINVAL;
    return ctx->prec == LGF_FP64 ? slab_fft_t<double>(ctx) : slab_fft_t<float>(ctx);
}

int lgf_slab_gbuild(lgf_slab *ctx, double alpha) {
    if (!ctx) return LGF_EINVAL;
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
    return ctx->prec == LGF_FP64 ? slab_update<double>(ctx) : slab_update<float>(ctx);
}

int lgf_slab_get_field(lgf_slab *ctx, void *d_field) {
    if (!ctx || !d_field) return sfail(ctx, LGF_EINVAL, "lgf_slab_get_field: null argument");
    if (ctx->prec == LGF_FP64) SCK(launch_field_get<double>((const C<double> *)ctx->W, (double *)d_field, ctx->gl, ctx->stream));
    else SCK(launch_field_get<float>((const C<float> *)ctx->W, (float *)d_field, ctx->gl, ctx->stream));
    ctx->launches++;
    return LGF_OK;
}

long long lgf_slab_launch_count(const lgf_slab *ctx) { return ctx ? ctx->launches : LGF_EINVAL; }

}  // extern "C"
