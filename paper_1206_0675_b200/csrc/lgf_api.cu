// lgf_api.cu -- the C ABI of liblgf (include/lgf.h): context, device buffers, tables, the FFT pass
// plan and the Algorithm-1 driver.  Part of the CUDA path; shares nothing with
// oracle/.  There is no CPU fallback anywhere in this file: without a CUDA device lgf_create fails.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/lgf.h"
#include "lgf_state.cuh"

using namespace lgf;

struct lgf_ctx {
    Geom g{};
    int device = 0;      // the CUDA device the context's buffers live on; every entry point makes it current
    int prec = 0;        // bytes per real
    int nr = 3;          // stored rows per link
    cudaStream_t stream = nullptr;
    void *links[2] = {nullptr, nullptr};   // C<R>[4][3*nr][V] each: the sweep reads one and writes the other
    void *W = nullptr;           // C<R>[4][V]   packed Delta / w
    void *G = nullptr;           // C<R>[6][V]   rows 0, 1 of g(x)
    void *Gacc = nullptr;        // C<R>[9][V]   accumulated transformation g_n ... g_1 (lgf_track_transform), or null
    bool w_is_delta = false;     // W holds Delta of the current configuration and `partial` its F / theta sums
    bool recorded = false;       // the current configuration's (F, theta) is already in the history
    int nb_partial = 0;          // number of per-block partial sums currently in `partial`
    double *partial = nullptr;   // per-block partial sums
    int partial_cap = 0;
    DevState *st = nullptr;
    DevState *h_st = nullptr;    // pinned mirror
    DevState *h_poll = nullptr;  // pinned: two slots for the pipelined look at the stop flag in lgf_fix
    cudaEvent_t poll_ev[2] = {nullptr, nullptr};
    double *hist = nullptr;      // (F, theta) pairs
    long long hist_cap = 0;
    double *d_scalar = nullptr;
    void *twiddle[4] = {nullptr, nullptr, nullptr, nullptr};   // C<R>[64] per axis, exp(-2 pi i m / L_mu)
    void *p2tab = nullptr;                                     // R[4][64]
    SweepMaps *sweep_maps = nullptr;   // TMA tensor maps of the staged sweep (lgf_sweep_tma.cu); null = k_sweep only
    // the *_host entry points: two chunk buffers in canonical layout, a copy stream and events, so that the PCIe copy of
    // chunk k + 1 overlaps the layout conversion of chunk k (no configuration-sized staging buffer)
    void *stage[2] = {nullptr, nullptr};
    long long stage_sites = 0;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_full[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr}, ev_start = nullptr;
    std::vector<AxisPass> passes;
    unsigned long long hb_sweeps = 0;   // heat-bath sweeps applied since the last set_links (selects the random stream)
    bool have_links = false;
    bool profiling = false;
    int tune_two_axis = 1;       // lgf_tune: use the two-axis FFT passes when available
    int tune_reg = 1;            // lgf_tune: use the register-line FFT sweeps when available
    int tune_reg2 = 1;           // lgf_tune: two-threads-per-line FFT sweeps where the lattice allows (0 = never)
    int tune_xy_planes = 0;      // lgf_tune: planes per CTA of the (x, y) pass (0 = planner's choice)
    int tune_zt_xc = 0;          // lgf_tune: consecutive (x, y) indices per CTA of the (z, t) pass
    int tune_fuse_g = 1;         // lgf_tune: end the last FFT sweep with the g-build (register-line plan only)
    int tune_sweep_share = -1;   // lgf_tune: hand A'_x, A'_y to the forward neighbours of the same CTA through shared
                                 // memory (1 / 0; -1 = automatic: 18-real and fp32 or a lattice beyond L2)
    int tune_hb_tz = 0;          // lgf_tune: z-planes per (z, t) tile of the heat-bath thread order (0 = automatic)
    int tune_reunit = 0;         // lgf_tune "reunit_every": project the new links onto SU(3) in every N-th update (0 = never)
    long long updates_enqueued = 0;   // host-side count of updates enqueued since the last set_links / thermalize
    int tune_pdl = 1;            // lgf_tune "pdl": launch the iteration's kernels with programmatic stream serialization
    int tune_fft_zt_cluster = -1; // lgf_tune "fft_zt_cluster": (z, t) tile split over a cluster of 2 / 4 CTAs; 0 = off; -1 = where it measured
    int tune_fft_bulk = -1;      // lgf_tune "fft_bulk": (x, y) FFT sweeps fed by cp.async.bulk: 1 / 0 / -1 = where it measured
                                 // faster (64-point fp64 planes: 64^4 FFT 1.98 -> 1.81 ms; neutral at 32^4 and 16^4)
    int tune_sweep_tma = -1;     // lgf_tune "sweep_tma" (see use_sweep_tma)
    int tune_sweep_rsplit = 1;   // lgf_tune "sweep_rsplit": register split between producer and compute warps (fp64 staged sweep)
    int tune_sweep_ahead = 0;    // lgf_tune "sweep_prefetch": CTAs ahead of which the sweep prefetches its tile into L2 (0 = off)
    int tune_sweep_minb = 0;     // lgf_tune "sweep_minb": resident CTAs per SM the sweep's register allocation allows (0 = automatic, 2, 3, 4, 5)
    int tune_sweep_tz = 0;       // lgf_tune: z-planes per (z, t) tile of the sweep's block order (0 = automatic, 1 = plain)
    struct Stamp { cudaEvent_t a, b; int cls; };
    std::vector<Stamp> stamps;
    double prof_ms[LGF_K_COUNT] = {0};
    long long prof_n[LGF_K_COUNT] = {0};
    long long launches = 0;
    std::string err;
};

static thread_local std::string g_err;   // errors with no context (lgf_create failures)

static int fail(lgf_ctx *ctx, int code, const std::string &msg) {
    if (ctx) ctx->err = msg;
    g_err = msg;
    return code;
}
static int cuda_fail(lgf_ctx *ctx, cudaError_t e, const char *what) {
    return fail(ctx, e == cudaErrorMemoryAllocation ? LGF_ENOMEM : LGF_ECUDA,
                std::string(what) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);     \
    } while (0)

// every entry point runs on the device the context was created on (the caller may have another one current)
#define ENTER(ctx)                                                                                    \
    do {                                                                                              \
        cudaError_t e_ = cudaSetDevice((ctx)->device);                                                \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, "cudaSetDevice");                            \
    } while (0)

// the context's stream with its dependent-launch setting, for the launchers
#define STRM(ctx) (lgf::LaunchStream((ctx)->stream, (ctx)->tune_pdl != 0))

// ---- host-side tables -----------------------------------------------------------------------------
static bool valid_len(int L) {
    static const int ok[] = {2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64};
    for (int v : ok) if (v == L) return true;
    return false;
}
static void line_factor(int L, int &N1, int &N2) {     // must agree with lgf::LineFactor<L>
    N1 = (L <= 8) ? L : ((L % 8 == 0) ? 8 : ((L % 4 == 0) ? 4 : ((L % 6 == 0) ? 6 : 3)));
    N2 = L / N1;
}
// cos and sin of 2 pi m / L by exact octant reduction of the fraction, then libm in long double
static void cossin_2pi(int m, int L, double &c, double &s) {
    long num = 8L * (m % L), den = 8L * L;
    double sc = 1.0, ss = 1.0;
    bool swap = false;
    if (2 * num > den) { num = den - num; ss = -ss; }
    if (4 * num > den) { num = den / 2 - num; sc = -sc; }
    if (8 * num > den) { num = den / 4 - num; swap = true; }
    const long double x = 2.0L * 3.14159265358979323846264338327950288L * (long double)num / (long double)den;
    long double cc = cosl(x), sv = sinl(x);
    if (8 * num == den) { cc = 0.70710678118654752440084436210484904L; sv = cc; }
    if (num == 0) { cc = 1.0L; sv = 0.0L; }
    if (swap) { const long double t = cc; cc = sv; sv = t; }
    c = sc * (double)cc;
    s = ss * (double)sv;
}

// the same tables for the slab-decomposed path (lgf_slab.cu)
namespace lgf {
bool host_valid_len(int L) { return valid_len(L); }
void host_line_factor(int L, int &N1, int &N2) { line_factor(L, N1, N2); }
void host_cossin_2pi(int m, int L, double &c, double &s) { cossin_2pi(m, L, c, s); }
}

template <class R>
static int upload_twiddles(lgf_ctx *ctx) {
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->g.L[mu];
        std::vector<R> tw(2 * 64, (R)0);
        for (int m = 0; m < L; m++) {
            double c, s;
            cossin_2pi(m, L, c, s);
            tw[2 * m] = (R)c;
            tw[2 * m + 1] = (R)(-s);                      // forward sign e^{-i}
        }
        CK(cudaMalloc(&ctx->twiddle[mu], sizeof(R) * 2 * 64));
        CK(cudaMemcpy(ctx->twiddle[mu], tw.data(), sizeof(R) * 2 * 64, cudaMemcpyHostToDevice));
    }
    CK(cudaMalloc(&ctx->p2tab, sizeof(R) * 4 * 64));
    return LGF_OK;
}
// p2tab[mu*64 + p] = 4 sin^2(pi k_mu(p) / L_mu), p = position along axis mu in k space: natural order
// (k = p) for axes transformed in registers, the permuted order of the in-place two-step transform
// (lgf_fft.cu header) otherwise.
template <class R>
static int upload_p2(lgf_ctx *ctx, const bool natural[4]) {
    std::vector<R> p2(4 * 64, (R)0);
    for (int mu = 0; mu < 4; mu++) {
        const int L = ctx->g.L[mu];
        int N1, N2;
        line_factor(L, N1, N2);
        for (int p = 0; p < L; p++) {
            const int k = natural[mu] ? p : (p / N2) + N1 * (p % N2);
            // 4 sin^2(pi k / L): sine of the half angle, pi k / L = 2 pi k / (2L)
            double c, s;
            cossin_2pi(k, 2 * L, c, s);
            p2[mu * 64 + p] = (R)(4.0 * s * s);
        }
    }
    CK(cudaMemcpyAsync(ctx->p2tab, p2.data(), sizeof(R) * 4 * 64, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return LGF_OK;
}

static long long largest_divisor_le(long long n, long long cap) {
    if (cap < 1) cap = 1;
    for (long long d = (cap < n ? cap : n); d >= 1; d--)
        if (n % d == 0) return d;
    return 1;
}

static long long pow2_divisor_le(long long n, long long cap) {
    long long d = 1;
    while (d * 2 <= cap && n % (d * 2) == 0) d *= 2;
    return d;
}

// FFT pass plan.  Preferred: three sweeps of the field -- (x, y) planes forward, (z, t) planes forward +
// scale + inverse, (x, y) planes inverse -- when two-axis kernels exist for the lattice's lengths and
// the tiles fit in shared memory; otherwise one pass per axis (forward x, y, z; forward + scale +
// inverse on t; inverse z, y, x).  tune_xy_planes / tune_zt_xc (> 0) override the tile sizes.
// one in-place shared-memory pass over one axis (k_fft_axis; any supported length)
static AxisPass make_axis_pass(const lgf_ctx *ctx, int axis, int mode) {
    const long long T = 2048;     // target complex elements per tile
    const size_t cbytes = 2 * (size_t)ctx->prec;
    const Geom &g = ctx->g;
    AxisPass p{};
    p.kind = PASS_AXIS;
    p.axis = axis;
    p.L = g.L[axis];
    p.mode = mode;
    p.S = g.S[axis];
    p.H = g.V / (p.S * p.L);
    if (p.S == 1) {
        p.nlo = 1;
        p.nhi = (int)largest_divisor_le(p.H, T / p.L);
        p.smem = (64 + (size_t)p.nhi * (p.L | 1)) * cbytes;
    } else {
        p.nlo = (int)largest_divisor_le(p.S, T / p.L);
        p.nhi = (int)largest_divisor_le(p.H, T / ((long long)p.L * p.nlo));
        p.smem = (64 + (size_t)p.nhi * p.L * p.nlo) * cbytes;
    }
    p.threads = 256;
    return p;
}

static int plan_passes(lgf_ctx *ctx) {
    const size_t cbytes = 2 * (size_t)ctx->prec;
    const Geom &g = ctx->g;
    auto make = [&](int axis, int mode) { return make_axis_pass(ctx, axis, mode); };
    auto finish = [&](const bool natural[4]) {
        return ctx->prec == LGF_FP64 ? upload_p2<double>(ctx, natural) : upload_p2<float>(ctx, natural);
    };
    ctx->passes.clear();
    auto plan_reg2 = [&]() {
        for (int w = 0; w < 3; w++) {
            AxisPass p{};
            p.kind = PASS_REG2;
            p.axis = w;
            ctx->passes.push_back(p);
        }
        const bool natural[4] = {true, true, true, true};
        return finish(natural);
    };
    // Two threads per line wherever those kernels exist (16-, 32-, 64-point axes).  Measured on B200 against
    // the one-thread family at 32^4 (warm, CUDA events): fp64 iteration 0.3886 -> 0.3854 ms, fp32 0.2402 ->
    // 0.2335 ms; at 64^4 (against the shared-memory passes) fp64 7.60 -> 6.72 ms, fp32 4.48 -> 3.78 ms.  A
    // per-sweep mix of the two families was tried and is not better (0.3908 ms).
    if (ctx->tune_two_axis && ctx->tune_reg2 != 0 && fft_reg2_supported(g)) return plan_reg2();
    if (ctx->tune_two_axis && ctx->tune_reg && fft_reg_supported(g)) {
        for (int w = 0; w < 3; w++) {
            AxisPass p{};
            p.kind = PASS_REG;
            p.axis = w;
            ctx->passes.push_back(p);
        }
        const bool natural[4] = {true, true, true, fft_reg_t_natural(g)};
        return finish(natural);
    }
    const bool permuted[4] = {false, false, false, false};
    const size_t SMEM_MAX = 200 * 1024;
    const long long MIN_GRID = 2 * 148;
    // (x, y) planes
    AxisPass xy{};
    bool have_xy = ctx->tune_two_axis && fft_pair_supported(PASS_XY, g.L[0], g.L[1]);
    if (have_xy) {
        const long long planes = 4LL * g.L[2] * g.L[3], psize = (long long)g.L[0] * g.L[1];
        long long P = largest_divisor_le(planes, 2048 / psize > 0 ? 2048 / psize : 1);
        while (P > 1 && planes / P < MIN_GRID) P = largest_divisor_le(planes, P - 1);
        if (ctx->tune_xy_planes > 0 && planes % ctx->tune_xy_planes == 0) P = ctx->tune_xy_planes;
        xy.kind = PASS_XY; xy.L = g.L[0]; xy.L2 = g.L[1]; xy.nhi = (int)P; xy.nlo = 1; xy.threads = 256;
        xy.smem = (128 + (size_t)P * g.L[1] * (g.L[0] | 1)) * cbytes;
        have_xy = xy.smem <= SMEM_MAX;
    }
    // (z, t) planes
    AxisPass zt{};
    bool have_zt = ctx->tune_two_axis && fft_pair_supported(PASS_ZT, g.L[2], g.L[3]);
    if (have_zt) {
        const long long plane = g.S[2], zsize = (long long)g.L[2] * g.L[3];
        const long long phase = 128 / (long long)cbytes;             // lanes per shared-memory phase
        // shortest run the planner accepts: 2 complex elements (32 B in fp64, 16 B in fp32).  Measured at 64^4
        // on B200: fp64 XC = 2 (128 KB tile) beats XC = 1 (2.87 vs 2.97 ms per FFT), fp32 XC = 2 (64 KB tile,
        // 3 CTAs per SM) beats the 32-byte rule's XC = 4 (1.62 vs 1.92 ms).
        const long long xc_min = pow2_divisor_le(plane, 2);
        long long XC = pow2_divisor_le(plane, (65536 / (long long)cbytes) / zsize > 0 ? (65536 / (long long)cbytes) / zsize : 1);
        while (XC > xc_min && (plane / XC) * 4 < MIN_GRID) XC /= 2;
        if (XC < xc_min) XC = xc_min;
        if (ctx->tune_zt_xc > 0 && plane % ctx->tune_zt_xc == 0) XC = ctx->tune_zt_xc;
        long long pitch = XC * g.L[2];
        if (XC < phase && pitch % phase == 0) pitch += XC;           // lanes (xc, t) -> distinct banks
        zt.kind = PASS_ZT; zt.L = g.L[2]; zt.L2 = g.L[3]; zt.mode = FFT_FWD_SCALE_INV; zt.nlo = (int)XC; zt.nhi = 1;
        zt.pitch = (int)pitch; zt.threads = 256;
        zt.smem = (128 + (size_t)pitch * g.L[3]) * cbytes;
        have_zt = zt.smem <= SMEM_MAX;
    }
    if (have_xy) { xy.mode = FFT_FWD; ctx->passes.push_back(xy); }
    else { ctx->passes.push_back(make(0, FFT_FWD)); ctx->passes.push_back(make(1, FFT_FWD)); }
    if (have_zt) ctx->passes.push_back(zt);
    else {
        ctx->passes.push_back(make(2, FFT_FWD));
        ctx->passes.push_back(make(3, FFT_FWD_SCALE_INV));
        ctx->passes.push_back(make(2, FFT_INV));
    }
    if (have_xy) { xy.mode = FFT_INV; ctx->passes.push_back(xy); }
    else { ctx->passes.push_back(make(1, FFT_INV)); ctx->passes.push_back(make(0, FFT_INV)); }
    return finish(permuted);
}

// ---- profiling brackets ---------------------------------------------------------------------------
struct Bracket {
    lgf_ctx *ctx;
    int cls;
    cudaEvent_t a = nullptr, b = nullptr;
    Bracket(lgf_ctx *c, int k) : ctx(c), cls(k) {
        ctx->launches++;
        if (ctx->profiling) {
            cudaEventCreate(&a);
            cudaEventCreate(&b);
            cudaEventRecord(a, ctx->stream);
        }
    }
    ~Bracket() {
        if (a) {
            cudaEventRecord(b, ctx->stream);
            ctx->stamps.push_back({a, b, cls});
        }
    }
};
static void drain_stamps(lgf_ctx *ctx) {
    for (auto &s : ctx->stamps) {
        float ms = 0.f;
        if (cudaEventSynchronize(s.b) == cudaSuccess && cudaEventElapsedTime(&ms, s.a, s.b) == cudaSuccess) {
            ctx->prof_ms[s.cls] += ms;
            ctx->prof_n[s.cls] += 1;
        }
        cudaEventDestroy(s.a);
        cudaEventDestroy(s.b);
    }
    ctx->stamps.clear();
}

// ---- typed steps ----------------------------------------------------------------------------------
template <class R>
static LinkPair<R> link_pair(lgf_ctx *ctx) {
    LinkPair<R> lp;
    lp.buf[0] = (C<R> *)ctx->links[0];
    lp.buf[1] = (C<R> *)ctx->links[1];
    return lp;
}
template <class R>
static int step_delta(lgf_ctx *ctx, const int *stop) {
    Bracket br(ctx, LGF_K_DELTA);
    CK(launch_delta<R>(ctx->nr, link_pair<R>(ctx), (C<R> *)ctx->W, ctx->g, ctx->partial, &ctx->nb_partial, stop, ctx->st,
                       STRM(ctx)));
    return LGF_OK;
}
static bool use_fft_bulk(const lgf_ctx *ctx) {
    return ctx->tune_fft_bulk > 0 || (ctx->tune_fft_bulk < 0 && ctx->g.L[0] == 64);
}
static int use_zt_cluster(const lgf_ctx *ctx) {
    const int nc = ctx->tune_fft_zt_cluster;
    if (nc > 0) return fft_reg2_zt_cluster_supported(ctx->g, nc) ? nc : 0;
    return 0;                                                // automatic = off: it measured slower
}
// true if the plan's last sweep can end with the g-build (a5) and write G instead of W
static bool can_fuse_g(const lgf_ctx *ctx) {
    if (!ctx->tune_fuse_g || ctx->passes.empty()) return false;
    const int kind = ctx->passes.back().kind;
    return kind == PASS_REG || (kind == PASS_REG2 && fft_reg2_gout(ctx->g, ctx->prec));
}
// a2-a4.  with_g: the last sweep also does a5 with step alpha (W is then NOT left holding w).
template <class R>
static int step_accelerate(lgf_ctx *ctx, bool with_g = false, double alpha = 0.0) {
    const R scale = (R)(16.0 / (double)ctx->g.V);        // p2max / V      (Alg. 1 lines 5, 7; R5, R7)
    for (const AxisPass &p : ctx->passes) {
        Bracket br(ctx, LGF_K_FFT);
        if (p.kind == PASS_REG) {
            const int which = (with_g && p.axis == 2) ? 3 : p.axis;
            CK(launch_fft_reg<R>(which, ctx->g, (C<R> *)ctx->W, (const R *)ctx->twiddle[3], (const R *)ctx->p2tab, scale,
                                 ctx->st, STRM(ctx), (C<R> *)ctx->G, (R)(0.5 * alpha)));
            continue;
        }
        if (p.kind == PASS_REG2) {
            const int which = (with_g && p.axis == 2) ? 3 : p.axis;
            CK(launch_fft_reg2<R>(which, ctx->g, (C<R> *)ctx->W, (const R *)ctx->p2tab, scale, ctx->st, STRM(ctx),
                                  (C<R> *)ctx->G, (R)(0.5 * alpha), use_fft_bulk(ctx), -1, use_zt_cluster(ctx)));
            continue;
        }
        const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2],
                          (const R *)ctx->twiddle[3]};
        CK(launch_fft_pass<R>(p, (C<R> *)ctx->W, ctx->g, tw, (const R *)ctx->p2tab, scale, ctx->st, STRM(ctx)));
    }
    return LGF_OK;
}
// the staged (TMA) sweep or the register sweep?  "sweep_tma": 1 = wherever it applies, 0 = never, -1 = where it
// measured faster than k_sweep on B200 (sweep_tma_auto, lgf_sweep_tma.cu, has the numbers)
static bool use_sweep_tma(const lgf_ctx *ctx) {
    return ctx->sweep_maps && (ctx->tune_sweep_tma > 0 || (ctx->tune_sweep_tma < 0 && sweep_tma_auto(ctx->g, ctx->nr, ctx->prec)));
}
// a5 then a6 + a1: g from the current W, then the fused sweep (new links into the other buffer, Delta of
// the new links into W, partial sums of F and theta)
static int step_finalize(lgf_ctx *ctx, double tol, int after_sweep, int record) {
    ctx->launches++;
    CK(launch_finalize(ctx->partial, ctx->nb_partial, ctx->g.V, tol, after_sweep, record, ctx->st, ctx->hist,
                       ctx->hist_cap, STRM(ctx)));
    return LGF_OK;
}
// The sweep also closes the iteration: it makes the new configuration current, and with record != 0 appends
// (F, theta) to the history and applies the loop test theta < tol (the k_finalize launch after the sweep).
template <class R>
static int step_update(lgf_ctx *ctx, double alpha, double tol, int record, bool g_ready = false) {
    if (!g_ready) {
        Bracket br(ctx, LGF_K_GBUILD);
        CK(launch_gbuild<R>((const C<R> *)ctx->W, (C<R> *)ctx->G, ctx->g, (R)(0.5 * alpha), ctx->st, STRM(ctx)));
    }
    if (ctx->Gacc) {                                      // Gacc <- g Gacc, with the g this update applies
        Bracket br(ctx, LGF_K_GBUILD);
        CK(launch_gacc<R>(1, (const C<R> *)ctx->G, (C<R> *)ctx->Gacc, (R *)nullptr, ctx->g, ctx->st, STRM(ctx)));
    }
    ctx->updates_enqueued++;
    const bool reunit = ctx->tune_reunit > 0 && ctx->updates_enqueued % ctx->tune_reunit == 0;
    if (use_sweep_tma(ctx)) {
        Bracket br(ctx, LGF_K_UPDATE);
        CK(launch_sweep_tma<R>(ctx->sweep_maps, ctx->nr, link_pair<R>(ctx), (const C<R> *)ctx->G, (C<R> *)ctx->W, ctx->g, ctx->partial,
                               &ctx->nb_partial, ctx->st, STRM(ctx), ctx->tune_sweep_tz, reunit, SweepHalo<R>(),
                               ctx->tune_sweep_rsplit != 0));
    } else {
        Bracket br(ctx, LGF_K_UPDATE);
        CK(launch_sweep<R>(ctx->nr, link_pair<R>(ctx), (const C<R> *)ctx->G, (C<R> *)ctx->W, ctx->g, ctx->partial,
                           &ctx->nb_partial, ctx->st, STRM(ctx), ctx->tune_sweep_tz, reunit, ctx->tune_sweep_share,
                           ctx->tune_sweep_ahead, ctx->tune_sweep_minb));
    }
    return step_finalize(ctx, tol, 1, record);
}

// Alg. 1 line 1: Delta, F, theta of the loaded configuration, recorded as history entry 0 with the stop
// test of line 2.  Skipped when W already holds Delta of the current configuration (left there by the
// previous sweep, whose finalize has recorded it).
template <class R>
static int first_measure(lgf_ctx *ctx, double tol) {
    int rc;
    if (!ctx->w_is_delta) {
        if ((rc = step_delta<R>(ctx, &ctx->st->done)) != LGF_OK) return rc;
        ctx->w_is_delta = true;
    }
    // W / `partial` may have been filled by lgf_measure or lgf_step_delta, which record nothing: the
    // history entry of this configuration (and the loop test) is still owed
    if (!ctx->recorded) {
        if ((rc = step_finalize(ctx, tol, 0, 1)) != LGF_OK) return rc;
        ctx->recorded = true;
    }
    return LGF_OK;
}
// One pass of the while-body of Algorithm 1 (lines 3-17): accelerate, g, sweep (update + measure), then
// the finalize that makes the new configuration current, records (F, theta) and applies the loop test.
// Every kernel returns immediately once the device-side `done` flag is set.
template <class R>
static int iteration(lgf_ctx *ctx, double alpha, double tol) {
    int rc;
    const bool fuse = can_fuse_g(ctx);
    if ((rc = step_accelerate<R>(ctx, fuse, alpha)) != LGF_OK) return rc;
    if ((rc = step_update<R>(ctx, alpha, tol, 1, fuse)) != LGF_OK) return rc;
    ctx->recorded = true;                                // the sweep's finalize appended the new configuration
    return LGF_OK;
}
// a1 on the current configuration without touching the history or the stop flag
template <class R>
static int measure_only(lgf_ctx *ctx) {
    int rc;
    if ((rc = step_delta<R>(ctx, &ctx->st->zero)) != LGF_OK) return rc;
    return step_finalize(ctx, -1.0, 0, 0);
}

template <class R>
static int apply_transform(lgf_ctx *ctx, const void *d_transform) {
    ctx->launches++;
    CK(launch_gacc<R>(3, nullptr, (C<R> *)ctx->G, (R *)const_cast<void *>(d_transform), ctx->g, ctx->st, STRM(ctx)));
    ctx->launches++;
    CK(launch_clear_done(ctx->st, STRM(ctx)));
    // the fused sweep with the given field in the place of g: U <- G U G(x+mu)^dag, Delta / F / theta of the result
    const int rc = step_update<R>(ctx, 0.0, -1.0, 0, true);
    if (rc != LGF_OK) return rc;
    ctx->launches++;
    CK(launch_reset_counters(ctx->st, STRM(ctx)));       // a new starting configuration: history and counters restart
    ctx->w_is_delta = true;                                  // ... whose Delta and partial sums the sweep has left behind
    ctx->recorded = false;
    ctx->updates_enqueued = 0;
    return LGF_OK;
}

// A_mu(k): packed algebra part of direction mu into W, forward transform with one pass per axis (works on every
// supported lattice; leaves each axis in the permuted order of the two-step line transform), unpack to natural
// order.  W is overwritten.
template <class R>
static int gluon_field(lgf_ctx *ctx, int mu, void *d_out) {
    ctx->launches++;
    CK(launch_algebra<R>(ctx->nr, link_pair<R>(ctx), (C<R> *)ctx->W, ctx->g, mu, ctx->st, STRM(ctx)));
    ctx->launches++;
    CK(launch_clear_done(ctx->st, STRM(ctx)));          // the FFT passes return at once while `done` is set
    const R *tw[4] = {(const R *)ctx->twiddle[0], (const R *)ctx->twiddle[1], (const R *)ctx->twiddle[2],
                      (const R *)ctx->twiddle[3]};
    int N1[4], N2[4];
    for (int axis = 0; axis < 4; axis++) {
        line_factor(ctx->g.L[axis], N1[axis], N2[axis]);
        const AxisPass p = make_axis_pass(ctx, axis, FFT_FWD);
        Bracket br(ctx, LGF_K_FFT);
        CK(launch_fft_pass<R>(p, (C<R> *)ctx->W, ctx->g, tw, (const R *)ctx->p2tab, (R)1, ctx->st, STRM(ctx)));
    }
    ctx->launches++;
    CK(launch_gluon_unpack<R>((const C<R> *)ctx->W, (R *)d_out, ctx->g, N1, N2, STRM(ctx)));
    ctx->w_is_delta = false;
    return LGF_OK;
}

#define DISPATCH(fn, ...) (ctx->prec == LGF_FP64 ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))

static int fetch_state(lgf_ctx *ctx) {
    CK(cudaMemcpyAsync(ctx->h_st, ctx->st, sizeof(DevState), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return LGF_OK;
}

// ---- C ABI ----------------------------------------------------------------------------------------
extern "C" {

const char *lgf_version(void) { return "liblgf 0.1 (sm_100a)"; }

const char *lgf_last_error(const lgf_ctx *ctx) { return ctx ? ctx->err.c_str() : g_err.c_str(); }

int lgf_create(const int dims[4], int precision, int link_storage, lgf_ctx **out) {
    if (!dims || !out) return fail(nullptr, LGF_EINVAL, "lgf_create: null argument");
    *out = nullptr;
    if (precision != LGF_FP32 && precision != LGF_FP64) return fail(nullptr, LGF_EINVAL, "lgf_create: bad precision");
    if (link_storage != LGF_LINKS_18 && link_storage != LGF_LINKS_12)
        return fail(nullptr, LGF_EINVAL, "lgf_create: bad link_storage");
    for (int mu = 0; mu < 4; mu++)
        if (!valid_len(dims[mu])) return fail(nullptr, LGF_EINVAL, "lgf_create: unsupported lattice extent");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, LGF_ECUDA, "lgf_create: no CUDA device (liblgf has no CPU path)");
    }
    lgf_ctx *ctx = new (std::nothrow) lgf_ctx();
    if (!ctx) return fail(nullptr, LGF_ENOMEM, "lgf_create: host allocation failed");
    cudaGetDevice(&ctx->device);
    ctx->prec = precision;
    ctx->nr = link_storage == LGF_LINKS_18 ? 3 : 2;
    long long S = 1;
    for (int mu = 0; mu < 4; mu++) { ctx->g.L[mu] = dims[mu]; ctx->g.S[mu] = S; S *= dims[mu]; }
    ctx->g.V = S;
    const size_t V = (size_t)S, cb = 2 * (size_t)precision;
    int rc = LGF_OK;
    auto alloc = [&](void **p, size_t bytes) {
        if (rc != LGF_OK) return;
        cudaError_t ee = cudaMalloc(p, bytes);
        if (ee != cudaSuccess) rc = cuda_fail(ctx, ee, "cudaMalloc");
    };
    alloc(&ctx->links[0], V * 4 * 3 * ctx->nr * cb);
    alloc(&ctx->links[1], V * 4 * 3 * ctx->nr * cb);
    alloc(&ctx->W, V * 4 * cb);
    alloc(&ctx->G, V * 6 * cb);
    ctx->partial_cap = (int)((V + 127) / 128) + 1;   // >= the CTA count of every kernel that writes per-CTA partial sums
    alloc((void **)&ctx->partial, sizeof(double) * 4 * ctx->partial_cap);
    alloc((void **)&ctx->st, sizeof(DevState));
    ctx->hist_cap = 1 << 20;
    alloc((void **)&ctx->hist, sizeof(double) * 2 * ctx->hist_cap);
    alloc((void **)&ctx->d_scalar, sizeof(double) * 4);
    if (rc == LGF_OK) {
        cudaError_t ee = cudaMallocHost((void **)&ctx->h_st, sizeof(DevState) + 4 * sizeof(double));
        if (ee != cudaSuccess) rc = cuda_fail(ctx, ee, "cudaMallocHost");
    }
    if (rc == LGF_OK) {
        cudaError_t ee = cudaMallocHost((void **)&ctx->h_poll, 2 * sizeof(DevState));
        for (int k = 0; k < 2 && ee == cudaSuccess; k++) ee = cudaEventCreateWithFlags(&ctx->poll_ev[k], cudaEventDisableTiming);
        if (ee != cudaSuccess) rc = cuda_fail(ctx, ee, "poll buffers");
    }
    if (rc == LGF_OK) rc = precision == LGF_FP64 ? upload_twiddles<double>(ctx) : upload_twiddles<float>(ctx);
    if (rc == LGF_OK) rc = plan_passes(ctx);
    if (rc == LGF_OK) ctx->sweep_maps = sweep_tma_maps_create(ctx->g, ctx->nr, ctx->prec, ctx->links[0], ctx->links[1], ctx->G);
    if (rc == LGF_OK) {
        cudaError_t ee = launch_reset_state(ctx->st, STRM(ctx));
        if (ee == cudaSuccess) ee = cudaStreamSynchronize(ctx->stream);
        if (ee != cudaSuccess) rc = cuda_fail(ctx, ee, "reset_state");
    }
    if (rc != LGF_OK) {
        g_err = ctx->err;
        lgf_destroy(ctx);
        return rc;
    }
    *out = ctx;
    return LGF_OK;
}

int lgf_destroy(lgf_ctx *ctx) {
    if (!ctx) return LGF_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    drain_stamps(ctx);
    cudaFree(ctx->links[0]);
    cudaFree(ctx->links[1]);
    cudaFree(ctx->W);
    cudaFree(ctx->G);
    cudaFree(ctx->Gacc);
    cudaFree(ctx->partial);
    cudaFree(ctx->st);
    cudaFree(ctx->hist);
    cudaFree(ctx->d_scalar);
    cudaFree(ctx->p2tab);
    cudaFree(ctx->stage[0]);
    cudaFree(ctx->stage[1]);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    for (int k = 0; k < 2; k++) {
        if (ctx->ev_full[k]) cudaEventDestroy(ctx->ev_full[k]);
        if (ctx->ev_free[k]) cudaEventDestroy(ctx->ev_free[k]);
    }
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    sweep_tma_maps_destroy(ctx->sweep_maps);
    for (int mu = 0; mu < 4; mu++) cudaFree(ctx->twiddle[mu]);
    if (ctx->h_st) cudaFreeHost(ctx->h_st);
    if (ctx->h_poll) cudaFreeHost(ctx->h_poll);
    for (int k = 0; k < 2; k++) if (ctx->poll_ev[k]) cudaEventDestroy(ctx->poll_ev[k]);
    cudaGetLastError();
    delete ctx;
    return LGF_OK;
}

int lgf_set_stream(lgf_ctx *ctx, void *cuda_stream) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    ctx->stream = (cudaStream_t)cuda_stream;
    return LGF_OK;
}

// after the internal link buffer 0 has been filled: accumulated transformation, state and host-side flags start again
static int links_loaded(lgf_ctx *ctx) {
    if (ctx->Gacc) {
        ctx->launches++;
        if (ctx->prec == LGF_FP64)
            CK(launch_gacc<double>(0, nullptr, (C<double> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
        else
            CK(launch_gacc<float>(0, nullptr, (C<float> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
    }
    ctx->launches++;
    CK(launch_reset_state(ctx->st, STRM(ctx)));          // also makes buffer 0 the current one
    ctx->have_links = true;
    ctx->w_is_delta = false;
    ctx->recorded = false;
    ctx->hb_sweeps = 0;
    ctx->updates_enqueued = 0;
    return LGF_OK;
}

int lgf_set_links(lgf_ctx *ctx, const void *d_links) {
    if (!ctx || !d_links) return fail(ctx, LGF_EINVAL, "lgf_set_links: null argument");
    ENTER(ctx);
    {
        Bracket br(ctx, LGF_K_CONVERT);
        if (ctx->prec == LGF_FP64)
            CK(launch_convert_in<double>(ctx->nr, (const double *)d_links, (C<double> *)ctx->links[0], ctx->g, STRM(ctx)));
        else
            CK(launch_convert_in<float>(ctx->nr, (const float *)d_links, (C<float> *)ctx->links[0], ctx->g, STRM(ctx)));
    }
    return links_loaded(ctx);
}

int lgf_get_links(lgf_ctx *ctx, void *d_links) {
    if (!ctx || !d_links) return fail(ctx, LGF_EINVAL, "lgf_get_links: null argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_get_links: no configuration loaded");
    ENTER(ctx);
    Bracket br(ctx, LGF_K_CONVERT);
    if (ctx->prec == LGF_FP64)
        CK(launch_convert_out<double>(ctx->nr, link_pair<double>(ctx), (double *)d_links, ctx->g, ctx->st, STRM(ctx)));
    else
        CK(launch_convert_out<float>(ctx->nr, link_pair<float>(ctx), (float *)d_links, ctx->g, ctx->st, STRM(ctx)));
    return LGF_OK;
}

static int ensure_staging(lgf_ctx *ctx) {
    if (ctx->stage[0]) return LGF_OK;
    const long long CH = 1LL << 16;                        // sites per chunk: 37.7 MB in fp64
    ctx->stage_sites = ctx->g.V < CH ? ctx->g.V : CH;
    for (int k = 0; k < 2; k++) {
        CK(cudaMalloc(&ctx->stage[k], (size_t)ctx->stage_sites * 72 * ctx->prec));
        CK(cudaEventCreateWithFlags(&ctx->ev_full[k], cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->ev_free[k], cudaEventDisableTiming));
    }
    CK(cudaEventCreateWithFlags(&ctx->ev_start, cudaEventDisableTiming));
    CK(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    return LGF_OK;
}

int lgf_set_links_host(lgf_ctx *ctx, const void *h_links) {
    if (!ctx || !h_links) return fail(ctx, LGF_EINVAL, "lgf_set_links_host: null argument");
    ENTER(ctx);
    int rc = ensure_staging(ctx);
    if (rc != LGF_OK) return rc;
    const size_t site_bytes = (size_t)72 * ctx->prec;
    CK(cudaEventRecord(ctx->ev_start, ctx->stream));       // the copies start after whatever the stream still does
    CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_start, 0));
    int c = 0;
    for (long long s0 = 0; s0 < ctx->g.V; s0 += ctx->stage_sites, c++) {
        const int b = c & 1;
        const long long n = ctx->g.V - s0 < ctx->stage_sites ? ctx->g.V - s0 : ctx->stage_sites;
        if (c >= 2) CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_free[b], 0));     // its conversion has read the buffer
        CK(cudaMemcpyAsync(ctx->stage[b], (const char *)h_links + (size_t)s0 * site_bytes, (size_t)n * site_bytes,
                           cudaMemcpyHostToDevice, ctx->copy_stream));
        CK(cudaEventRecord(ctx->ev_full[b], ctx->copy_stream));
        CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_full[b], 0));
        {
            Bracket br(ctx, LGF_K_CONVERT);
            if (ctx->prec == LGF_FP64)
                CK(launch_convert_in<double>(ctx->nr, (const double *)ctx->stage[b], (C<double> *)ctx->links[0], ctx->g, STRM(ctx), s0, n));
            else
                CK(launch_convert_in<float>(ctx->nr, (const float *)ctx->stage[b], (C<float> *)ctx->links[0], ctx->g, STRM(ctx), s0, n));
        }
        CK(cudaEventRecord(ctx->ev_free[b], ctx->stream));
    }
    rc = links_loaded(ctx);
    if (rc != LGF_OK) return rc;
    CK(cudaStreamSynchronize(ctx->stream));
    return LGF_OK;
}

int lgf_get_links_host(lgf_ctx *ctx, void *h_links) {
    if (!ctx || !h_links) return fail(ctx, LGF_EINVAL, "lgf_get_links_host: null argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_get_links_host: no configuration loaded");
    ENTER(ctx);
    int rc = ensure_staging(ctx);
    if (rc != LGF_OK) return rc;
    const size_t site_bytes = (size_t)72 * ctx->prec;
    int c = 0;
    for (long long s0 = 0; s0 < ctx->g.V; s0 += ctx->stage_sites, c++) {
        const int b = c & 1;
        const long long n = ctx->g.V - s0 < ctx->stage_sites ? ctx->g.V - s0 : ctx->stage_sites;
        if (c >= 2) CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_free[b], 0));          // its copy has left the buffer
        {
            Bracket br(ctx, LGF_K_CONVERT);
            if (ctx->prec == LGF_FP64)
                CK(launch_convert_out<double>(ctx->nr, link_pair<double>(ctx), (double *)ctx->stage[b], ctx->g, ctx->st, STRM(ctx), s0, n));
            else
                CK(launch_convert_out<float>(ctx->nr, link_pair<float>(ctx), (float *)ctx->stage[b], ctx->g, ctx->st, STRM(ctx), s0, n));
        }
        CK(cudaEventRecord(ctx->ev_full[b], ctx->stream));
        CK(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_full[b], 0));
        CK(cudaMemcpyAsync((char *)h_links + (size_t)s0 * site_bytes, ctx->stage[b], (size_t)n * site_bytes, cudaMemcpyDeviceToHost,
                           ctx->copy_stream));
        CK(cudaEventRecord(ctx->ev_free[b], ctx->copy_stream));
    }
    CK(cudaStreamSynchronize(ctx->copy_stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return LGF_OK;
}

int lgf_iterate(lgf_ctx *ctx, double alpha, int n) {
    if (!ctx || n < 0) return fail(ctx, LGF_EINVAL, "lgf_iterate: bad argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_iterate: no configuration loaded");
    ENTER(ctx);
    ctx->launches++;
    CK(launch_clear_done(ctx->st, STRM(ctx)));
    // tol = -1: theta >= 0 never stops the loop; only a NaN does
    int rc = DISPATCH(first_measure, ctx, -1.0);
    if (rc != LGF_OK) return rc;
    for (int i = 0; i < n; i++)
        if ((rc = DISPATCH(iteration, ctx, alpha, -1.0)) != LGF_OK) return rc;
    return LGF_OK;
}

int lgf_measure(lgf_ctx *ctx, double *F, double *theta, double *plaquette) {
    if (!ctx) return LGF_EINVAL;
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_measure: no configuration loaded");
    ENTER(ctx);
    if (plaquette) {                 // uses the second half of the partial-sum buffer
        int nb = 0;
        double *part = ctx->partial + 2 * ctx->partial_cap;
        {
            Bracket br(ctx, LGF_K_PLAQ);
            if (ctx->prec == LGF_FP64)
                CK(launch_plaquette<double>(ctx->nr, link_pair<double>(ctx), ctx->g, part, &nb, ctx->st, STRM(ctx)));
            else
                CK(launch_plaquette<float>(ctx->nr, link_pair<float>(ctx), ctx->g, part, &nb, ctx->st, STRM(ctx)));
        }
        ctx->launches++;
        CK(launch_sum1(part, nb, 1.0 / (18.0 * (double)ctx->g.V), ctx->d_scalar, STRM(ctx)));
        double *hp = reinterpret_cast<double *>(ctx->h_st + 1);
        CK(cudaMemcpyAsync(hp, ctx->d_scalar, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    }
    if (F || theta) {
        const int rc = DISPATCH(measure_only, ctx);
        if (rc != LGF_OK) return rc;
        ctx->w_is_delta = true;
    }
    const int rc = fetch_state(ctx);
    if (rc != LGF_OK) return rc;
    if (F) *F = ctx->h_st->F;
    if (theta) *theta = ctx->h_st->theta;
    if (plaquette) *plaquette = *reinterpret_cast<double *>(ctx->h_st + 1);
    return LGF_OK;
}

// Algorithm 1 on the configuration already loaded in the context.
static long long fix_loaded(lgf_ctx *ctx, double alpha, double tol, long long max_iter) {
    const int CHUNK = 16;      // iterations enqueued between two looks at the device-side stop flag
    int rc = DISPATCH(first_measure, ctx, tol);                         // line 1 (+ the first loop test)
    if (rc != LGF_OK) return rc;
    // The host looks at the device-side stop flag once per chunk, one chunk behind: chunk k + 1 is already
    // enqueued when the copy of the flag taken after chunk k is waited for, so the GPU never idles on the
    // host (a look with a full synchronisation every 16 iterations cost 9 % at 32^4).  Iterations enqueued
    // past convergence return at once: every kernel tests the flag.
    long long issued = 0;
    int enq = 0, seen = 0;          // looks (flag copies) enqueued / waited for; look k lives in slot k & 1
    bool done = false;
    while (!done && issued < max_iter) {
        const long long n = (max_iter - issued < CHUNK) ? (max_iter - issued) : CHUNK;
        for (long long i = 0; i < n; i++)
            if ((rc = DISPATCH(iteration, ctx, alpha, tol)) != LGF_OK) return rc;
        issued += n;
        // at most one look is outstanding here (enq - seen <= 1), so slot enq & 1 is free
        CK(cudaMemcpyAsync(&ctx->h_poll[enq & 1], ctx->st, sizeof(DevState), cudaMemcpyDeviceToHost, ctx->stream));
        CK(cudaEventRecord(ctx->poll_ev[enq & 1], ctx->stream));
        enq++;
        if (enq - seen >= 2) {      // wait for the look taken one chunk ago; the chunk just enqueued keeps the GPU busy
            CK(cudaEventSynchronize(ctx->poll_ev[seen & 1]));
            done = ctx->h_poll[seen & 1].done != 0;
            seen++;
        }
    }
    if ((rc = fetch_state(ctx)) != LGF_OK) return rc;
    // iterations enqueued past convergence were no-ops: the projection schedule ("reunit_every") of a later call
    // must count the updates that were applied, not the ones that were enqueued
    ctx->updates_enqueued = ctx->h_st->n_updates;
    if (ctx->h_st->nan) return fail(ctx, LGF_ENAN, "lgf_fix: theta is NaN/Inf");
    return ctx->h_st->n_updates;
}

long long lgf_fix(lgf_ctx *ctx, void *d_links, double alpha, double tol, long long max_iter) {
    if (!ctx || !d_links || max_iter < 0) return fail(ctx, LGF_EINVAL, "lgf_fix: bad argument");
    ENTER(ctx);
    int rc = lgf_set_links(ctx, d_links);
    if (rc != LGF_OK) return rc;
    const long long it = fix_loaded(ctx, alpha, tol, max_iter);
    if (it < 0) return it;
    if ((rc = lgf_get_links(ctx, d_links)) != LGF_OK) return rc;
    CK(cudaStreamSynchronize(ctx->stream));
    return it;
}

long long lgf_fix_host(lgf_ctx *ctx, void *h_links, double alpha, double tol, long long max_iter) {
    if (!ctx || !h_links || max_iter < 0) return fail(ctx, LGF_EINVAL, "lgf_fix_host: bad argument");
    ENTER(ctx);
    int rc = lgf_set_links_host(ctx, h_links);
    if (rc != LGF_OK) return rc;
    const long long it = fix_loaded(ctx, alpha, tol, max_iter);
    if (it < 0) return it;
    if ((rc = lgf_get_links_host(ctx, h_links)) != LGF_OK) return rc;
    return it;
}

int lgf_history(lgf_ctx *ctx, long long first, long long count, double *F, double *theta) {
    if (!ctx || first < 0 || count < 0) return fail(ctx, LGF_EINVAL, "lgf_history: bad argument");
    ENTER(ctx);
    int rc = fetch_state(ctx);
    if (rc != LGF_OK) return rc;
    const long long have = ctx->h_st->n_hist < ctx->hist_cap ? ctx->h_st->n_hist : ctx->hist_cap;
    if (first + count > have) return fail(ctx, LGF_EINVAL, "lgf_history: range beyond the recorded entries");
    if (count == 0) return LGF_OK;
    std::vector<double> buf(2 * (size_t)count);
    CK(cudaMemcpyAsync(buf.data(), ctx->hist + 2 * first, sizeof(double) * 2 * count, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    for (long long i = 0; i < count; i++) {
        if (F) F[i] = buf[2 * i];
        if (theta) theta[i] = buf[2 * i + 1];
    }
    return LGF_OK;
}

long long lgf_iterations(lgf_ctx *ctx) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    const int rc = fetch_state(ctx);
    if (rc != LGF_OK) return rc;
    return ctx->h_st->n_updates;
}

long long lgf_history_length(lgf_ctx *ctx) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    const int rc = fetch_state(ctx);
    if (rc != LGF_OK) return rc;
    return ctx->h_st->n_hist;
}

int lgf_step_delta(lgf_ctx *ctx, double *F, double *theta) {
    if (!ctx) return LGF_EINVAL;
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_step_delta: no configuration loaded");
    ENTER(ctx);
    int rc = DISPATCH(measure_only, ctx);
    if (rc != LGF_OK) return rc;
    ctx->w_is_delta = true;
    if (F || theta) {
        if ((rc = fetch_state(ctx)) != LGF_OK) return rc;
        if (F) *F = ctx->h_st->F;
        if (theta) *theta = ctx->h_st->theta;
    }
    return LGF_OK;
}

int lgf_step_accelerate(lgf_ctx *ctx) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    ctx->launches++;
    CK(launch_clear_done(ctx->st, STRM(ctx)));
    ctx->w_is_delta = false;
    return DISPATCH(step_accelerate, ctx, false, 0.0);
}

int lgf_step_update(lgf_ctx *ctx, double alpha) {
    if (!ctx) return LGF_EINVAL;
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_step_update: no configuration loaded");
    ENTER(ctx);
    ctx->launches++;
    CK(launch_clear_done(ctx->st, STRM(ctx)));
    const int rc = DISPATCH(step_update, ctx, alpha, -1.0, 0, false);
    if (rc != LGF_OK) return rc;
    ctx->w_is_delta = true;            // the sweep left Delta of the new links in W
    ctx->recorded = false;             // ... but nothing about them in the history
    return LGF_OK;
}

int lgf_get_field(lgf_ctx *ctx, void *d_field) {
    if (!ctx || !d_field) return fail(ctx, LGF_EINVAL, "lgf_get_field: null argument");
    ENTER(ctx);
    ctx->launches++;
    if (ctx->prec == LGF_FP64) CK(launch_field_get<double>((const C<double> *)ctx->W, (double *)d_field, ctx->g, STRM(ctx)));
    else CK(launch_field_get<float>((const C<float> *)ctx->W, (float *)d_field, ctx->g, STRM(ctx)));
    return LGF_OK;
}

int lgf_set_field(lgf_ctx *ctx, const void *d_field) {
    if (!ctx || !d_field) return fail(ctx, LGF_EINVAL, "lgf_set_field: null argument");
    ENTER(ctx);
    ctx->launches++;
    if (ctx->prec == LGF_FP64) CK(launch_field_set<double>((C<double> *)ctx->W, (const double *)d_field, ctx->g, STRM(ctx)));
    else CK(launch_field_set<float>((C<float> *)ctx->W, (const float *)d_field, ctx->g, STRM(ctx)));
    ctx->w_is_delta = false;
    return LGF_OK;
}

// heat-bath (overrelax = false) or overrelaxation sweeps of the internal configuration
static int monte_carlo_sweeps(lgf_ctx *ctx, double beta, int nsweeps, unsigned long long seed, bool overrelax) {
    for (int mu = 0; mu < 4; mu++)
        if (ctx->g.L[mu] % 2) return fail(ctx, LGF_EINVAL, "the checkerboard update needs even extents");
    const unsigned long long key = heatbath_key(seed);
    for (int sw = 0; sw < nsweeps; sw++) {
        for (int mu = 0; mu < 4; mu++)
            for (int parity = 0; parity < 2; parity++) {
                Bracket br(ctx, LGF_K_HEATBATH);
                if (ctx->prec == LGF_FP64)
                    CK(launch_heatbath<double>(ctx->nr, link_pair<double>(ctx), ctx->g, ctx->st, beta, key, ctx->hb_sweeps,
                                               mu, parity, STRM(ctx), overrelax, ctx->tune_hb_tz));
                else
                    CK(launch_heatbath<float>(ctx->nr, link_pair<float>(ctx), ctx->g, ctx->st, beta, key, ctx->hb_sweeps, mu,
                                              parity, STRM(ctx), overrelax, ctx->tune_hb_tz));
            }
        if (!overrelax) ctx->hb_sweeps++;                // only heat-bath sweeps consume random numbers
    }
    // a new configuration: the history, the counters and the accumulated transformation start again
    ctx->launches++;
    CK(launch_reset_counters(ctx->st, STRM(ctx)));
    ctx->w_is_delta = false;
    ctx->recorded = false;
    ctx->updates_enqueued = 0;
    if (ctx->Gacc) {
        ctx->launches++;
        if (ctx->prec == LGF_FP64)
            CK(launch_gacc<double>(0, nullptr, (C<double> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
        else
            CK(launch_gacc<float>(0, nullptr, (C<float> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
    }
    return LGF_OK;
}

int lgf_thermalize(lgf_ctx *ctx, double beta, int nsweeps, unsigned long long seed) {
    if (!ctx || nsweeps < 0 || !(beta > 0.0)) return fail(ctx, LGF_EINVAL, "lgf_thermalize: bad argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_thermalize: no configuration loaded");
    ENTER(ctx);
    return monte_carlo_sweeps(ctx, beta, nsweeps, seed, false);
}

int lgf_overrelax(lgf_ctx *ctx, int nsweeps) {
    if (!ctx || nsweeps < 0) return fail(ctx, LGF_EINVAL, "lgf_overrelax: bad argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_overrelax: no configuration loaded");
    ENTER(ctx);
    return monte_carlo_sweeps(ctx, 0.0, nsweeps, 0, true);
}

int lgf_track_transform(lgf_ctx *ctx, int on) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    if (!on) {
        cudaFree(ctx->Gacc);
        ctx->Gacc = nullptr;
        return LGF_OK;
    }
    if (!ctx->Gacc) CK(cudaMalloc(&ctx->Gacc, (size_t)ctx->g.V * 9 * 2 * ctx->prec));
    ctx->launches++;
    if (ctx->prec == LGF_FP64)
        CK(launch_gacc<double>(0, nullptr, (C<double> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
    else
        CK(launch_gacc<float>(0, nullptr, (C<float> *)ctx->Gacc, nullptr, ctx->g, ctx->st, STRM(ctx)));
    return LGF_OK;
}

int lgf_get_transform(lgf_ctx *ctx, void *d_transform) {
    if (!ctx || !d_transform) return fail(ctx, LGF_EINVAL, "lgf_get_transform: null argument");
    if (!ctx->Gacc) return fail(ctx, LGF_ESTATE, "lgf_get_transform: tracking is off (lgf_track_transform)");
    ENTER(ctx);
    ctx->launches++;
    if (ctx->prec == LGF_FP64)
        CK(launch_gacc<double>(2, nullptr, (C<double> *)ctx->Gacc, (double *)d_transform, ctx->g, ctx->st, STRM(ctx)));
    else
        CK(launch_gacc<float>(2, nullptr, (C<float> *)ctx->Gacc, (float *)d_transform, ctx->g, ctx->st, STRM(ctx)));
    return LGF_OK;
}

int lgf_gluon_field(lgf_ctx *ctx, int mu, void *d_out) {
    if (!ctx || !d_out || mu < 0 || mu > 3) return fail(ctx, LGF_EINVAL, "lgf_gluon_field: bad argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_gluon_field: no configuration loaded");
    ENTER(ctx);
    return ctx->prec == LGF_FP64 ? gluon_field<double>(ctx, mu, d_out) : gluon_field<float>(ctx, mu, d_out);
}

int lgf_apply_transform(lgf_ctx *ctx, const void *d_transform) {
    if (!ctx || !d_transform) return fail(ctx, LGF_EINVAL, "lgf_apply_transform: null argument");
    if (!ctx->have_links) return fail(ctx, LGF_ESTATE, "lgf_apply_transform: no configuration loaded");
    ENTER(ctx);
    return ctx->prec == LGF_FP64 ? apply_transform<double>(ctx, d_transform) : apply_transform<float>(ctx, d_transform);
}

int lgf_tune(lgf_ctx *ctx, const char *key, int value) {
    if (!ctx || !key) return fail(ctx, LGF_EINVAL, "lgf_tune: null argument");
    ENTER(ctx);
    const std::string k(key);
    if (k == "fft_two_axis") ctx->tune_two_axis = value;
    else if (k == "fft_reg") ctx->tune_reg = value;
    else if (k == "fft_reg2") ctx->tune_reg2 = value;
    else if (k == "fft_xy_planes") ctx->tune_xy_planes = value;
    else if (k == "fft_zt_xc") ctx->tune_zt_xc = value;
    else if (k == "fuse_g") ctx->tune_fuse_g = value;
    else if (k == "pdl") ctx->tune_pdl = value != 0;               // programmatic dependent launch of this context's kernels
    else if (k == "sweep_tz") ctx->tune_sweep_tz = value;
    else if (k == "hb_tz") ctx->tune_hb_tz = value;
    else if (k == "sweep_share") ctx->tune_sweep_share = value;
    else if (k == "sweep_tma") ctx->tune_sweep_tma = value;
    else if (k == "fft_bulk") ctx->tune_fft_bulk = value;
    else if (k == "fft_zt_cluster") ctx->tune_fft_zt_cluster = value;
    else if (k == "sweep_rsplit") ctx->tune_sweep_rsplit = value;
    else if (k == "sweep_prefetch") ctx->tune_sweep_ahead = value < 0 ? 0 : value;
    else if (k == "sweep_minb") ctx->tune_sweep_minb = (value == 2 || value == 3 || value == 4 || value == 5) ? value : 0;
    else if (k == "reunit_every") ctx->tune_reunit = value < 0 ? 0 : value;
    else return fail(ctx, LGF_EINVAL, "lgf_tune: unknown key " + k);
    CK(cudaStreamSynchronize(ctx->stream));
    return plan_passes(ctx);
}

int lgf_fft_passes(const lgf_ctx *ctx) { return ctx ? (int)ctx->passes.size() : LGF_EINVAL; }

int lgf_set_profiling(lgf_ctx *ctx, int on) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    drain_stamps(ctx);
    ctx->profiling = on != 0;
    for (int k = 0; k < LGF_K_COUNT; k++) { ctx->prof_ms[k] = 0.0; ctx->prof_n[k] = 0; }
    return LGF_OK;
}

int lgf_kernel_times(lgf_ctx *ctx, double *ms, long long *launches) {
    if (!ctx) return LGF_EINVAL;
    ENTER(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    drain_stamps(ctx);
    for (int k = 0; k < LGF_K_COUNT; k++) {
        if (ms) ms[k] = ctx->prof_ms[k];
        if (launches) launches[k] = ctx->prof_n[k];
    }
    return LGF_OK;
}

int lgf_kernel_names(const lgf_ctx *ctx, char *buf, int cap) {
    if (!ctx || !buf || cap <= 0) return LGF_EINVAL;
    std::string s = "update=" + (use_sweep_tma(ctx) ? sweep_tma_kernel_name(ctx->g, ctx->nr, ctx->prec, false, ctx->tune_sweep_rsplit != 0)
                                                  : sweep_kernel_name(ctx->g, ctx->nr, ctx->prec, false, ctx->tune_sweep_share,
                                                                      ctx->tune_sweep_minb)) + ";fft=";
    const bool fuse = can_fuse_g(ctx);
    for (size_t i = 0; i < ctx->passes.size(); i++) {
        const AxisPass &p = ctx->passes[i];
        if (i) s += "|";
        if (p.kind == PASS_REG2) s += fft_reg2_kernel_name((fuse && p.axis == 2) ? 3 : p.axis, ctx->g, ctx->prec, use_fft_bulk(ctx), use_zt_cluster(ctx));
        else if (p.kind == PASS_REG) s += p.axis == 1 ? "k_fftr_zt<" : "k_fftr_xy<";
        else s += p.kind == PASS_XY ? "k_fft_xy<" : (p.kind == PASS_ZT ? "k_fft_zt<" : "k_fft_axis<");
    }
    s += std::string(";gbuild=k_gbuild<") + (ctx->prec == 8 ? "double>" : "float>");
    s += std::string(";delta=k_delta<") + (ctx->prec == 8 ? "double, " : "float, ") + std::to_string(ctx->nr) + ">";
    if ((int)s.size() + 1 > cap) return LGF_EINVAL;
    memcpy(buf, s.c_str(), s.size() + 1);
    return LGF_OK;
}

long long lgf_launch_count(const lgf_ctx *ctx) { return ctx ? ctx->launches : LGF_EINVAL; }

double lgf_algorithmic_bytes(const lgf_ctx *ctx, int kernel_class) {
    if (!ctx) return 0.0;
    const double V = (double)ctx->g.V, R = (double)ctx->prec, nl = 6.0 * ctx->nr;
    switch (kernel_class) {
        case LGF_K_DELTA: return V * (4.0 * nl + 8.0) * R;        // read 4 links, write packed Delta
        case LGF_K_FFT: return V * 3.0 * 16.0 * R;                // three read+write sweeps of the packed field
        case LGF_K_UPDATE: return V * (8.0 * nl + 16.0) * R;      // fused sweep: read w-equivalent + 4 links, write 4 links + Delta
        case LGF_K_GBUILD: return V * 20.0 * R;                   // read w (8), write rows 0, 1 of g (12)
        case LGF_K_ITERATION: return V * (12.0 * nl + 64.0) * R;  // SURVEY.md section 8(d) yard-stick
        case LGF_K_PLAQ: return V * 4.0 * nl * R;
        case LGF_K_HEATBATH: return V * 36.0 * nl * R;            // one SWEEP = 8 class passes, each reading every
                                                                  // link once (4 V) and writing V / 2
        case LGF_K_CONVERT: return V * (72.0 + 4.0 * nl) * R;
        default: return 0.0;
    }
}

}  // extern "C"
