// lgf_state.cuh -- device-resident control block of one context and the launch-side declarations
// shared by the translation units of liblgf.  Part of the CUDA path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include "lgf_su3.cuh"
#include "lgf_pdl.cuh"

namespace lgf {

// Lives in device memory; written only by k_finalize / k_reset, read by every kernel of the
// iteration so that Algorithm 1's "while theta >= eps" needs no host round trip:
// once `done` is set every later kernel of the enqueued iterations returns immediately.
struct DevState {
    long long n_hist;     // (F, theta) entries recorded since the last set_links
    long long n_updates;  // link updates applied since the last set_links
    int done;             // theta < tol seen (or NaN)
    int nan;              // theta was NaN / Inf
    double F, theta;      // last measured values
    int zero;             // always 0: the `stop` word handed to kernels that must run regardless of `done`
    int cur;              // which of the two link buffers holds the current configuration (0 / 1); the
                          // sweep reads buffer `cur` and writes the other one, k_finalize flips it
};



// The two link buffers (ping-pong: the fused sweep needs U_mu(x - mu) of the OLD configuration while
// other threads already write the new one).
template <class R>
struct LinkPair {
    C<R> *buf[2];
};

enum FftMode { FFT_FWD = 0, FFT_INV = 1, FFT_FWD_SCALE_INV = 2 };

// (PASS_REG2: the two-threads-per-line register sweeps of lgf_fft_reg2.cu; `axis` as for PASS_REG)
enum PassKind {
    PASS_AXIS = 0,        // one lattice axis per pass (any supported length)
    PASS_XY = 1,          // whole (x, y) planes: both axes transformed in one shared-memory tile
    PASS_ZT = 2,          // (z, t) planes of nlo consecutive (x, y) indices: forward z, t, scale, inverse t, z
    PASS_REG2 = 4,
    PASS_REG = 3          // register-resident line transforms (lgf_fft_reg.cu); `axis` = 0: (x, y) forward,
                          // 1: (z, t) forward + scale + inverse, 2: (x, y) inverse, 3: (x, y) inverse ending in the
                      // g-build (writes G, not W)
};

// One FFT pass (see lgf_fft.cu).
struct AxisPass {
    int kind;             // PassKind
    int axis;             // PASS_AXIS: 0..3
    int L;                // PASS_AXIS: length of that axis; PASS_XY: Lx; PASS_ZT: Lz
    int L2;               // PASS_XY: Ly; PASS_ZT: Lt
    int mode;             // FftMode
    long long S;          // global stride of the axis (elements)
    long long H;          // number of "hi" blocks: V / (S * L)
    int nlo, nhi;         // tile extents: nlo consecutive "lo" indices (lo < S), nhi "hi" indices
                          // (PASS_XY: nhi = planes per CTA; PASS_ZT: nlo = consecutive (x, y) indices per CTA)
    int pitch;            // PASS_ZT: shared-memory stride of t (nlo * Lz + padding)
    int threads;
    size_t smem;
};

// Where g and U_t across the ends of the t range come from: all null on one GPU (periodic inside the buffers);
// on a t-slab (lgf_slab.cu) the neighbouring ranks' halo copies.  One sweep / Delta kernel serves both paths.
template <class R>
struct SweepHalo {
    const C<R> *ghi = nullptr;   // rows 0, 1 of g on the slice above the slab, C<R>[6][S3]
    const C<R> *glo = nullptr;   // ... on the slice below
    C<R> *uhalo = nullptr;       // U_t of the slice below, C<R>[3 NR][S3]; the sweep stores its new value back
};

// launchers implemented in the .cu files (R = float / double)
template <class R>
cudaError_t launch_fft_pass(const AxisPass &p, C<R> *W, const Geom &g, const R *const twiddle[4] /*[2*64] per axis*/,
                            const R *p2tab /*[4][64] permuted 4 sin^2*/, R scale, const DevState *st,
                            LaunchStream stream);
// register-line fast path (lgf_fft_reg.cu): available for this lattice?  is the t axis left in natural k order?
bool fft_reg_supported(const Geom &g);
bool fft_reg_t_natural(const Geom &g);
template <class R>
cudaError_t launch_fft_reg(int which, const Geom &g, C<R> *W, const R *twiddle_t, const R *p2tab, R scale,
                           const DevState *st, LaunchStream stream, C<R> *G = nullptr, R half_alpha = 0);
// two-threads-per-line register sweeps (lgf_fft_reg2.cu)
bool fft_reg2_supported(const Geom &g);
bool fft_reg2_gout(const Geom &g, int prec);
bool fft_reg2_xy_supported(const Geom &g);      // the (x, y) sweeps alone, any (Lz, Lt): the slabs of lgf_slab.cu
bool fft_reg2_xy_gout(const Geom &g, int prec);
bool fft_reg2_xy_by_component(const Geom &g, int prec);
template <class R>
cudaError_t launch_fft_reg2(int which, const Geom &g, C<R> *W, const R *p2tab, R scale, const DevState *st,
                            LaunchStream stream, C<R> *G, R half_alpha, bool bulk = false /* (x, y) planes by bulk copies */,
                            int comp = -1 /* >= 0: forward (x, y) sweep of this packed component only */,
                            int zt_cluster = 0 /* 2 / 4: the (z, t) tile split over a cluster of that many CTAs */);
bool fft_reg2_zt_cluster_supported(const Geom &g, int nc);
// true if a PASS_XY (first two axes) / PASS_ZT (last two axes) kernel is instantiated for these lengths
bool fft_pair_supported(int kind, int La, int Lb);

template <class R>
cudaError_t launch_delta(int nr, LinkPair<R> links, C<R> *W, const Geom &g, double *partial, int *nblocks,
                         const int *stop, const DevState *st, LaunchStream stream,
                         const SweepHalo<R> &halo = SweepHalo<R>());
template <class R>
cudaError_t launch_gbuild(const C<R> *W, C<R> *G, const Geom &g, R half_alpha, const DevState *st, LaunchStream stream);
template <class R>
cudaError_t launch_sweep(int nr, LinkPair<R> links, const C<R> *G, C<R> *W, const Geom &g, double *partial,
                         int *nblocks, const DevState *st, LaunchStream stream, int order_tz /* 0 auto, 1 plain */,
                         bool reunit /* project every new link onto SU(3) */,
                         int share_mode /* A'_x, A'_y through shared memory: 1 / 0 / -1 = where it measured faster */,
                         int ahead /* L2 bulk prefetch of the tile `ahead` CTAs later (0 = none) */,
                         int minb /* resident CTAs per SM the register allocation allows: 0 = automatic (sweep_minb_of), 2, 3, 4 / 5 (fp32) */,
                         const SweepHalo<R> &halo = SweepHalo<R>());
template <class R>
cudaError_t launch_plaquette(int nr, LinkPair<R> links, const Geom &g, double *partial, int *nblocks,
                             const DevState *st, LaunchStream stream);
template <class R>
cudaError_t launch_convert_in(int nr, const R *canon, C<R> *links0, const Geom &g, LaunchStream stream, long long s0 = 0,
                              long long n = -1 /* sites s0 .. s0 + n - 1 from a chunk buffer; -1: all from s0 on */);
template <class R>
cudaError_t launch_convert_out(int nr, LinkPair<R> links, R *canon, const Geom &g, const DevState *st,
                               LaunchStream stream, long long s0 = 0, long long n = -1);
// accumulated gauge transformation: op 0 = set to identity, 1 = Gacc <- g Gacc, 2 = copy out (canonical [s][3][3]),
// 3 = (A = G, out = canonical input field) rows 0, 1 of the SU(3) projection of a given transformation into G
template <class R>
cudaError_t launch_gacc(int op, const C<R> *G, C<R> *A, R *out, const Geom &g, const DevState *st, LaunchStream stream);
// gluon field: W <- packed A_mu(x) of one direction; unpack of its forward transform into natural-order 3 x 3 A_mu(k)
template <class R>
cudaError_t launch_algebra(int nr, LinkPair<R> links, C<R> *W, const Geom &g, int mu, const DevState *st, LaunchStream stream);
template <class R>
cudaError_t launch_gluon_unpack(const C<R> *W, R *out, const Geom &g, const int N1[4], const int N2[4], LaunchStream stream);
template <class R>
cudaError_t launch_field_get(const C<R> *W, R *field, const Geom &g, LaunchStream stream);
template <class R>
cudaError_t launch_field_set(C<R> *W, const R *field, const Geom &g, LaunchStream stream);

// thermalisation (lgf_heatbath.cu): one class (mu, parity) of heat-bath sweep number `sweep`
unsigned long long heatbath_key(unsigned long long seed);
template <class R>
cudaError_t launch_heatbath(int nr, LinkPair<R> links, const Geom &g, const DevState *st, double beta,
                            unsigned long long key, unsigned long long sweep, int mu, int parity, LaunchStream stream,
                            bool overrelax /* R28: alpha = (V^dag)^2, no random numbers */,
                            int order_tz /* z-planes per (z, t) tile of the thread order: 0 = automatic */);
cudaError_t launch_reset_counters(DevState *st, LaunchStream stream);

// the staged sweep (lgf_sweep_tma.cu): TMA tensor copies into a shared-memory ring, persistent warp-specialised CTAs
bool sweep_tma_supported(const Geom &g, int nr, int prec);
bool sweep_tma_auto(const Geom &g, int nr, int prec);      // ... and measured faster than k_sweep for this lattice / variant
struct SweepMaps;     // the TMA tensor maps over a context's two link buffers and its g field
SweepMaps *sweep_tma_maps_create(const Geom &g, int nr, int prec, void *links0, void *links1, void *G);   // null: does not apply
void sweep_tma_maps_destroy(SweepMaps *m);
template <class R>
cudaError_t launch_sweep_tma(const SweepMaps *maps, int nr, LinkPair<R> links, const C<R> *G, C<R> *W, const Geom &g, double *partial,
                             int *nblocks, const DevState *st, LaunchStream stream, int order_tz, bool reunit, const SweepHalo<R> &halo,
                             bool rsplit = true /* fp64: move the producer warps' registers to the compute warps (setmaxnreg) */);
std::string sweep_tma_kernel_name(const Geom &g, int nr, int prec, bool reunit, bool rsplit);

// kernel instantiations as a profiler names them (lgf_kernel_names)
std::string fft_reg2_kernel_name(int which, const Geom &g, int prec, bool bulk = false, int zt_cluster = 0);
int sweep_minb_of(const Geom &g, int prec, bool reunit, bool share, int minb);
std::string sweep_kernel_name(const Geom &g, int nr, int prec, bool reunit, int share_mode, int minb);
bool sweep_uses_share(const Geom &g, int nr, int prec, int share_mode);
// block order of a sweep whose CTAs take `nt` consecutive sites: (z, t)-tiled when a t slice of traffic exceeds L2
BlockOrder sweep_block_order(const Geom &g, int nr, int prec, int order_tz, int nt);

// F / theta finalisation (precision independent)
// after_sweep: the partial sums come from a sweep (flip `cur`, count the update); record: append (F, theta)
// to the history and apply the stop test theta < tol
cudaError_t launch_finalize(const double *partial, int nblocks, long long V, double tol, int after_sweep, int record,
                            DevState *st, double *hist, long long hist_cap, LaunchStream stream);
cudaError_t launch_sum1(const double *partial, int nblocks, double norm, double *out, LaunchStream stream);
cudaError_t launch_reset_state(DevState *st, LaunchStream stream);
cudaError_t launch_clear_done(DevState *st, LaunchStream stream);

}  // namespace lgf
