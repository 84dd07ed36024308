/*
 * lgf.h -- C ABI of liblgf: Fourier-accelerated steepest-descent Landau gauge fixing of a 4-D SU(3)
 * lattice gauge configuration on one NVIDIA B200 (sm_100a).
 *
 * Method: Cardoso, Silva, Bicudo, Oliveira, "Landau Gauge Fixing on GPUs", arXiv:1206.0675.
 * Citations below are "PAPER.md:<line>" of the extracted text plus the equation / algorithm line.
 *
 * One iteration (Algorithm 1) on the configuration {U_mu(x)}:
 *   a1  A_mu(x)  = [(U_mu(x) - U_mu(x)^dag) / 2i] - (1/3) tr[.] 1                       (eq. 7, :75)
 *       Delta(x) = sum_mu [A_mu(x - mu) - A_mu(x)]                                       (eq. 5, :63)
 *       F        = sum_x sum_mu Re tr U_mu(x) / (4 * 3 * V)                              (eq. 3, :52)
 *       theta    = sum_x tr[Delta(x) Delta(x)^dag] / (3 V)                               (eq. 6, :70)
 *   a2  4-D forward FFT of every independent component of Delta                         (Alg. 1 line 4)
 *   a3  multiply by p2max / p2(k), p2 = 4 sum_mu sin^2(pi k_mu / L_mu), p2max = 16, k = 0 -> 0 (line 5, :66)
 *   a4  4-D inverse FFT, normalised by 1/V  ->  w(x)                                    (lines 6-7)
 *   a5  g(x) = reunitarise(1 + i (alpha/2) w(x))   (first-order exp, Gram-Schmidt on rows, row 2 from eq. 8; :66, :148)
 *   a6  U_mu(x) <- g(x) U_mu(x) g(x + mu)^dag  for all x, mu                            (eq. 2, :45; line 14)
 *
 * All of it runs in hand-written CUDA kernels; there is no CPU fallback: every entry point returns
 * LGF_ECUDA if no usable device is present.
 *
 * Conventions
 *   dims[4] = {Lx, Ly, Lz, Lt}; periodic; site index s = x + Lx*(y + Ly*(z + Lz*t)) (x fastest).
 *   Each L_mu must be one of 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64; otherwise LGF_EINVAL.
 *   CANONICAL link layout (what callers pass in and get back): site-major array of structures
 *     links[s][mu][i][j][re/im], mu = 0..3 = x, y, z, t, row-major 3x3, i.e. 72 reals per site,
 *     of type float (LGF_FP32) or double (LGF_FP64) matching the context's precision.
 *     As a torch tensor: shape [Lt, Lz, Ly, Lx, 4, 3, 3, 2].  Always 18 reals per link, whatever the
 *     internal storage.  The library never keeps a caller pointer after the call returns.
 *   Internally links live in a structure-of-arrays layout (18 or 12 reals per link; with
 *     LGF_LINKS_12 only the first two rows are stored and the third is rebuilt as (row0 x row1)^*,
 *     eq. 8); the context owns that storage, the FFT work fields, tables,
 *     reduction scratch and the (F, theta) history.
 *   "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers (pageable or pinned).
 *   All work is enqueued on the context's stream (default: the legacy default stream 0; set it with
 *     lgf_set_stream).  Calls that return values to the host synchronise that stream.
 *   Error handling: every function returns LGF_OK (0) or a negative LGF_E* code (lgf_fix*: the number
 *     of iterations >= 0, or a negative code); nothing throws or aborts across the ABI.  The message
 *     of the last failure is available from lgf_last_error.  One context per host thread.
 */
#ifndef LGF_H
#define LGF_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lgf_ctx lgf_ctx; /* opaque */

enum { LGF_FP32 = 4, LGF_FP64 = 8 };           /* precision = bytes per real                      */
enum { LGF_LINKS_18 = 18, LGF_LINKS_12 = 12 }; /* internal reals per link      */
enum {
    LGF_OK = 0,
    LGF_EINVAL = -1, /* bad argument (dims, precision, storage, null pointer, range)              */
    LGF_ENOMEM = -2, /* device or host allocation failed                                          */
    LGF_ECUDA = -3,  /* CUDA runtime error or no device; see lgf_last_error                       */
    LGF_ESTATE = -4, /* call out of order (e.g. iterate before any links were set)                */
    LGF_ENAN = -5    /* theta became NaN/Inf; iteration stopped                                   */
};

/* Create a context for a lattice of the given dims, arithmetic precision (LGF_FP32 / LGF_FP64; the
 * kernels compute and store in that type, cross-site sums for F and theta are accumulated in fp64)
 * and internal link storage.  Allocates all device buffers on the current CUDA device. */
int lgf_create(const int dims[4], int precision, int link_storage, lgf_ctx **out);
int lgf_destroy(lgf_ctx *ctx);

/* cuda_stream is a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); the caller owns it. */
int lgf_set_stream(lgf_ctx *ctx, void *cuda_stream);

/* Copy a configuration in canonical layout into the context (converts to the internal layout) /
 * copy the current configuration out.  Resets the iteration counter and the history (set only).
 * Asynchronous on the context's stream for device pointers; the host variants return after the
 * host buffer may be reused / has been filled. */
int lgf_set_links(lgf_ctx *ctx, const void *d_links);
int lgf_get_links(lgf_ctx *ctx, void *d_links);
int lgf_set_links_host(lgf_ctx *ctx, const void *h_links);
int lgf_get_links_host(lgf_ctx *ctx, void *h_links);

/* n iterations of Algorithm 1's loop body [a2..a4 -> a5 -> a6 + a1 of the new links] on the internal
 * configuration with step alpha (the paper uses 0.08), regardless of theta.  History
 * entry k holds (F, theta) of the configuration after k updates since the last set_links (entry 0 =
 * the loaded configuration, recorded by the first call), so n iterations from a fresh configuration
 * leave n + 1 entries.  Never blocks the host. */
int lgf_iterate(lgf_ctx *ctx, double alpha, int n);

/* F, theta (a1) and the average plaquette
 *   P = sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag] / (6 * 3 * V)
 * of the current internal configuration.  Any of the out-pointers may be NULL.  Synchronises. */
int lgf_measure(lgf_ctx *ctx, double *F, double *theta, double *plaquette);

/* Algorithm 1: load the configuration at d_links / h_links, then
 *   measure; while (theta >= tol && it < max_iter) { update; measure; ++it }
 * and write the gauge-fixed configuration back to the same buffer.  Returns the number of updates
 * applied (0 if the input already satisfies theta < tol; max_iter if it did not converge -- check
 * with lgf_measure or lgf_history), or a negative LGF_E* code.  History entry n (n = 0..it) holds
 * (F, theta) of the configuration after n updates.  Synchronises. */
long long lgf_fix(lgf_ctx *ctx, void *d_links, double alpha, double tol, long long max_iter);
long long lgf_fix_host(lgf_ctx *ctx, void *h_links, double alpha, double tol, long long max_iter);

/* Copy history entries first .. first+count-1 into F[] and theta[] (host arrays, either may be
 * NULL).  Entries are those recorded since the last set_links / fix.  Synchronises. */
int lgf_history(lgf_ctx *ctx, long long first, long long count, double *F, double *theta);

/* Number of updates applied since the last set_links / fix (synchronises), or a negative code. */
long long lgf_iterations(lgf_ctx *ctx);
/* Number of (F, theta) history entries recorded since the last set_links / fix (synchronises). */
long long lgf_history_length(lgf_ctx *ctx);

/* ---- single steps of the path, exposed so that each row of the hot path can be checked against
 * ---- the oracle element by element (tests) and profiled on its own (bench) ---------------------- */

/* a1 only: Delta(x) of the current configuration into the packed work field W (and F, theta, not
 * recorded in the history).  F / theta may be NULL.  Synchronises if either is non-NULL. */
int lgf_step_delta(lgf_ctx *ctx, double *F, double *theta);
/* a2-a4 only: W <- F^-1 [(16/p2) F W] / V in place. */
int lgf_step_accelerate(lgf_ctx *ctx);
/* a5 + a6 only: g(x) from the current W with step alpha, then the link transform (the fused sweep
 * also leaves Delta of the new configuration in W; nothing is recorded in the history). */
int lgf_step_update(lgf_ctx *ctx, double alpha);
/* The work field as full 3x3 complex matrices, d_field[s][i][j][re/im] (18 reals per site, context
 * precision).  get: unpack W (hermitian traceless by construction).  set: pack a hermitian
 * traceless field into W (the anti-hermitian / trace parts of the argument are ignored). */
int lgf_get_field(lgf_ctx *ctx, void *d_field);
int lgf_set_field(lgf_ctx *ctx, const void *d_field);

/* ---- thermalisation ------------------------------------------------ */

/* nsweeps heat-bath sweeps of the internal configuration with the SU(3) Wilson action
 *   S = beta sum_p [1 - Re tr U_p / 3]
 * -- the producer of the paper's kind of input ("generated via importance sampling using, for example, the
 * Wilson action"; beta = 5.8, 6.0, 6.2, :211).  The paper names no algorithm; this is the
 * Cabibbo-Marinari pseudo-heat-bath over the three SU(2) subgroups with Creutz / Kennedy-Pendleton sampling
 * in checkerboard order, driven by counter-based uniform numbers (readings R24-R27), so that the
 * result is a deterministic function of (loaded configuration, beta, seed, number of sweeps applied since
 * set_links) whatever the split into calls.  Arithmetic in double whatever the context's precision.  All
 * extents must be even (LGF_EINVAL otherwise).  Resets the history, the iteration counter and the
 * accumulated transformation, as loading a new configuration would.  Asynchronous. */
int lgf_thermalize(lgf_ctx *ctx, double beta, int nsweeps, unsigned long long seed);
/* nsweeps microcanonical overrelaxation sweeps (same order and subgroups, alpha = (V^dag)^2 instead of the
 * heat-bath draw, R28): every step leaves the action unchanged, no random numbers are used, so the
 * plaquette is conserved to rounding while the links move by O(1) -- interleaved with lgf_thermalize it
 * shortens the autocorrelation of the ensemble.  Same state reset and error behaviour as lgf_thermalize. */
int lgf_overrelax(lgf_ctx *ctx, int nsweeps);

/* ---- accumulated gauge transformation ----------------------------- */

/* on != 0: keep G(x) = g_n(x) ... g_1(x), the product of the rotations g_k(x) (a5) of all updates applied
 * since the last set_links / fix, so that the current configuration is
 *   U_mu(x) = G(x) U0_mu(x) G(x + mu)^dag        (eq. 2, composed over the iterations)
 * with U0 the loaded one -- what a user needs to carry other fields (quark sources, propagators,
 * PAPER.md:21) into the same gauge.  Costs one extra pass per iteration (12 + 18 + 18 reals per site) and
 * 18 reals per site of device memory.  G is reset to 1 by set_links / fix and by this call.  on == 0
 * frees the storage.  Synchronises. */
int lgf_track_transform(lgf_ctx *ctx, int on);
/* Copy G out: d_transform[s][i][j][re/im], 18 reals per site in the context's precision (as a torch tensor:
 * [Lt, Lz, Ly, Lx, 3, 3] complex).  LGF_ESTATE if tracking is off.  Asynchronous on the context's stream. */
int lgf_get_transform(lgf_ctx *ctx, void *d_transform);

/* Gluon field of direction mu (0..3) in momentum space -- what a Landau-gauge configuration is fixed for
 * (gluon propagator):
 *   d_out[k][i][j] = sum_x exp(-2 pi i sum_nu k_nu x_nu / L_nu) A_mu(x)_ij,   k = kx + Lx (ky + Ly (kz + Lz kt)),
 * A_mu(x) the hermitian traceless algebra part of the current U_mu(x) (eq. 7), unnormalised, the link's field
 * taken at the site x (multiply by exp(-i pi k_mu / L_mu) for the mid-point convention); 18 reals per k in the
 * context's precision (as a torch tensor: [Lt, Lz, Ly, Lx, 3, 3] complex indexed by (kt, kz, ky, kx)).
 * With this convention eq. 5 reads F[Delta](k) = sum_mu (exp(-2 pi i k_mu / L_mu) - 1) A_mu(k): in Landau gauge
 * the field is transverse mode by mode.  Uses the work field (a following lgf_iterate recomputes Delta).
 * Asynchronous. */
int lgf_gluon_field(lgf_ctx *ctx, int mu, void *d_out);

/* Apply a given gauge transformation to the internal configuration: U_mu(x) <- G(x) U_mu(x) G(x + mu)^dag
 * (eq. 2) with d_transform[s][i][j][re/im] in the layout lgf_get_transform writes (18 reals per
 * site, the context's precision).  Each G(x) is first projected onto SU(3) (Gram-Schmidt on rows 0, 1, row 2
 * from eq. 8), so a transformation accumulated in float and converted to double may be passed: the result is
 * an exact gauge transform of the loaded links -- every gauge-invariant quantity is preserved to rounding.
 * Use: find G cheaply (an fp32 context with lgf_track_transform), apply it to the original fp64 links here,
 * finish with lgf_fix in fp64.  Restarts the history and the counters like loading a configuration; an
 * accumulated transformation that is being tracked is multiplied by G.  Asynchronous. */
int lgf_apply_transform(lgf_ctx *ctx, const void *d_transform);

/* ---- tuning --------------------------------------------------------------------------------------- */

/* Override a planner choice of THIS context (takes effect from the next iteration; results are unchanged up
 * to rounding, except for "reunit_every").  Keys: "fft_two_axis" (1 = use the three-sweep two-axis FFT passes when the lattice
 * allows, 0 = one pass per axis), "fft_reg" (1 = use the register-line sweeps when the lattice allows), "fft_xy_planes" ((x, y) planes per CTA, 0 = automatic),
 * "fft_zt_xc" (consecutive (x, y) indices per CTA of the (z, t) pass, 0 = automatic), "fft_reg2" (1 = two
 * threads per line where the lattice allows), "fuse_g" (1 = the last FFT sweep ends with the g-build),
 * "sweep_tz" (z-planes per (z, t) tile of the sweep's CTA order, 0 = automatic, 1 = plain order), "hb_tz" (the
 * same for the thread order of lgf_thermalize / lgf_overrelax, 0 = automatic),
 * "sweep_share" (1 / 0 / -1 = automatic: backward x, y neighbours of the same CTA hand over their algebra parts
 * through shared memory instead of being recomputed), "pdl" (1 / 0: programmatic dependent launch of the
 * iteration's kernels, so that each kernel's launch overlaps the tail of the one before),
 * "sweep_tma" (1 / 0 / -1 = where it measured faster: the persistent staged sweep fed by TMA tensor copies,
 * k_sweep_tma, instead of the register sweep), "sweep_rsplit" (1 / 0: the staged sweep's fp64 register split by
 * setmaxnreg), "sweep_prefetch" (CTAs ahead of which the register sweep prefetches its tile into L2, 0 = off), "sweep_minb"
 * (resident CTAs per SM the register sweep's register allocation allows: 0 = automatic -- 3 in fp64, 4 or 5 in fp32 on
 * lattices that fill them -- or 2 / 3 / 4 / 5), "fft_bulk" (1 / 0 / -1 = where it measured faster: (x, y) FFT
 * sweeps fed by cp.async.bulk), "fft_zt_cluster" (2 / 4: a 64 x 64 (z, t) FFT tile split over a thread-block
 * cluster of that many CTAs with the transposition through distributed shared memory, k_fftr2_zt_cluster; 0 /
 * -1 = the one-CTA tile, which measured faster), "reunit_every" (N > 0: in every
 * N-th update the new links are projected back onto SU(3) inside the sweep; 0 = never, the method as the
 * paper states it -- this key DOES change the result, by the rounding drift it removes; meant for fp32 runs
 * of thousands of iterations).
 * Unknown key or NULL: LGF_EINVAL.  Synchronises. */
int lgf_tune(lgf_ctx *ctx, const char *key, int value);
/* Number of FFT kernel launches per iteration under the current plan (3 or up to 7). */
int lgf_fft_passes(const lgf_ctx *ctx);

/* ---- instrumentation ------------------------------------------------------------------------- */

/* Kernel classes for per-kernel timing. */
enum { LGF_K_DELTA = 0, LGF_K_FFT = 1, LGF_K_UPDATE = 2, LGF_K_GBUILD = 3, LGF_K_CONVERT = 4,
       LGF_K_PLAQ = 5, LGF_K_HEATBATH = 6, LGF_K_COUNT = 7,
       LGF_K_ITERATION = 100 /* lgf_algorithmic_bytes only: the whole-iteration yard-stick */ };
/* When on != 0 every kernel launch is bracketed by CUDA events on the context's stream. */
int lgf_set_profiling(lgf_ctx *ctx, int on);
/* Sum of the event-measured durations (ms) and the number of launches per kernel class since
 * profiling was switched on (arrays of LGF_K_COUNT entries, either may be NULL).  Synchronises. */
int lgf_kernel_times(lgf_ctx *ctx, double *ms, long long *launches);
/* Total number of kernels this context has launched since creation. */
/* The kernel instantiations this context launches for one iteration, as a profiler names them:
 * "update=k_sweep<double, 3, 0, 0, 3>;fft=k_fftr2_xy<...>|k_fftr2_zt<...>|...;gbuild=...;delta=..." into buf (cap bytes
 * including the terminator; LGF_EINVAL if too small).  bench.py uses it to refuse a stored ncu capture of a kernel
 * this build no longer launches. */
int lgf_kernel_names(const lgf_ctx *ctx, char *buf, int cap);
long long lgf_launch_count(const lgf_ctx *ctx);
/* Algorithmic bytes one launch-set of the given kernel class must move for ONE iteration
 * (DESIGN.md "Algorithmic bytes"): e.g. LGF_K_DELTA -> V * (4*n_l + 8) * bytes_per_real;
 * LGF_K_UPDATE is the fused sweep (a6 + a1): V * (8*n_l + 16); LGF_K_ITERATION the whole-iteration
 * yard-stick V * (12*n_l + 64) of SURVEY.md section 8(d). */
double lgf_algorithmic_bytes(const lgf_ctx *ctx, int kernel_class);

const char *lgf_last_error(const lgf_ctx *ctx);
const char *lgf_version(void);

/* ---- one configuration sharded over several GPUs ------
 *
 * Slab decomposition over t: rank r of nranks owns the slices t = r T .. (r+1) T - 1, T = Lt / nranks -- a
 * contiguous piece of the canonical configuration, [T, Lz, Ly, Lx, 4, 3, 3, 2] as a tensor.  nranks must divide
 * Lt and Lz (LGF_EINVAL otherwise): for the t lines of the 4-D FFT the field is redistributed into z-slabs
 * (rank r: z = r Zl .. (r+1) Zl - 1, Zl = Lz / nranks, all t) by an all-to-all.  Every entry point below is
 * LOCAL to one rank: it works on that rank's slab and on device buffers the caller passes in, and the caller
 * moves those buffers between ranks (NCCL send/recv, all-to-all, all-reduce through torch.distributed in
 * paper_1206_0675_b200/slab.py) -- no kernel waits on another rank.  One iteration of Algorithm 1
 * is, on every rank:
 *   halo_pack(LINKS) -> [send to r+1, receive from r-1] -> halo_unpack(LINKS) -> delta(sums) -> [all-reduce sums:
 *   F = sums[0] / (12 V), theta = sums[1] / (3 V), V the GLOBAL volume (eqs. 3, 6)] -> fft_forward(send) ->
 *   [all-to-all] -> fft_t(recv, send) -> [all-to-all] -> fft_inverse_g(recv, alpha) -> halo_pack(G) ->
 *   [send to r-1, receive from r+1] -> halo_unpack(G) -> update,
 * or, with the fused form of the last step (what paper_1206_0675_b200/slab.py iterates with): one such round of
 * halo(LINKS) + delta at the start, then per iteration fft_forward .. fft_inverse_g -> halo_pack(G), halo_pack(G_UP)
 * -> [exchange both ways] -> halo_unpack(G), halo_unpack(G_UP) -> sweep(sums) -> [all-reduce sums].
 * With nranks = 1 the "exchanges" are copies of a rank's send buffer into its own receive buffer (periodic wrap).
 * The result equals the one-GPU path's up to the rounding order of the F / theta sums and of the FFT passes.
 * Same precision / storage / error conventions as above; messages from lgf_slab_last_error.  All calls are
 * asynchronous on the context's stream (default: stream 0). */
typedef struct lgf_slab lgf_slab; /* opaque */
enum { LGF_HALO_LINKS = 0, /* U_t on one 3-D slice: 18 or 12 reals per site (the context's link storage)       */
       LGF_HALO_G = 1,     /* rows 0, 1 of g(x) on one 3-D slice: 12 reals per site                             */
       LGF_HALO_G_UP = 2   /* the same, travelling the other way (fused sweep)                                  */ };

int lgf_slab_create(const int dims[4] /* GLOBAL extents */, int precision, int link_storage, int rank, int nranks,
                    lgf_slab **out);
int lgf_slab_destroy(lgf_slab *ctx);
int lgf_slab_set_stream(lgf_slab *ctx, void *cuda_stream);
/* this rank's slab in canonical layout (72 reals per site, Lx Ly Lz T sites, t slowest) */
int lgf_slab_set_links(lgf_slab *ctx, const void *d_links);
int lgf_slab_get_links(lgf_slab *ctx, void *d_links);
/* number of REALS of one halo buffer (Lx Ly Lz sites times the reals per site above) */
long long lgf_slab_halo_elems(const lgf_slab *ctx, int which);
/* pack: LGF_HALO_LINKS = U_t of the slab's LAST slice (the rank above needs it as U_t(x - t), eq. 5);
 * LGF_HALO_G = g of the slab's FIRST slice (the rank below needs it as g(x + t), eq. 2) into d_send.
 * unpack: take the neighbour's packed slice from d_recv into the context's halo storage. */
int lgf_slab_halo_pack(lgf_slab *ctx, int which, void *d_send);
int lgf_slab_halo_unpack(lgf_slab *ctx, int which, const void *d_recv);
/* a1 on the slab: Delta(x) into the work field; d_sums[0] = sum Re tr U_mu(x), d_sums[1] = sum tr(Delta Delta^dag)
 * over the slab's sites (device doubles, fixed summation order). */
int lgf_slab_delta(lgf_slab *ctx, double *d_sums);
/* The 4-D FFT around the two all-to-alls.  An all-to-all buffer holds 8 reals per local site, ordered
 * [c][q][tl][zl][y][x]: c = 0..3 the packed component of the work field -- each component's quarter of the buffer is
 * an all-to-all of its own --, chunk q (1 / nranks of the quarter) the part that goes to / came from rank q, tl / zl
 * the t / z index inside the chunk (t = q T + tl on the t-slab side's peer, z = q Zl + zl).  The passes next to an all-to-all read and write these buffers directly:
 *   fft_forward:   forward x, y in place, forward z from the work field into d_send                (Alg. 1 line 4)
 *   fft_t:         t lines of this rank's z-slab, d_recv -> d_send (distinct buffers): forward t, times
 *                  p2max / (V p2(k)) with the zero mode set to 0, inverse t                       (lines 4-7)
 *   fft_inverse:   inverse z from d_recv into the work field, inverse y, x: w(x) in the work field  (line 6)
 *   fft_inverse_g: the same, ending in a5, g(x) = GS(1 + i (alpha / 2) w(x)) (line 10) -- fused into the last
 *                  sweep where the lattice allows (the work field then does not hold w) */
int lgf_slab_fft_forward(lgf_slab *ctx, void *d_send);
int lgf_slab_fft_t(lgf_slab *ctx, const void *d_recv, void *d_send);
int lgf_slab_fft_inverse(lgf_slab *ctx, const void *d_recv);
int lgf_slab_fft_inverse_g(lgf_slab *ctx, const void *d_recv, double alpha);
/* The same passes one packed component at a time (comp = 0..3; the four components of the work field are independent
 * fields, and the exchange buffers are component-major, so a component's quarter is one contiguous all-to-all): the
 * caller can run the exchange of component c on another stream while the kernels of component c + 1 run on the
 * context's.  fft_forward_comp = forward x, y and z of that component into its quarter of d_send; fft_t_comp = its t
 * lines, quarter of d_recv -> quarter of d_send; fft_zinv_comp = inverse z of its quarter of d_recv into the work
 * field; then ONCE lgf_slab_fft_xyinv = inverse y, x of all four components (with_g != 0: ending in a5, which needs
 * all of w(x)).  Available when every axis takes the register-line passes (extents 16 / 32 / 64 and whole CTAs of
 * planes per component): lgf_slab_by_component returns 1, else 0 and these calls return LGF_ESTATE. */
int lgf_slab_by_component(const lgf_slab *ctx);
int lgf_slab_fft_forward_comp(lgf_slab *ctx, void *d_send, int comp);
int lgf_slab_fft_t_comp(lgf_slab *ctx, const void *d_recv, void *d_send, int comp);
int lgf_slab_fft_zinv_comp(lgf_slab *ctx, const void *d_recv, int comp);
int lgf_slab_fft_xyinv(lgf_slab *ctx, int with_g, double alpha);
/* a5: g(x) = GS(1 + i (alpha / 2) w(x)) on the slab */
int lgf_slab_gbuild(lgf_slab *ctx, double alpha);
/* a6: U_mu(x) <- g(x) U_mu(x) g(x + mu)^dag on the slab, in place */
int lgf_slab_update(lgf_slab *ctx);
/* a6 + a1 fused (the iteration loop's form): the new links go to the context's second link buffer, and Delta, F
 * and theta of the NEW configuration (Alg. 1 line 17) come out of the same pass -- work field and d_sums as for
 * lgf_slab_delta.  Needs g of BOTH neighbouring slices: halo_pack(LGF_HALO_G) -> rank r-1 (as before) and
 * halo_pack(LGF_HALO_G_UP) = g of the slab's LAST slice -> rank r+1, each followed by halo_unpack with the same id
 * on the receiver; and the U_t halo of the current configuration, which must have been exchanged once
 * (halo_pack / halo_unpack(LGF_HALO_LINKS), e.g. by the first lgf_slab_delta round) after set_links or after an
 * lgf_slab_update -- LGF_ESTATE otherwise.  The sweep itself keeps that halo current from then on, so an iteration
 * of sweeps exchanges 24 reals per boundary site instead of 12 + 18 (or 12 + 12). */
int lgf_slab_sweep(lgf_slab *ctx, double *d_sums);
/* Algorithm 1's control on the device (lines 1, 2, 17), the slab twin of what lgf_iterate /
 * lgf_fix do inside: d_sums (device, 2 doubles) = the sums of lgf_slab_delta / lgf_slab_sweep AFTER the all-reduce
 * over the ranks.  Computes F = sums[0] / (12 V_global) (eq. 3) and theta = sums[1] / (3 V_global) (eq. 6) into the
 * context's device-resident state; record != 0: appends (F, theta) to the history and applies the loop test --
 * theta < tol, or a NaN / Inf theta, sets the `done` flag, after which every iteration kernel of this context
 * (FFT passes, g-build, update, sweep, the sum of the partial sums, finalize itself) returns at once, so iterations
 * enqueued past convergence cost nothing and the host needs no per-iteration read-back.  after_sweep != 0: the sums
 * come from lgf_slab_sweep -- the second link buffer becomes the current one and the update counter advances;
 * REQUIRED after every lgf_slab_sweep (the sweep itself flips nothing).  Every rank calls it with the same sums, so
 * every rank takes the same decision.  lgf_slab_delta always runs (it is a measurement). */
int lgf_slab_finalize(lgf_slab *ctx, const double *d_sums, double tol, int after_sweep, int record);
/* clears the `done` flag (start of a new iterate / fix) */
int lgf_slab_clear_done(lgf_slab *ctx);
/* lgf_slab_poll enqueues an asynchronous copy of the state into pinned host memory and returns at once (at most two
 * outstanding, LGF_ESTATE beyond); lgf_slab_poll_wait waits for the OLDEST outstanding one and reports what it saw
 * (any out-pointer may be NULL).  A driver that enqueues a chunk of iterations, polls, enqueues the next chunk and
 * only then waits for the first look never lets the GPU idle on the host. */
int lgf_slab_poll(lgf_slab *ctx);
int lgf_slab_poll_wait(lgf_slab *ctx, int *done, int *nan_seen, long long *n_updates, double *F, double *theta);
/* the recorded (F, theta) entries, as lgf_history / lgf_history_length; synchronise the stream */
long long lgf_slab_history_length(lgf_slab *ctx);
int lgf_slab_history(lgf_slab *ctx, long long first, long long count, double *F, double *theta);
/* the slab's work field as full 3 x 3 matrices, 18 reals per local site (as lgf_get_field) */
int lgf_slab_get_field(lgf_slab *ctx, void *d_field);
long long lgf_slab_launch_count(const lgf_slab *ctx);
const char *lgf_slab_last_error(const lgf_slab *ctx);

/* ---- a measurement that allocates nothing -------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it): F = sum Re tr U / (12 V) (eq. 3) and theta = sum tr(Delta Delta^dag) / (3 V) (eqs. 5-7, :63-76) of
 * a configuration given in the canonical layout (d_links: device, 72 reals per site, `precision` bytes per real),
 * written to d_F_theta[0], d_F_theta[1] (device, two doubles) asynchronously on `cuda_stream` -- no context, no
 * cudaMalloc / cudaFree, no allocating call.  The per-block partial sums live in ONE fixed device array inside the
 * library (128 KB, held by every GPU that loads it until exit), so the lattice is limited to LGF_STATIC_MAX_SITES
 * sites (32^4 and 32^3 x 64 fit; beyond: LGF_EINVAL, use lgf_create / lgf_measure).  Every call shares that array:
 * calls that overlap on the GPU (different streams or host threads) race on it -- serialise them.  Per-site terms in
 * the working precision, sums in fp64, fixed summation order (R14).  Errors: LGF_E* with the message from
 * lgf_static_last_error() (per host thread). */
#define LGF_STATIC_MAX_SITES 2097152
int lgf_measure_static(const int dims[4], int precision, const void *d_links, double *d_F_theta, void *cuda_stream);
const char *lgf_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LGF_H */
