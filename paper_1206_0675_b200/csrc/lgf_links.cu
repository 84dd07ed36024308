// lgf_links.cu -- the link-side kernels of the gauge-fixing iteration:
//   k_delta     a1: A_mu, Delta(x), per-block partial sums for F and theta   (eqs. 3, 5-7; Alg. 1 line 1)
//   k_gbuild    a5: g(x) = GS(1 + i (alpha/2) w(x))                          (Alg. 1 line 10)
//   k_sweep     a6 + a1 fused: U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag (Alg. 1 line 14) and, in the same pass,
//               Delta, F, theta of the NEW configuration (Alg. 1 line 17) -- the links are read once
//               and written once per iteration
//   k_plaquette average plaquette partial sums (gauge-invariant check)
//   k_finalize  final fixed-order sum, F / theta normalisation, history, stop test (Alg. 1 line 2)
//   layout conversion canonical AoS <-> internal SoA, packed field <-> full 3x3 field
// Part of liblgf (CUDA path).  Shares nothing with oracle/.
#include <cstdio>
#include <string>

#include "lgf_state.cuh"
#include "lgf_pdl.cuh"

namespace lgf {

constexpr int SITE_THREADS = 256;
constexpr int SWEEP_THREADS = 128;

// ---- a1 -------------------------------------------------------------------------------------------
template <class R, int NR>
__global__ void __launch_bounds__(SITE_THREADS) k_delta(LinkPair<R> lp, C<R> *__restrict__ W, Geom g,
                                                         double *__restrict__ partial, const int *__restrict__ stop,
                                                         const DevState *__restrict__ st, SweepHalo<R> halo) {
    if (*stop) return;
    const C<R> *__restrict__ links = st->cur ? lp.buf[1] : lp.buf[0];
    __shared__ double scratch[SITE_THREADS / 32][2];
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
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
            // (t-slab: the slice below the slab lives on another rank; its U_t is in the halo copy, s < S3 there)
            if (mu == 3 && halo.uhalo && c[3] == 0) load_link<R, NR>(halo.uhalo, g.S[3], 0, s, u);
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

// ---- a5 -------------------------------------------------------------------------------------------
// g(x) from w(x); rows 0 and 1 are stored (G[e][s], e = 0..5), row 2 is (row0 x row1)^* by construction
// (eq. 8), so rebuilding it on load reproduces it exactly.
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_gbuild(const C<R> *__restrict__ W, C<R> *__restrict__ G, Geom g,
                                                          R half_alpha, const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    C<R> gx[9];
    build_g(load_herm(W, g.V, s), half_alpha, gx);
#pragma unroll
    for (int e = 0; e < 6; e++) G[(long long)e * g.V + s] = gx[e];
}

__device__ __forceinline__ void finalize_tail(double f, double t, long long V, double tol, int after_sweep, int record,
                                              DevState *st, double *__restrict__ hist, long long hist_cap) {
    const double F = f / (12.0 * (double)V);          // eq. 3: 1 / (4 N_c V)
    const double theta = t / (3.0 * (double)V);       // eq. 6: 1 / (N_c V)
    st->F = F;
    st->theta = theta;
    if (after_sweep) {                                // the sweep wrote the other buffer: make it current
        st->cur = 1 - st->cur;
        st->n_updates += 1;
    }
    if (record) {
        const long long n = st->n_hist;
        if (n < hist_cap) { hist[2 * n] = F; hist[2 * n + 1] = theta; }
        st->n_hist = n + 1;
        if (!(theta == theta) || theta > 1e300) { st->done = 1; st->nan = 1; }
        else if (theta < tol) st->done = 1;           // Alg. 1 line 2: loop while theta >= eps
    }
}

template <class R>
__device__ __forceinline__ void herm_to_smem(R *__restrict__ slot, int stride, const Herm<R> &a) {
    slot[0] = a.m01.x; slot[stride] = a.m01.y; slot[2 * stride] = a.m02.x; slot[3 * stride] = a.m02.y;
    slot[4 * stride] = a.m12.x; slot[5 * stride] = a.m12.y; slot[6 * stride] = a.m00; slot[7 * stride] = a.m11;
}
template <class R>
__device__ __forceinline__ Herm<R> herm_from_smem(const R *__restrict__ slot, int stride) {
    Herm<R> a;
    a.m01 = mk<R>(slot[0], slot[stride]);
    a.m02 = mk<R>(slot[2 * stride], slot[3 * stride]);
    a.m12 = mk<R>(slot[4 * stride], slot[5 * stride]);
    a.m00 = slot[6 * stride];
    a.m11 = slot[7 * stride];
    return a;
}

// ---- a6 + a1 fused --------------------------------------------------------------------------------
// One thread per site x.  For every direction: the site's own new link U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag
// is computed, stored to the other link buffer and its algebra part subtracted from Delta(x); the new
// link of the backward neighbour, U'_mu(x-mu) = g(x-mu) U_mu(x-mu) g(x)^dag, is recomputed (its inputs
// are L1/L2 hits: the neighbouring thread reads the same lines) and its algebra part added.  Reads
// buffer `cur`, writes buffer 1-cur (k_finalize flips `cur`), so no thread ever sees a half-updated
// neighbourhood (Jacobi update, R10).
// SHARE: a CTA's 128 consecutive sites are whole x lines when Lx divides 128 (four lines at 32^4), so the
// backward x neighbour of a site, and for most lines the backward y neighbour, belongs to the same CTA and has
// just computed the very A'_mu the site needs.  Those two are handed over through shared memory (one barrier
// per CTA, flat indexing) instead of being recomputed; neighbours outside the CTA, and z and t, are recomputed
// as before.  At 32^4: 6.25 link transforms per site instead of 8.
// The register allocation is asked to allow 3 CTAs per SM: 168 registers, no spills in fp64 / 18-real (2 would
// allow 255 registers at 8 warps per SM, 4 would force spills at 128).
constexpr int SWEEP_MINB = 3;
// L2 prefetch (sm_90+ bulk prefetch, SASS UBLKPF): one instruction asks the memory system to bring `bytes`
// contiguous bytes into L2; nothing is written to the SM, no register or shared memory is held.
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
template <class R, int NR, bool REUNIT, bool SHARE, int MINB>
__global__ void __launch_bounds__(SWEEP_THREADS, MINB)
    k_sweep(LinkPair<R> lp, const C<R> *__restrict__ G, C<R> *__restrict__ W, Geom g, double *__restrict__ partial,
            const DevState *__restrict__ st, BlockOrder bo, int ahead, SweepHalo<R> halo) {
    pdl_enter();
    if (st->done) return;
    const int cur = st->cur;
    // (a select between the two kernel parameters, not an indexed load of the parameter array: the pointers stay
    // in the global address space -- LDG / STG instead of generic LD / ST -- and the array is not copied to the stack)
    const C<R> *__restrict__ src = cur ? lp.buf[1] : lp.buf[0];
    C<R> *__restrict__ dst = cur ? lp.buf[0] : lp.buf[1];
    __shared__ double scratch[SWEEP_THREADS / 32][2];
    __shared__ R sA[SHARE ? 2 * 8 * SWEEP_THREADS : 1];          // A'_x, A'_y of the CTA's sites
    // The kernel is latency-bound (12 warps per SM, half of their time waiting on DRAM): the CTA that will run
    // `ahead` blocks later finds its own links and g(x) -- 4 * 3 NR + 6 planes of 128 consecutive sites -- in L2
    // already, because this CTA asks for them now: one bulk prefetch per plane, issued by the first threads.
    if (ahead > 0 && blockIdx.x + ahead < gridDim.x) {
        constexpr int NP = 4 * 3 * NR;
        const long long pb = block_base(bo, blockIdx.x + ahead) * SWEEP_THREADS;
        const long long left = g.V - pb;
        const unsigned bytes = (unsigned)((left < SWEEP_THREADS ? left : SWEEP_THREADS) * sizeof(C<R>));
        if (threadIdx.x < NP) prefetch_l2_bulk(src + (long long)threadIdx.x * g.V + pb, bytes);
        else if (threadIdx.x < NP + 6) prefetch_l2_bulk(G + (long long)(threadIdx.x - NP) * g.V + pb, bytes);
    }
    const long long base = block_base(bo, blockIdx.x) * SWEEP_THREADS;
    const long long s = base + threadIdx.x;
    const bool live = s < g.V;
    double f = 0.0, t = 0.0;
    int c[4] = {0, 0, 0, 0};
    C<R> gx[9];
    Herm<R> d = herm_zero<R>();
    R retr = 0;
    // the site's own new link in direction mu: transformed, stored, - A'_mu(x) into d; returns A'_mu(x)
    auto own = [&](int mu) {
        C<R> u[9], gn[9], p[9];
        load_link<R, NR>(src, g.V, mu, s, u);
        // (t-slab: g of the slice above the slab comes from the neighbour's halo copy)
        if (mu == 3 && halo.ghi && c[3] == g.L[3] - 1) load_g(halo.ghi, g.S[3], s - g.S[3] * (long long)(g.L[3] - 1), gn);
        else load_g(G, g.V, site_fwd(g, s, c, mu), gn);
        transform_link<NR>(gx, u, gn, p);                           // Alg. 1 line 14, eq. 2
        if constexpr (REUNIT) project_su3(p);
        store_link<R, NR>(dst, g.V, mu, s, p);
        retr += p[0].x + p[4].x + p[8].x;                           // eq. 3 on the new link
        const Herm<R> a = algebra_part(p);
        herm_sub(d, a);                                             // - A'_mu(x)
        return a;
    };
    // + A'_mu(x - mu): the backward neighbour's new link recomputed (its inputs are L1 / L2 hits)
    auto bwd = [&](int mu, long long sb) {
        C<R> u[9], gn[9], p[9];
        // (t-slab: the slice below lives on another rank -- its old U_t and its g are in the halo copies, and the
        // new U_t is stored back, so that the halo copy stays the neighbour's current link without another exchange)
        const bool below = mu == 3 && halo.uhalo && c[3] == 0;
        if (below) {
            load_link<R, NR>(halo.uhalo, g.S[3], 0, s, u);          // s < S3 here: the (x, y, z) index
            load_g(halo.glo, g.S[3], s, gn);
        } else {
            load_link<R, NR>(src, g.V, mu, sb, u);
            load_g(G, g.V, sb, gn);
        }
        transform_link<NR>(gn, u, gx, p);
        if constexpr (REUNIT) project_su3(p);                       // the same link the neighbour stores
        if (below) store_link<R, NR>(halo.uhalo, g.S[3], 0, s, p);
        herm_add(d, algebra_part(p));                               // eq. 5
    };
    if (live) {
        site_coords(g, s, c);
        load_g(G, g.V, s, gx);
    }
    if constexpr (!SHARE) {
        if (live) {
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {                        // own and backward link interleaved: the two
                own(mu);                                            // touch neighbouring cache lines
                bwd(mu, site_bwd(g, s, c, mu));
            }
        }
    } else {
        if (live) {
#pragma unroll
            for (int mu = 0; mu < 2; mu++)
                herm_to_smem(sA + mu * 8 * SWEEP_THREADS + threadIdx.x, SWEEP_THREADS, own(mu));
        }
        __syncthreads();
        if (live) {
#pragma unroll
            for (int mu = 0; mu < 4; mu++) {
                if (mu >= 2) own(mu);
                const long long sb = site_bwd(g, s, c, mu);
                const long long off = sb - base;
                if (mu < 2 && off >= 0 && off < SWEEP_THREADS)
                    herm_add(d, herm_from_smem(sA + mu * 8 * SWEEP_THREADS + (int)off, SWEEP_THREADS));
                else
                    bwd(mu, sb);
            }
        }
    }
    if (live) {
        store_herm(W, g.V, s, d);
        f = (double)retr;
        t = (double)herm_norm2(d);
    }
    // k_finalize closes the iteration in a launch of its own: folding it in here (release fence + ticket per
    // CTA, last CTA finalises) costs more than that launch, because the fence holds each of the 8192
    // short-lived CTAs until its link stores are acknowledged (measured 0.271 -> 0.317 ms at 32^4 fp64)
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) {
        partial[2 * blockIdx.x] = f;
        partial[2 * blockIdx.x + 1] = t;
    }
}

// ---- accumulated gauge transformation ------------------------------
// Gacc(x) <- g(x) Gacc(x): after n updates Gacc(x) = g_n(x) ... g_1(x), the transformation that takes the
// loaded configuration to the current one, U_mu(x) = Gacc(x) U0_mu(x) Gacc(x + mu)^dag (eq. 2, PAPER.md:45,
// composed).  Gacc is stored like a link plane set: Gacc[e][s], e = 0..8 (all three rows: products of
// many g drift off SU(3) by rounding, which eq. 8 would hide rather than carry).
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_gacc(const C<R> *__restrict__ G, C<R> *__restrict__ A, Geom g,
                                                        const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    C<R> gx[9], a[9], out[9];
    load_g(G, g.V, s, gx);
#pragma unroll
    for (int e = 0; e < 9; e++) a[e] = A[(long long)e * g.V + s];
    mat_mul<3>(gx, a, out);
#pragma unroll
    for (int e = 0; e < 9; e++) A[(long long)e * g.V + s] = out[e];
}
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_gacc_identity(C<R> *__restrict__ A, Geom g) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
#pragma unroll
    for (int e = 0; e < 9; e++) A[(long long)e * g.V + s] = mk<R>((e % 4 == 0) ? (R)1 : (R)0, (R)0);
}
// canonical transformation field in[s][i][j] -> rows 0, 1 of its projection onto SU(3) in the layout of G
// (lgf_apply_transform: the given matrices may be a float product converted to double, i.e. off SU(3) by 1e-7)
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_g_from_canonical(const R *__restrict__ in, C<R> *__restrict__ G, Geom g) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    const C<R> *src = reinterpret_cast<const C<R> *>(in) + s * 9;
    C<R> m[9];
#pragma unroll
    for (int e = 0; e < 9; e++) m[e] = src[e];
    project_su3(m);
#pragma unroll
    for (int e = 0; e < 6; e++) G[(long long)e * g.V + s] = m[e];
}
// canonical output: out[s][i][j] complex, 18 reals per site
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_gacc_get(const C<R> *__restrict__ A, R *__restrict__ out, Geom g) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    C<R> *dst = reinterpret_cast<C<R> *>(out) + s * 9;
#pragma unroll
    for (int e = 0; e < 9; e++) dst[e] = A[(long long)e * g.V + s];
}

// ---- gluon field in momentum space ---------------------------------
// k_algebra: W <- packed A_mu(x), the hermitian traceless algebra part of the links of ONE direction (eq. 7).
// k_gluon_unpack: after the forward transform of W (one pass per axis, lgf_fft.cu, which leaves position
// p = N2 k1 + k2 of a line holding frequency k = k1 + N1 k2), rebuild the full 3 x 3 matrix A_mu(k) in natural
// k order.  The packing put two REAL fields into W[3] = M00 + i M11 and kept only the upper off-diagonals, so
//   A01(k) = W0(k), A10(k) = conj(W0(-k))   (M10(x) = conj(M01(x)));  likewise 02 / 20 from W1, 12 / 21 from W2;
//   A00(k) = (W3(k) + conj(W3(-k))) / 2,  A11(k) = (W3(k) - conj(W3(-k))) / (2i),  A22 = -A00 - A11.
template <class R, int NR>
__global__ void __launch_bounds__(SITE_THREADS) k_algebra(LinkPair<R> lp, C<R> *__restrict__ W, Geom g, int mu,
                                                           const DevState *__restrict__ st) {
    const C<R> *__restrict__ links = lp.buf[st->cur];
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    C<R> u[9];
    load_link<R, NR>(links, g.V, mu, s, u);
    store_herm(W, g.V, s, algebra_part(u));
}
struct AxisPerm {
    int N1[4], N2[4];          // line factorisation of each axis (LineFactor<L>)
};
__device__ __forceinline__ long long kspace_pos(const Geom &g, const AxisPerm &pm, const int (&k)[4]) {
    long long p = 0;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) p += g.S[mu] * (long long)(pm.N2[mu] * (k[mu] % pm.N1[mu]) + k[mu] / pm.N1[mu]);
    return p;
}
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_gluon_unpack(const C<R> *__restrict__ W, R *__restrict__ out, Geom g,
                                                                AxisPerm pm) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;      // natural k index
    if (s >= g.V) return;
    int k[4], m[4];
    site_coords(g, s, k);
#pragma unroll
    for (int mu = 0; mu < 4; mu++) m[mu] = k[mu] == 0 ? 0 : g.L[mu] - k[mu];         // -k
    const long long pk = kspace_pos(g, pm, k), pm_k = kspace_pos(g, pm, m);
    const C<R> w0 = W[pk], w1 = W[g.V + pk], w2 = W[2 * g.V + pk], w3 = W[3 * g.V + pk];
    const C<R> c0 = conj(W[pm_k]), c1 = conj(W[g.V + pm_k]), c2 = conj(W[2 * g.V + pm_k]), c3 = conj(W[3 * g.V + pm_k]);
    const R h = (R)0.5;
    const C<R> a00 = h * (w3 + c3);
    const C<R> dif = h * (w3 - c3);
    const C<R> a11 = mk<R>(dif.y, -dif.x);                                            // dif / i
    C<R> *dst = reinterpret_cast<C<R> *>(out) + s * 9;
    dst[0] = a00; dst[1] = w0; dst[2] = w1;
    dst[3] = c0; dst[4] = a11; dst[5] = w2;
    dst[6] = c1; dst[7] = c2; dst[8] = mk<R>(-a00.x - a11.x, -a00.y - a11.y);
}

// ---- plaquette ------------------------------------------------------------------------------------
template <class R, int NR>
__global__ void __launch_bounds__(SITE_THREADS) k_plaquette(LinkPair<R> lp, Geom g, double *__restrict__ partial,
                                                             const DevState *__restrict__ st) {
    const C<R> *__restrict__ links = lp.buf[st->cur];
    __shared__ double scratch[SITE_THREADS / 32][2];
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    double p = 0.0, dummy = 0.0;
    if (s < g.V) {
        int c[4];
        site_coords(g, s, c);
        R acc = 0;
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                C<R> a[9], b[9], t1[9], t2[9];
                load_link<R, NR>(links, g.V, mu, s, a);
                load_link<R, NR>(links, g.V, nu, site_fwd(g, s, c, mu), b);
                mat_mul<3>(a, b, t1);                                   // U_mu(x) U_nu(x+mu)
                load_link<R, NR>(links, g.V, mu, site_fwd(g, s, c, nu), a);
                mat_mul_dag<3>(t1, a, t2);                              // ... U_mu(x+nu)^dag
                load_link<R, NR>(links, g.V, nu, s, b);
                // Re tr(t2 b^dag) = sum_ij Re(t2_ij conj(b_ij))
#pragma unroll
                for (int e = 0; e < 9; e++) acc += t2[e].x * b[e].x + t2[e].y * b[e].y;
            }
        p = (double)acc;
    }
    block_sum2(p, dummy, scratch);
    if (threadIdx.x == 0) partial[blockIdx.x] = p;
}

// ---- reductions' last stage -----------------------------------------------------------------------
// One block; fixed summation order (thread i takes partials i, i+1024, ...), so F and theta are
// bit-reproducible from run to run.
__global__ void __launch_bounds__(1024) k_finalize(const double *__restrict__ partial, int nblocks, long long V,
                                                    double tol, int after_sweep, int record, DevState *st,
                                                    double *__restrict__ hist, long long hist_cap) {
    pdl_enter();
    if ((record || after_sweep) && st->done) return;      // the kernels before this one did not run
    __shared__ double scratch[32][2];
    double f = 0.0, t = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += 1024) {
        f += partial[2 * i];
        t += partial[2 * i + 1];
    }
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) finalize_tail(f, t, V, tol, after_sweep, record, st, hist, hist_cap);
}

__global__ void __launch_bounds__(1024) k_sum1(const double *__restrict__ partial, int nblocks, double norm,
                                                double *out) {
    __shared__ double scratch[32][2];
    double f = 0.0, t = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += 1024) f += partial[i];
    block_sum2(f, t, scratch);
    if (threadIdx.x == 0) *out = f * norm;
}

__global__ void k_reset_state(DevState *st) {
    st->n_hist = 0; st->n_updates = 0; st->done = 0; st->nan = 0; st->F = 0.0; st->theta = 0.0; st->zero = 0;
    st->cur = 0;
}
__global__ void k_clear_done(DevState *st) { st->done = 0; }

// ---- layout conversion ----------------------------------------------------------------------------
// canonical: canon[((s*4 + mu)*9 + e)*2 + re/im]      (include/lgf.h)
// `canon` holds the n sites s0 .. s0 + n - 1 (a chunk of the configuration, or all of it)
template <class R, int NR>
__global__ void __launch_bounds__(SITE_THREADS) k_convert_in(const R *__restrict__ canon, C<R> *__restrict__ links,
                                                              Geom g, long long s0, long long n) {
    const long long i = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (i >= n) return;
    const long long s = s0 + i;
    const C<R> *src = reinterpret_cast<const C<R> *>(canon) + i * 36;
#pragma unroll
    for (int mu = 0; mu < 4; mu++)
#pragma unroll
        for (int e = 0; e < 3 * NR; e++) links[((long long)mu * (3 * NR) + e) * g.V + s] = src[mu * 9 + e];
}
template <class R, int NR>
__global__ void __launch_bounds__(SITE_THREADS) k_convert_out(LinkPair<R> lp, R *__restrict__ canon, Geom g,
                                                               const DevState *__restrict__ st, long long s0, long long n) {
    const C<R> *__restrict__ links = st->cur ? lp.buf[1] : lp.buf[0];
    const long long i = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (i >= n) return;
    const long long s = s0 + i;
    C<R> *dst = reinterpret_cast<C<R> *>(canon) + i * 36;
#pragma unroll
    for (int mu = 0; mu < 4; mu++) {
        C<R> u[9];
        load_link<R, NR>(links, g.V, mu, s, u);
#pragma unroll
        for (int e = 0; e < 9; e++) dst[mu * 9 + e] = u[e];
    }
}

// packed hermitian traceless field <-> full 3x3 field  field[(s*9 + e)*2 + re/im]
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_field_get(const C<R> *__restrict__ W, R *__restrict__ field, Geom g) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    const Herm<R> h = load_herm(W, g.V, s);
    C<R> *dst = reinterpret_cast<C<R> *>(field) + s * 9;
    dst[0] = mk<R>(h.m00, 0); dst[1] = h.m01; dst[2] = h.m02;
    dst[3] = conj(h.m01); dst[4] = mk<R>(h.m11, 0); dst[5] = h.m12;
    dst[6] = conj(h.m02); dst[7] = conj(h.m12); dst[8] = mk<R>(-h.m00 - h.m11, 0);
}
template <class R>
__global__ void __launch_bounds__(SITE_THREADS) k_field_set(C<R> *__restrict__ W, const R *__restrict__ field, Geom g) {
    const long long s = (long long)blockIdx.x * SITE_THREADS + threadIdx.x;
    if (s >= g.V) return;
    const C<R> *m = reinterpret_cast<const C<R> *>(field) + s * 9;
    // hermitian traceless part of m: (m + m^dag)/2 - tr/3
    Herm<R> h;
    const R hf = (R)0.5;
    h.m01 = hf * (m[1] + conj(m[3]));
    h.m02 = hf * (m[2] + conj(m[6]));
    h.m12 = hf * (m[5] + conj(m[7]));
    const R tr3 = (m[0].x + m[4].x + m[8].x) * (R)(1.0 / 3.0);
    h.m00 = m[0].x - tr3;
    h.m11 = m[4].x - tr3;
    store_herm(W, g.V, s, h);
}

// ---- launchers ------------------------------------------------------------------------------------
static inline int site_blocks(const Geom &g) { return (int)((g.V + SITE_THREADS - 1) / SITE_THREADS); }

template <class R>
cudaError_t launch_delta(int nr, LinkPair<R> links, C<R> *W, const Geom &g, double *partial, int *nblocks,
                         const int *stop, const DevState *st, LaunchStream stream, const SweepHalo<R> &halo) {
    const int nb = site_blocks(g);
    *nblocks = nb;
    if (nr == 3) k_delta<R, 3><<<nb, SITE_THREADS, 0, stream>>>(links, W, g, partial, stop, st, halo);
    else k_delta<R, 2><<<nb, SITE_THREADS, 0, stream>>>(links, W, g, partial, stop, st, halo);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_gbuild(const C<R> *W, C<R> *G, const Geom &g, R half_alpha, const DevState *st, LaunchStream stream) {
    return launch_pdl(k_gbuild<R>, dim3(site_blocks(g)), dim3(SITE_THREADS), 0, stream, W, G, g, half_alpha, st);
}
// one t slice of sweep traffic against L2 (the t-backward neighbours are that far behind in the plain order)
static bool sweep_slice_beyond_l2(const Geom &g, int nr, int prec) {
    const long long plane = (long long)g.L[0] * g.L[1];
    return (double)plane * (8.0 * 6.0 * nr + 28.0) * prec * g.L[2] > 64.0e6;
}
// A'_x, A'_y through shared memory (SHARE): automatic where it measured faster on B200 -- 18-real storage,
// x lines that divide the CTA, and fp32 (32^4: 0.1718 -> 0.1601 ms; 64^4: 2.61 -> 2.42 ms) or a lattice beyond
// L2 (64^4 fp64: 4.42 -> 4.26 ms); neutral within 1.5 % otherwise, +1.7 % at 24^3 x 48.
bool sweep_uses_share(const Geom &g, int nr, int prec, int share_mode) {
    return share_mode >= 0 ? share_mode != 0
                           : (nr == 3 && SWEEP_THREADS % g.L[0] == 0 && (prec == 4 || sweep_slice_beyond_l2(g, nr, prec)));
}
// Resident CTAs per SM the sweep is compiled for (its register cap).  minb = 0: automatic -- 3 (168 registers) in fp64;
// in fp32, where a thread's loads carry half the bytes and the sweep is short of bytes in flight, 5 (96 registers) for
// the SHARE variant and 4 (128 registers) for the plain one, once the grid fills them.  Measured on B200, iteration
// time at 3 / 4 / 5 CTAs: 32^4 fp32/18 (SHARE) 0.2029 / 0.2018 / 0.1964 ms; 24^3 x 48 fp32/18 (plain) 0.1590 / 0.1484 /
// 0.1583 ms (at 96 registers the plain variant spills); 64^4 fp32/18 3.57 -> 3.48 ms at 5; 16^4 (512 CTAs) 0.0208 ->
// 0.0210 ms at 5, so small lattices keep 3; 6 CTAs (80 registers, spills) lost everywhere.  The SU(3)-projecting
// variant (REUNIT) exists for 3 only.
int sweep_minb_of(const Geom &g, int prec, bool reunit, bool share, int minb) {
    if (reunit) return SWEEP_MINB;
    if (minb == 2) return 2;
    if (prec != 4) return SWEEP_MINB;
    if (minb == 4 || minb == 5) return minb;
    const long long nb = (g.V + SWEEP_THREADS - 1) / SWEEP_THREADS;
    if (minb <= 0 && share && nb >= 5 * 148) return 5;
    if (minb <= 0 && !share && nb >= 4 * 148) return 4;
    return SWEEP_MINB;
}
// the instantiation launch_sweep picks, as a profiler prints it (bench.py matches ncu captures against it)
std::string sweep_kernel_name(const Geom &g, int nr, int prec, bool reunit, int share_mode, int minb) {
    char buf[96];
    const bool share = sweep_uses_share(g, nr, prec, share_mode);
    snprintf(buf, sizeof buf, "k_sweep<%s, %d, %d, %d, %d>", prec == 8 ? "double" : "float", nr, reunit ? 1 : 0, share ? 1 : 0,
             sweep_minb_of(g, prec, reunit, share, minb));
    return buf;
}
// (z, t)-tiled block order when the (x, y) plane is a whole number of CTAs of `nt` sites; TZ: about 24 MB of traffic
// (1.3 kB per site in fp64 / 18-real) between a site and its t-neighbour
BlockOrder sweep_block_order(const Geom &g, int nr, int prec, int order_tz, int nt) {
    BlockOrder bo{0, 1, g.L[2], g.L[3]};
    const long long plane = (long long)g.L[0] * g.L[1];
    if (order_tz != 1 && plane % nt == 0) {
        int tz = order_tz;
        if (tz <= 0) {
            // automatic: only when one t slice of traffic does not fit in L2 (measured on B200: neutral at
            // 32^4 where it fits, -4 % sweep time at 64^4 where it does not)
            const double per_plane = (double)plane * (8.0 * 6.0 * nr + 28.0) * prec;
            tz = 1;
            if (sweep_slice_beyond_l2(g, nr, prec))
                while (tz * 2 <= g.L[2] && g.L[2] % (tz * 2) == 0 && per_plane * tz * 2 <= 24.0e6) tz *= 2;
        }
        if (tz > 1 && g.L[2] % tz == 0) { bo.nxy = (int)(plane / nt); bo.tz = tz; }
    }
    return bo;
}
template <class R>
cudaError_t launch_sweep(int nr, LinkPair<R> links, const C<R> *G, C<R> *W, const Geom &g, double *partial,
                         int *nblocks, const DevState *st, LaunchStream stream, int order_tz, bool reunit, int share_mode,
                         int ahead, int minb, const SweepHalo<R> &halo) {
    const int nb = (int)((g.V + SWEEP_THREADS - 1) / SWEEP_THREADS);
    *nblocks = nb;
    const BlockOrder bo = sweep_block_order(g, nr, (int)sizeof(R), order_tz, SWEEP_THREADS);
    const bool share = sweep_uses_share(g, nr, (int)sizeof(R), share_mode);
#define LGF_SWK(RU, SH, MB)                                                                              \
    if (nr == 3) return launch_pdl(k_sweep<R, 3, RU, SH, MB>, dim3(nb), dim3(SWEEP_THREADS), 0, stream, links, G, W, g, partial, st, bo, ahead, halo); \
    else return launch_pdl(k_sweep<R, 2, RU, SH, MB>, dim3(nb), dim3(SWEEP_THREADS), 0, stream, links, G, W, g, partial, st, bo, ahead, halo);
    const int mb = sweep_minb_of(g, (int)sizeof(R), reunit, share, minb);
    if constexpr (sizeof(R) == 4) {
        if (mb == 5) {
            if (share) { LGF_SWK(false, true, 5) }
            else { LGF_SWK(false, false, 5) }
        }
        if (mb == 4) {
            if (share) { LGF_SWK(false, true, 4) }
            else { LGF_SWK(false, false, 4) }
        }
    }
    if (mb == 2) {
        if (share) { LGF_SWK(false, true, 2) }
        else { LGF_SWK(false, false, 2) }
    }
    if (reunit && share) { LGF_SWK(true, true, SWEEP_MINB) }
    else if (reunit) { LGF_SWK(true, false, SWEEP_MINB) }
    else if (share) { LGF_SWK(false, true, SWEEP_MINB) }
    else { LGF_SWK(false, false, SWEEP_MINB) }
#undef LGF_SWK
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_plaquette(int nr, LinkPair<R> links, const Geom &g, double *partial, int *nblocks,
                             const DevState *st, LaunchStream stream) {
    const int nb = site_blocks(g);
    *nblocks = nb;
    if (nr == 3) k_plaquette<R, 3><<<nb, SITE_THREADS, 0, stream>>>(links, g, partial, st);
    else k_plaquette<R, 2><<<nb, SITE_THREADS, 0, stream>>>(links, g, partial, st);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_convert_in(int nr, const R *canon, C<R> *links0, const Geom &g, LaunchStream stream, long long s0, long long n) {
    if (n < 0) n = g.V - s0;
    const int nb = (int)((n + SITE_THREADS - 1) / SITE_THREADS);
    if (nr == 3) k_convert_in<R, 3><<<nb, SITE_THREADS, 0, stream>>>(canon, links0, g, s0, n);
    else k_convert_in<R, 2><<<nb, SITE_THREADS, 0, stream>>>(canon, links0, g, s0, n);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_convert_out(int nr, LinkPair<R> links, R *canon, const Geom &g, const DevState *st,
                               LaunchStream stream, long long s0, long long n) {
    if (n < 0) n = g.V - s0;
    const int nb = (int)((n + SITE_THREADS - 1) / SITE_THREADS);
    if (nr == 3) k_convert_out<R, 3><<<nb, SITE_THREADS, 0, stream>>>(links, canon, g, st, s0, n);
    else k_convert_out<R, 2><<<nb, SITE_THREADS, 0, stream>>>(links, canon, g, st, s0, n);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_gacc(int op, const C<R> *G, C<R> *A, R *out, const Geom &g, const DevState *st, LaunchStream stream) {
    const int nb = site_blocks(g);
    if (op == 3) k_g_from_canonical<R><<<nb, SITE_THREADS, 0, stream>>>(out, A, g);      // out = input field, A = G
    else if (op == 0) k_gacc_identity<R><<<nb, SITE_THREADS, 0, stream>>>(A, g);
    else if (op == 1) return launch_pdl(k_gacc<R>, dim3(nb), dim3(SITE_THREADS), 0, stream, G, A, g, st);
    else k_gacc_get<R><<<nb, SITE_THREADS, 0, stream>>>(A, out, g);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_algebra(int nr, LinkPair<R> links, C<R> *W, const Geom &g, int mu, const DevState *st, LaunchStream stream) {
    const int nb = site_blocks(g);
    if (nr == 3) k_algebra<R, 3><<<nb, SITE_THREADS, 0, stream>>>(links, W, g, mu, st);
    else k_algebra<R, 2><<<nb, SITE_THREADS, 0, stream>>>(links, W, g, mu, st);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_gluon_unpack(const C<R> *W, R *out, const Geom &g, const int N1[4], const int N2[4], LaunchStream stream) {
    AxisPerm pm;
    for (int mu = 0; mu < 4; mu++) { pm.N1[mu] = N1[mu]; pm.N2[mu] = N2[mu]; }
    k_gluon_unpack<R><<<site_blocks(g), SITE_THREADS, 0, stream>>>(W, out, g, pm);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_field_get(const C<R> *W, R *field, const Geom &g, LaunchStream stream) {
    k_field_get<R><<<site_blocks(g), SITE_THREADS, 0, stream>>>(W, field, g);
    return cudaGetLastError();
}
template <class R>
cudaError_t launch_field_set(C<R> *W, const R *field, const Geom &g, LaunchStream stream) {
    k_field_set<R><<<site_blocks(g), SITE_THREADS, 0, stream>>>(W, field, g);
    return cudaGetLastError();
}

cudaError_t launch_finalize(const double *partial, int nblocks, long long V, double tol, int after_sweep, int record,
                            DevState *st, double *hist, long long hist_cap, LaunchStream stream) {
    return launch_pdl(k_finalize, dim3(1), dim3(1024), 0, stream, partial, nblocks, V, tol, after_sweep, record, st, hist,
                      hist_cap);
}
cudaError_t launch_sum1(const double *partial, int nblocks, double norm, double *out, LaunchStream stream) {
    k_sum1<<<1, 1024, 0, stream>>>(partial, nblocks, norm, out);
    return cudaGetLastError();
}
cudaError_t launch_reset_state(DevState *st, LaunchStream stream) {
    k_reset_state<<<1, 1, 0, stream>>>(st);
    return cudaGetLastError();
}
cudaError_t launch_clear_done(DevState *st, LaunchStream stream) {
    k_clear_done<<<1, 1, 0, stream>>>(st);
    return cudaGetLastError();
}

#define LGF_INST(R)                                                                                                   \
    template cudaError_t launch_delta<R>(int, LinkPair<R>, C<R> *, const Geom &, double *, int *, const int *,        \
                                         const DevState *, LaunchStream, const SweepHalo<R> &);                       \
    template cudaError_t launch_gbuild<R>(const C<R> *, C<R> *, const Geom &, R, const DevState *, LaunchStream);     \
    template cudaError_t launch_sweep<R>(int, LinkPair<R>, const C<R> *, C<R> *, const Geom &, double *, int *,       \
                                         const DevState *, LaunchStream, int, bool, int, int, int, const SweepHalo<R> &);                                   \
    template cudaError_t launch_plaquette<R>(int, LinkPair<R>, const Geom &, double *, int *, const DevState *,       \
                                             LaunchStream);                                                           \
    template cudaError_t launch_convert_in<R>(int, const R *, C<R> *, const Geom &, LaunchStream, long long, long long); \
    template cudaError_t launch_convert_out<R>(int, LinkPair<R>, R *, const Geom &, const DevState *, LaunchStream, long long, long long); \
    template cudaError_t launch_gacc<R>(int, const C<R> *, C<R> *, R *, const Geom &, const DevState *, LaunchStream); \
    template cudaError_t launch_algebra<R>(int, LinkPair<R>, C<R> *, const Geom &, int, const DevState *, LaunchStream); \
    template cudaError_t launch_gluon_unpack<R>(const C<R> *, R *, const Geom &, const int[4], const int[4], LaunchStream); \
    template cudaError_t launch_field_get<R>(const C<R> *, R *, const Geom &, LaunchStream);                          \
    template cudaError_t launch_field_set<R>(C<R> *, const R *, const Geom &, LaunchStream);
LGF_INST(float)
LGF_INST(double)

}  // namespace lgf
