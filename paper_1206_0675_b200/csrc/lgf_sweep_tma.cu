// lgf_sweep_tma.cu -- the fused a6 + a1 sweep (U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag, eq. 2 / Alg. 1 line 14, and
// Delta, F, theta of the NEW links, eqs. 3, 5-7 / line 17) as a persistent, warp-specialised kernel whose inputs
// arrive through a ring of shared-memory stages filled by the TMA engine -- one 2-D tensor copy
// (cp.async.bulk.tensor, SASS UTMALDG) per stage: box = the tile's sites x the planes of a link or of g -- and
// signalled by mbarriers.  Part of liblgf (CUDA path).  Shares nothing with oracle/.
//
// Why it exists, and what it measured (B200, 32^4; DESIGN.md section 6 has the table).  The register sweep k_sweep
// (lgf_links.cu) holds three 3 x 3 complex matrices per thread (168 registers in fp64, 12 warps per SM) and is
// latency-bound: a probe with the same access pattern and no arithmetic streams the sweep's bytes in 213 us at 64
// warps per SM but needs 256 us at 12 warps and 342 us once the neighbour re-reads go through the load pipe.  Here
// the bytes in flight live in shared memory instead of registers: one producer thread keeps the ring full while
// four compute warps work, every operand is read from shared memory, and a tile's x / y neighbours are served from
// the staged planes instead of being loaded again (4 + 1/R + 2 link transforms per site instead of 8).
// Result at 32^4 (sweep time, staged / register): fp64/18 269 / 283 us, fp64/12 212 / 227, fp32/12 114 / 134, but
// fp32/18 164 / 160; it loses at 64^4 and 24^3 x 48 (table at sweep_tma_auto) -- the context uses it where it won
// (lgf_tune "sweep_tma": -1 = that rule, 1 = wherever it applies, 0 = never).  What it took to get there, each step measured:
//   * 1-D bulk copies (one per plane, 105 per tile) cost the issuing warp 73 cycles each, whatever their size:
//     tensor maps (14 copies per tile) removed that bottleneck;
//   * the producer is ONE thread (about one instruction per five cycles): 64-bit index arithmetic and a byte-granular
//     ring allocator made it the bottleneck at 1500 cycles per stage -- 32-bit arithmetic, equal slots;
//   * a stage that is needed for several steps (the tile's g rows) pins everything behind it in an in-order ring:
//     it has a buffer and a barrier pair of its own;
//   * a slot is handed back as soon as its operands are in registers, not after the arithmetic -- and "in registers"
//     has to be enforced (see loaded_bits);
//   * fp64: setmaxnreg moves the idle producer warps' registers to the compute warps (no spills at 216 registers);
//     no warp may exit before the others once registers have been moved, and the idle warps may take their registers
//     back only after the compute warps have released them (named barrier; without it: a timing-dependent deadlock).
//
// Tile: R whole x lines of one (z, t) plane, NT = R Lx <= 128 consecutive sites, one compute thread per site.
// Per tile: a preamble (g of the tile, g of lines y0 - 1 and y0 + R, U_y of line y0 - 1) and ten ring stages, in the
// order they are consumed (NPL = 3 NR stored planes per link):
//    1 UX U_x    2 UY U_y    3 UZ U_z    4 g(x+z^)    5 U_z(x-z^)    6 g(x-z^)    7 UT U_t    8 g(x+t^)    9 U_t(x-t^)   10 g(x-t^)
// x: the backward neighbour's A'_x is handed over through shared memory (the whole periodic line is in the CTA);
// y: likewise for rows 1 .. R-1, recomputed from the staged line y0 - 1 for row 0; z, t: recomputed as in k_sweep.
// The halo policy SweepHalo serves the t-slab decomposition (lgf_slab.cu) as in k_sweep.
#include <new>

#include <cuda.h>          // CUtensorMap and the cuTensorMapEncodeTiled prototype (resolved at run time, not linked)

#include "lgf_pdl.cuh"
#include "lgf_state.cuh"
#include "lgf_tma.cuh"

namespace lgf {

constexpr int SWT_MAXSLOT = 8;

struct SweepTileCfg {
    int Lx, R, NT;          // tile: R rows of Lx sites, NT = R Lx compute threads
    int nyb;                // tiles per (x, y) plane = Ly / R
    int nslot;              // ring of equal slots, each the size of one link-plane set of a tile (size_u)
    int size_u, size_g;     // bytes of a tile's planes of one link / of g
    int row_u, row_g;       // bytes of one staged x line of all link planes / g planes, rounded up to 128
    int size_gt;            // the tile's preamble: g of the tile, g of lines y0 - 1 and y0 + R, U_y of line y0 - 1
    unsigned zero;          // always 0 (see loaded_bits)
    long long ntiles;
};
// ring position: slot index and the parity of the phase being waited for
struct RingPos {
    int slot, phase;
    __device__ __forceinline__ void next(int nslot) {
        if (++slot == nslot) { slot = 0; phase ^= 1; }
    }
};
// The tensor maps of one context: link buffers 0 / 1 and g, each as a 2-D tensor (2 V reals) x (planes) with a
// box of one tile (2 NT reals) or of one x line (2 Lx reals) by the planes of one link / of g.
struct alignas(64) SweepMaps {
    CUtensorMap u_body[2], u_row[2], g_body, g_row;
};

template <class R>
__device__ __forceinline__ void smem_load_g(const C<R> *p, int stride, C<R> (&gx)[9]) {
#pragma unroll
    for (int e = 0; e < 6; e++) gx[e] = p[e * stride];
    reconstruct_row2(gx);
}
template <int NR, class R>
__device__ __forceinline__ void smem_load_link(const C<R> *p, int stride, C<R> (&u)[9]) {
#pragma unroll
    for (int e = 0; e < 3 * NR; e++) u[e] = p[e * stride];
    if constexpr (NR == 2) reconstruct_row2(u);
}
// The values just read from a stage must have ARRIVED in registers before the stage is handed back to the copy
// engine.  Issuing the shared-memory loads is not enough: the arrive on the "empty" barrier does not queue behind
// them, and with eight warps bursting 16-byte loads the load pipe can be hundreds of cycles behind -- long enough
// for the producer to wake, issue the next tensor copy and have it land on data not yet read (new links that
// differed from run to run, only when producer and consumers were both fast).  So the arrive is made to DEPEND on
// the loaded registers: its count operand is 1 + (bits of every loaded value & zero), `zero` a kernel parameter
// the compiler cannot see through.
__device__ __forceinline__ unsigned loaded_bits(const C<double> (&m)[9], int n) {
    unsigned a = 0;
#pragma unroll
    for (int e = 0; e < 9; e++)
        if (e < n) a |= (unsigned)__double2loint(m[e].x) | (unsigned)__double2loint(m[e].y);
    return a;
}
__device__ __forceinline__ unsigned loaded_bits(const C<float> (&m)[9], int n) {
    unsigned a = 0;
#pragma unroll
    for (int e = 0; e < 9; e++)
        if (e < n) a |= __float_as_uint(m[e].x) | __float_as_uint(m[e].y);
    return a;
}
// packed A' (8 reals) <-> four complex slots
template <class R>
__device__ __forceinline__ void smem_put_herm(C<R> *p, int stride, const Herm<R> &a) {
    p[0] = a.m01; p[stride] = a.m02; p[2 * stride] = a.m12; p[3 * stride] = mk<R>(a.m00, a.m11);
}
template <class R>
__device__ __forceinline__ Herm<R> smem_get_herm(const C<R> *p, int stride) {
    Herm<R> a;
    a.m01 = p[0]; a.m02 = p[stride]; a.m12 = p[2 * stride];
    const C<R> d = p[3 * stride];
    a.m00 = d.x; a.m11 = d.y;
    return a;
}

// RSPLIT (fp64, tiles of 128 sites): the CTA is two warpgroups, the four compute warps and a producer group of which
// one thread works; setmaxnreg moves the producer group's registers to the compute warps (40 / 216 per thread
// instead of 128 each), which three 3 x 3 complex fp64 matrices plus the accumulators need to stay out of local
// memory (0.330 -> 0.280 ms at 32^4).
template <class R, int NR, bool REUNIT, bool RSPLIT>
__global__ void __launch_bounds__(RSPLIT ? 256 : 160, RSPLIT ? 2 : 0) __maxnreg__(RSPLIT ? 128 : (sizeof(R) == 8 ? 168 : 128))
    k_sweep_tma(const __grid_constant__ SweepMaps maps, LinkPair<R> lp, const C<R> *__restrict__ G, C<R> *__restrict__ W, Geom g,
                double *__restrict__ partial, const DevState *__restrict__ st, BlockOrder bo, SweepTileCfg tc, SweepHalo<R> halo) {
    pdl_enter();
    if (st->done) return;
    const int cur = st->cur;
    C<R> *__restrict__ dst = cur ? lp.buf[0] : lp.buf[1];
    constexpr int NPL = 3 * NR;
    constexpr unsigned E = sizeof(C<R>);
    extern __shared__ __align__(128) unsigned char smem[];
    const int NT = tc.NT, Lx = tc.Lx, RW = tc.R, nslot = tc.nslot;
    // shared memory: [ring: nslot x size_u][the tile's preamble][A'_x, A'_y of the tile: 2 x 4 x NT complex]
    // [barriers][scratch]
    unsigned char *gtbuf = smem + (size_t)nslot * tc.size_u;
    C<R> *sA = reinterpret_cast<C<R> *>(gtbuf + tc.size_gt);
    uint64_t *full = reinterpret_cast<uint64_t *>(gtbuf + tc.size_gt + (size_t)8 * NT * E);
    uint64_t *empty = full + SWT_MAXSLOT;
    uint64_t *gt_full = empty + SWT_MAXSLOT, *gt_empty = gt_full + 1;
    double *scratch = reinterpret_cast<double *>(gt_empty + 1);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ncw = NT >> 5;                                  // compute warps; warp ncw holds the producer thread
    if (tid == 0) {
        for (int i = 0; i < nslot; i++) { mbar_init(&full[i], 1); mbar_init(&empty[i], ncw); }
        mbar_init(gt_full, 1);
        mbar_init(gt_empty, ncw);
        mbar_init_fence();
    }
    __syncthreads();
    const int Lz = g.L[2];
    const long long V = g.V;
    if constexpr (RSPLIT) {
        if (warp >= ncw) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 216;");
    }
    if (warp >= ncw) {
        // ---- producer: ONE thread; a stage is one tensor copy.  32-bit arithmetic and straight-line code only.
        // (With the register split no warp may exit before the others -- warps that left right after giving up their
        // registers corrupted the compute warps' extra registers: everyone meets at the CTA's last barrier.)
        if (lane == 0 && warp == ncw) {
            const CUtensorMap *mu_body = &maps.u_body[cur], *mu_row = &maps.u_row[cur];
            const int Ly = g.L[1], Lt = g.L[3], S2 = (int)g.S[2], S3 = (int)g.S[3];
            const unsigned gbytes = 6u * NT * E, ubytes = (unsigned)NPL * NT * E;
            RingPos rp{0, 1};                                 // a fresh barrier lets the wait for parity 1 pass
            unsigned it = 0;
            for (long long k = blockIdx.x; k < tc.ntiles; k += gridDim.x, it++) {
                const unsigned tl = (unsigned)block_base(bo, (unsigned)k);
                const int yb = (int)(tl % (unsigned)tc.nyb);
                const unsigned r = tl / (unsigned)tc.nyb;
                const int cz = (int)(r % (unsigned)Lz), ct = (int)(r / (unsigned)Lz);
                const int s0 = (int)tl * NT, y0 = yb * RW, plane0 = s0 - y0 * Lx;
                const int szp = s0 + (cz == Lz - 1 ? -(Lz - 1) : 1) * S2, szm = s0 + (cz == 0 ? Lz - 1 : -1) * S2;
                const int stp = s0 + (ct == Lt - 1 ? -(Lt - 1) : 1) * S3, stm = s0 + (ct == 0 ? Lt - 1 : -1) * S3;
                const int rowm = plane0 + ((y0 == 0 ? Ly : y0) - 1) * Lx, rowp = plane0 + (y0 + RW == Ly ? 0 : y0 + RW) * Lx;
                // the preamble into its own buffer, once the consumers are done with the previous tile's
                mbar_wait(gt_empty, (it & 1) ^ 1);
                mbar_arrive_expect_tx(gt_full, (6u * (NT + 2 * Lx) + (unsigned)NPL * Lx) * E);
                tma_load_2d(gtbuf, &maps.g_body, 2 * s0, 0, gt_full);
                tma_load_2d(gtbuf + tc.size_g, &maps.g_row, 2 * rowm, 0, gt_full);
                tma_load_2d(gtbuf + tc.size_g + tc.row_g, &maps.g_row, 2 * rowp, 0, gt_full);
                tma_load_2d(gtbuf + tc.size_g + 2 * tc.row_g, mu_row, 2 * rowm, NPL, gt_full);
                auto stage_u = [&](int mu, int at) {          // the planes of link mu of the tile at site `at`
                    mbar_wait(&empty[rp.slot], rp.phase);
                    uint64_t *fb = &full[rp.slot];
                    mbar_arrive_expect_tx(fb, ubytes);
                    tma_load_2d(smem + (size_t)rp.slot * tc.size_u, mu_body, 2 * at, mu * NPL, fb);
                    rp.next(nslot);
                };
                auto stage_g = [&](int at) {
                    mbar_wait(&empty[rp.slot], rp.phase);
                    uint64_t *fb = &full[rp.slot];
                    mbar_arrive_expect_tx(fb, gbytes);
                    tma_load_2d(smem + (size_t)rp.slot * tc.size_u, &maps.g_body, 2 * at, 0, fb);
                    rp.next(nslot);
                };
                // across the ends of a t-slab g and U_t come from the neighbours' halo copies: plain 1-D bulk copies
                auto stage_halo = [&](const C<R> *hp, int np) {
                    mbar_wait(&empty[rp.slot], rp.phase);
                    uint64_t *fb = &full[rp.slot];
                    mbar_arrive_expect_tx(fb, (unsigned)np * NT * E);
                    for (int e = 0; e < np; e++)
                        bulk_g2s(smem + (size_t)rp.slot * tc.size_u + (size_t)e * NT * E, hp + (long long)e * S3, NT * E, fb);
                    rp.next(nslot);
                };
                stage_u(0, s0);                               // 1 UX
                stage_u(1, s0);                               // 2 UY
                stage_u(2, s0);                               // 3 UZ
                stage_g(szp);                                 // 4 g(x + z^)
                stage_u(2, szm);                              // 5 U_z(x - z^)
                stage_g(szm);                                 // 6 g(x - z^)
                stage_u(3, s0);                               // 7 UT
                if (halo.ghi && ct == Lt - 1) stage_halo(halo.ghi + (s0 - S3 * (Lt - 1)), 6);
                else stage_g(stp);                            // 8 g(x + t^)
                if (halo.uhalo && ct == 0) stage_halo(halo.uhalo + s0, NPL);
                else stage_u(3, stm);                         // 9 U_t(x - t^)
                if (halo.glo && ct == 0) stage_halo(halo.glo + s0, 6);
                else stage_g(stm);                            // 10 g(x - t^)
            }
        }
        if constexpr (!RSPLIT) return;
        // Back to the launch-time register count for the common tail -- but only AFTER the compute warps have given
        // their extra registers back (named barrier 3: they arrive after their setmaxnreg.dec, this group waits).
        // Without that order the three idle warps of this group, which get here at once, re-took the registers they
        // had just released before the compute warps could claim them, and the compute warps then spun in their
        // setmaxnreg.inc for ever: a timing-dependent hang (seen at 16^3 x 32 slabs and with the projecting variant).
        if constexpr (RSPLIT) {
            asm volatile("bar.sync 3, 256;" ::: "memory");
            asm volatile("setmaxnreg.inc.sync.aligned.u32 128;");
        }
    } else {
    // ---- consumers: one thread per site of the tile ---------------------------------------------------------
    RingPos rp{0, 0};
    const int x = tid % Lx, ry = tid / Lx;
    const int xp = x + 1 == Lx ? 0 : x + 1, xm = x == 0 ? Lx - 1 : x - 1;
    C<R> *sAx = sA, *sAy = sA + 4 * NT;
    const C<R> *stage;                                        // where the stage just acquired lives
    auto acquire = [&]() {                                    // wait for the next stage; returns its slot
        const int b = rp.slot;
        stage = reinterpret_cast<const C<R> *>(smem + (size_t)b * tc.size_u);
        mbar_wait(&full[b], rp.phase);
        rp.next(nslot);
        return b;
    };
    // The warp has its operands in registers (dep: see loaded_bits): hand the bytes back to the producer BEFORE the
    // arithmetic, so that a stage occupies the ring while it is in flight, not while it is being used.
    auto release = [&](int b, unsigned dep) {
        __syncwarp();
        if (lane == 0) mbar_arrive_count(&empty[b], 1u + (dep & tc.zero));
    };
    double f = 0.0, t = 0.0;
    unsigned it = 0;
    for (long long k = blockIdx.x; k < tc.ntiles; k += gridDim.x, it++) {
        const long long tl = block_base(bo, (unsigned)k);
        const int ct = (int)((tl / tc.nyb) / Lz);
        const long long s = tl * NT + tid;
        Herm<R> d = herm_zero<R>();
        R retr = 0;
        C<R> gx[9];
        // the site's own new link in direction mu: stored, - A'_mu(x) into d; returns A'_mu(x)
        auto own = [&](int mu, const C<R> (&u)[9], const C<R> (&gn)[9]) {
            C<R> p[9];
            transform_link<NR>(gx, u, gn, p);                 // Alg. 1 line 14, eq. 2
            if constexpr (REUNIT) project_su3(p);
            store_link<R, NR>(dst, V, mu, s, p);
            retr += p[0].x + p[4].x + p[8].x;                 // eq. 3 on the new link
            const Herm<R> a = algebra_part(p);
            herm_sub(d, a);                                   // - A'_mu(x)
            return a;
        };
        // + A'_mu(x - mu): the backward neighbour's new link recomputed
        auto bwd = [&](const C<R> (&u)[9], const C<R> (&gb)[9], C<R> (&p)[9]) {
            transform_link<NR>(gb, u, gx, p);
            if constexpr (REUNIT) project_su3(p);             // the same link the neighbour stores
            herm_add(d, algebra_part(p));                     // eq. 5
        };
        mbar_wait(gt_full, it & 1);
        const C<R> *gt = reinterpret_cast<const C<R> *>(gtbuf);                              // [6][NT] g of the tile
        const C<R> *gt_m = reinterpret_cast<const C<R> *>(gtbuf + tc.size_g);                // [6][Lx] g of line y0 - 1
        const C<R> *gt_p = reinterpret_cast<const C<R> *>(gtbuf + tc.size_g + tc.row_g);     // [6][Lx] g of line y0 + R
        const C<R> *uy_m = reinterpret_cast<const C<R> *>(gtbuf + tc.size_g + 2 * tc.row_g); // [NPL][Lx] U_y of line y0 - 1
        smem_load_g(gt + tid, NT, gx);
        {
            C<R> u[9], gn[9];
            const int bU = acquire();                         // 1 UX
            smem_load_link<NR>(stage + tid, NT, u);
            release(bU, loaded_bits(u, NPL));
            smem_load_g(gt + ry * Lx + xp, NT, gn);
            bar_sync_named(2, NT);                            // everyone has read the previous tile's A'_x, A'_y
            smem_put_herm(sAx + tid, NT, own(0, u, gn));
        }
        {
            const int bU = acquire();                         // 2 UY
            if (ry == 0) {                                    // line y0 - 1 belongs to another tile: its new link is recomputed
                C<R> ub[9], gb[9], p[9];
                smem_load_link<NR>(uy_m + x, Lx, ub);
                smem_load_g(gt_m + x, Lx, gb);
                bwd(ub, gb, p);
            }
            C<R> u[9], gn[9];
            smem_load_link<NR>(stage + tid, NT, u);
            if (ry + 1 < RW) smem_load_g(gt + tid + Lx, NT, gn);
            else smem_load_g(gt_p + x, Lx, gn);
            const unsigned dep = loaded_bits(u, NPL) | loaded_bits(gn, 6);
            release(bU, dep);
            if (lane == 0) mbar_arrive_count(gt_empty, 1u + (dep & tc.zero));      // the preamble is free too
            smem_put_herm(sAy + tid, NT, own(1, u, gn));
        }
        bar_sync_named(1, NT);                                // A'_x, A'_y of the whole tile are in place
        herm_add(d, smem_get_herm(sAx + ry * Lx + xm, NT));   // + A'_x(x - x^): the periodic line is inside the tile
        if (ry > 0) herm_add(d, smem_get_herm(sAy + tid - Lx, NT));         // + A'_y(x - y^)
#pragma unroll
        for (int mu = 2; mu < 4; mu++) {
            {
                C<R> u[9], gn[9];
                const int bU = acquire();                     // 3: U_z, 7: U_t
                smem_load_link<NR>(stage + tid, NT, u);
                release(bU, loaded_bits(u, NPL));
                const int bG = acquire();                     // 4: g(x + z^), 8: g(x + t^)
                smem_load_g(stage + tid, NT, gn);
                release(bG, loaded_bits(gn, 6));
                own(mu, u, gn);
            }
            {
                C<R> u[9], gb[9], p[9];
                const int bU = acquire();                     // 5: U_z(x - z^), 9: U_t(x - t^)
                smem_load_link<NR>(stage + tid, NT, u);
                release(bU, loaded_bits(u, NPL));
                const int bG = acquire();                     // 6: g(x - z^), 10: g(x - t^)
                smem_load_g(stage + tid, NT, gb);
                release(bG, loaded_bits(gb, 6));
                bwd(u, gb, p);
                // t-slab: the slice below lives on another rank; keep its halo copy of U_t current (lgf_slab.cu)
                if (mu == 3 && halo.uhalo && ct == 0) store_link<R, NR>(halo.uhalo, g.S[3], 0, s, p);
            }
        }
        store_herm(W, V, s, d);
        f += (double)retr;
        t += (double)herm_norm2(d);                           // eq. 6
    }
    // per-CTA partial sums in a fixed order (k_finalize adds the CTAs' sums, again in a fixed order)
    f = warp_sum(f);
    t = warp_sum(t);
    if (lane == 0) { scratch[2 * warp] = f; scratch[2 * warp + 1] = t; }
    bar_sync_named(1, NT);
    if (tid == 0) {
        double sf = 0.0, stt = 0.0;
        for (int w = 0; w < ncw; w++) { sf += scratch[2 * w]; stt += scratch[2 * w + 1]; }
        partial[2 * blockIdx.x] = sf;
        partial[2 * blockIdx.x + 1] = stt;
    }
    if constexpr (RSPLIT) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 128;");
        asm volatile("bar.arrive 3, 256;" ::: "memory");
    }
    }
    if constexpr (RSPLIT) __syncthreads();
}

// ---- configuration and launcher ---------------------------------------------------------------------------
static int num_sms() {
    static int n = 0;
    if (!n) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    }
    return n;
}
template <class R> constexpr int sweep_tma_minb() { return sizeof(R) == 8 ? 2 : 3; }

// Tile and ring for this lattice, or false if the staged sweep does not apply (x lines that are not a multiple of
// 16 bytes, no whole number of warps per tile, a ring of fewer than 3 slots): the caller then takes k_sweep.
static bool sweep_tma_config(const Geom &g, int nr, int prec, int minb, SweepTileCfg *out) {
    const int Lx = g.L[0], Ly = g.L[1], E = 2 * prec;
    if ((Lx * E) % 16 != 0 || 2 * g.V > 0x7fffffffLL) return false;
    int R = 0;
    for (int r = Ly; r >= 1; r--)
        if (Ly % r == 0 && r * Lx <= 128 && (r * Lx) % 32 == 0) { R = r; break; }
    if (!R) return false;
    SweepTileCfg tc;
    tc.Lx = Lx; tc.R = R; tc.NT = R * Lx; tc.nyb = Ly / R;
    tc.size_u = 3 * nr * tc.NT * E;                           // multiples of 128: NT is a multiple of 32
    tc.size_g = 6 * tc.NT * E;
    if (tc.size_g > tc.size_u) return false;
    tc.row_u = (3 * nr * Lx * E + 127) / 128 * 128;
    tc.row_g = (6 * Lx * E + 127) / 128 * 128;
    tc.size_gt = tc.size_g + 2 * tc.row_g + tc.row_u;
    // shared memory of one SM shared by `minb` CTAs (1 KB of each is the system's, 1 KB of slack for allocation
    // granularity); preamble buffer, A'_x, A'_y, barriers, scratch
    const int budget = 233472 / minb - 2048 - tc.size_gt - 8 * tc.NT * E - (2 * SWT_MAXSLOT + 2) * 8 - 64;
    tc.nslot = budget / tc.size_u;
    if (tc.nslot > SWT_MAXSLOT) tc.nslot = SWT_MAXSLOT;
    if (tc.nslot < 3) return false;
    tc.zero = 0;
    tc.ntiles = g.V / tc.NT;
    *out = tc;
    return true;
}
bool sweep_tma_supported(const Geom &g, int nr, int prec) {
    SweepTileCfg tc;
    return sweep_tma_config(g, nr, prec, prec == 8 ? 2 : 3, &tc);
}

// Where the staged sweep measured faster than k_sweep on B200 (sweep time in us, staged / register):
//   32^4    fp64/18 269 / 283   fp64/12 212 / 227   fp32/12 114 / 134   but fp32/18 164 / 160
//   64^4    fp32/12 1880 / 2038                      but fp64/18 5005 / 4464, fp64/12 3863 / 3738, fp32/18 2652 / 2457
//           (x lines of 64 sites: tiles of two lines, half of the y neighbours recomputed)
//   24^3 x 48 (tiles of 96 sites, no register split)  fp64/18 232 / 175, fp32/18 124 / 115;   16^4: equal
// i.e. tiles of 128 sites in at least 4 lines, except fp32 / 18-real; and fp32 / 12-real on any 128-site tile.
bool sweep_tma_auto(const Geom &g, int nr, int prec) {
    SweepTileCfg tc;
    if (!sweep_tma_config(g, nr, prec, prec == 8 ? 2 : 3, &tc) || tc.NT != 128) return false;
    if (prec == 4) return nr == 2;
    return tc.R >= 4;
}

// cuTensorMapEncodeTiled is a driver entry point; liblgf links only the runtime, so it is looked up at run time.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}
// (2 V reals) x (nplanes) tensor over a plane set, box = (2 box_sites reals) x (box_planes)
static bool encode_planes(CUtensorMap *m, void *base, int prec, long long V, int nplanes, int box_sites, int box_planes) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[2] = {(cuuint64_t)(2 * V), (cuuint64_t)nplanes};
    const cuuint64_t strides[1] = {(cuuint64_t)(2 * V) * (cuuint64_t)prec};
    const cuuint32_t box[2] = {(cuuint32_t)(2 * box_sites), (cuuint32_t)box_planes};
    const cuuint32_t es[2] = {1, 1};
    return fn(m, prec == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
              CU_TENSOR_MAP_L2_PROMOTION_L2_256B,             // (NONE / 64 B / 128 B / 256 B measured alike)
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
SweepMaps *sweep_tma_maps_create(const Geom &g, int nr, int prec, void *links0, void *links1, void *G) {
    SweepTileCfg tc;
    if (!sweep_tma_config(g, nr, prec, prec == 8 ? 2 : 3, &tc)) return nullptr;
    if (2 * tc.NT > 256) return nullptr;                      // box extents are limited to 256 elements
    SweepMaps *m = new (std::nothrow) SweepMaps();
    if (!m) return nullptr;
    void *lk[2] = {links0, links1};
    bool ok = true;
    for (int b = 0; b < 2 && ok; b++)
        ok = encode_planes(&m->u_body[b], lk[b], prec, g.V, 4 * 3 * nr, tc.NT, 3 * nr) &&
             encode_planes(&m->u_row[b], lk[b], prec, g.V, 4 * 3 * nr, tc.Lx, 3 * nr);
    ok = ok && encode_planes(&m->g_body, G, prec, g.V, 6, tc.NT, 6) && encode_planes(&m->g_row, G, prec, g.V, 6, tc.Lx, 6);
    if (!ok) { delete m; return nullptr; }
    return m;
}
void sweep_tma_maps_destroy(SweepMaps *m) { delete m; }
std::string sweep_tma_kernel_name(const Geom &g, int nr, int prec, bool reunit, bool rsplit) {
    SweepTileCfg tc;
    if (!sweep_tma_config(g, nr, prec, prec == 8 ? 2 : 3, &tc)) return "";
    char buf[96];
    snprintf(buf, sizeof buf, "k_sweep_tma<%s, %d, %d, %d>", prec == 8 ? "double" : "float", nr, reunit ? 1 : 0,
             (prec == 8 && tc.NT == 128 && rsplit) ? 1 : 0);
    return buf;
}

template <class R, int NR, bool REUNIT, bool RSPLIT>
static cudaError_t launch_sweep_tma_as(const SweepMaps &maps, LinkPair<R> links, const C<R> *G, C<R> *W, const Geom &g,
                                       double *partial, int *nblocks, const DevState *st, LaunchStream stream, const BlockOrder &bo,
                                       const SweepTileCfg &tc, const SweepHalo<R> &halo) {
    auto kern = k_sweep_tma<R, NR, REUNIT, RSPLIT>;
    const size_t smem = (size_t)tc.nslot * tc.size_u + tc.size_gt + (size_t)8 * tc.NT * sizeof(C<R>) +
                        (2 * SWT_MAXSLOT + 2) * sizeof(uint64_t) + 64;
    if (cudaError_t e = ensure_dynamic_smem(kern, smem); e != cudaSuccess) return e;
    long long nb = (long long)sweep_tma_minb<R>() * num_sms();
    if (nb > tc.ntiles) nb = tc.ntiles;
    *nblocks = (int)nb;
    return launch_pdl(kern, dim3((unsigned)nb), dim3(tc.NT + (RSPLIT ? 128 : 32)), smem, stream, maps, links, G, W, g, partial, st, bo,
                      tc, halo);
}

template <class R>
cudaError_t launch_sweep_tma(const SweepMaps *maps, int nr, LinkPair<R> links, const C<R> *G, C<R> *W, const Geom &g, double *partial,
                             int *nblocks, const DevState *st, LaunchStream stream, int order_tz, bool reunit, const SweepHalo<R> &halo,
                             bool rsplit) {
    SweepTileCfg tc;
    if (!maps || !sweep_tma_config(g, nr, (int)sizeof(R), sweep_tma_minb<R>(), &tc)) return cudaErrorInvalidValue;
    const BlockOrder bo = sweep_block_order(g, nr, (int)sizeof(R), order_tz, tc.NT);
    constexpr bool DBL = sizeof(R) == 8;
#define LGF_GO(NRV, RU)                                                                                                  \
    {                                                                                                                    \
        if (DBL && tc.NT == 128 && rsplit)                                                                               \
            return launch_sweep_tma_as<R, NRV, RU, DBL>(*maps, links, G, W, g, partial, nblocks, st, stream, bo, tc, halo); \
        return launch_sweep_tma_as<R, NRV, RU, false>(*maps, links, G, W, g, partial, nblocks, st, stream, bo, tc, halo); \
    }
    if (nr == 3) {
        if (reunit) LGF_GO(3, true)
        LGF_GO(3, false)
    }
    if (reunit) LGF_GO(2, true)
    LGF_GO(2, false)
#undef LGF_GO
}
template cudaError_t launch_sweep_tma<float>(const SweepMaps *, int, LinkPair<float>, const C<float> *, C<float> *, const Geom &, double *,
                                             int *, const DevState *, LaunchStream, int, bool, const SweepHalo<float> &, bool);
template cudaError_t launch_sweep_tma<double>(const SweepMaps *, int, LinkPair<double>, const C<double> *, C<double> *, const Geom &,
                                              double *, int *, const DevState *, LaunchStream, int, bool, const SweepHalo<double> &, bool);

}  // namespace lgf
