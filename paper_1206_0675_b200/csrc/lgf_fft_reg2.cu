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

// ---- inverse (x, y) sweep ending in the g-build with ONE plane per CTA (64-point planes) ----------------------
// 64^4 fp64: a plane is 64 KB, so a CTA holds one component of one (z, t) slice and a5 -- which needs all of w(x) --
// used to be a separate pass over the field (k_gbuild: 1.07 GB read + 1.6 GB written, 0.39 ms of a 6.5 ms iteration,
// and the sweep before it wrote w only for that pass to read it back).  Here the four CTAs that hold the four
// components of a slice form a THREAD-BLOCK CLUSTER: each transforms its plane (brought on chip by one bulk copy),
// the cluster synchronises, and every CTA builds g for a quarter of the slice's sites, reading the other three
// components out of its neighbours' shared memory (distributed shared memory, ld.shared::cluster: 3 x 16 KB per CTA and
// plane).  w is never written; rows 0, 1 of g go straight to G.
template <class R, int L>
__global__ void __cluster_dims__(4, 1, 1) __launch_bounds__(2 * L, 3)
    k_fftr2_xy_gcluster(C<R> *__restrict__ W, const DevState *__restrict__ st, C<R> *__restrict__ G, long long V, int nzt, R half_alpha) {
    pdl_enter();
    if (st->done) return;                                    // (the same decision in all four CTAs of a cluster)
    constexpr int M = L / 2;
    constexpr int PX = L | 1;
    constexpr unsigned PLANE_BYTES = L * L * sizeof(C<R>);
    using S = SplitDft<L, PAIR_MASK, R>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C<R> *tile = reinterpret_cast<C<R> *>(smem_raw);
    __shared__ uint64_t bar;
    const int tid = threadIdx.x;
    const int h = (tid >> 4) & 1;
    const int i = (tid >> 5) * 16 + (tid & 15);
    const unsigned c = cluster_ctarank();                    // packed component = rank in the cluster
    const long long slice = blockIdx.x / 4;
    if (tid == 0) {
        mbar_init(&bar, 1);
        mbar_init_fence();
        mbar_arrive_expect_tx(&bar, PLANE_BYTES);
        bulk_g2s(tile, W + ((long long)c * nzt + slice) * (L * L), PLANE_BYTES, &bar);
    }
    __syncthreads();
    mbar_wait(&bar, 0);
    C<R> v[M];
#pragma unroll
    for (int j = 0; j < M; j++) v[j] = tile[(2 * j + h) * L + i];            // kx = 2 j + h at ky = i (dense plane)
    __syncthreads();
    S::inverse(v, h);
#pragma unroll
    for (int m = 0; m < M; m++) tile[i * PX + m + M * h] = v[m];             // tile[ky][x]
    __syncthreads();
#pragma unroll
    for (int j = 0; j < M; j++) v[j] = tile[(2 * j + h) * PX + i];           // column x = i, ky = 2 j + h
    S::inverse(v, h);
    __syncthreads();
#pragma unroll
    for (int m = 0; m < M; m++) tile[(m + M * h) * PX + i] = v[m];           // tile[y][x] of this component
    cluster_sync_all();                                                      // all four components are in place
    const uint32_t t0 = smem_u32(tile);
    uint32_t tk[4];
#pragma unroll
    for (int k = 0; k < 4; k++) tk[k] = dsmem_map(t0, k);
    const long long s0 = slice * (L * L);
    const int sub = (int)c * 2 + h;                                          // 0 .. 7: this thread's rows y = sub + 8 mm
#pragma unroll 2
    for (int mm = 0; mm < L / 8; mm++) {
        const int y = sub + 8 * mm;
        const uint32_t off = (uint32_t)((y * PX + i) * sizeof(C<R>));
        Herm<R> w;
        dsmem_ld(tk[0] + off, w.m01.x, w.m01.y);
        dsmem_ld(tk[1] + off, w.m02.x, w.m02.y);
        dsmem_ld(tk[2] + off, w.m12.x, w.m12.y);
        dsmem_ld(tk[3] + off, w.m00, w.m11);
        C<R> gx[9];
        build_g(w, half_alpha, gx);
        const long long s = s0 + y * L + i;
#pragma unroll
        for (int e = 0; e < 6; e++) G[(long long)e * V + s] = gx[e];
    }
    // nobody leaves while its tile is being read.  The loads above have returned (the G stores used their values), so
    // the arrival needs no fence -- a releasing one would wait for those stores to reach memory
    cluster_arrive_relaxed();
    cluster_wait();
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
    static constexpr int MINB = (LZ <= 32 && LT <= 32 && SMEM <= 110 * 1024) ? (sizeof(R) == 8 ? 2 : 3) : 0;
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

// ---- (z, t) tile split over a thread-block cluster ----------------------------------------------------
// 64 x 64 fp64: the tile of XC = 2 consecutive (kx, ky) indices is 128 KB, so k_fftr2_zt runs ONE CTA of 256 threads per
// SM and its load, transform and store phases cannot overlap with anything (ncu at 64^4: 0.99 ms for 2.09 GB,
// fp64 pipe 32 % busy, DRAM 33 %).  Here NC CTAs of a cluster share the tile: CTA q holds the z lines of t in
// [q Lt / NC, (q + 1) Lt / NC) and, for the t lines, the rows kz in [q Lz / NC, (q + 1) Lz / NC) -- a 1 / NC part
// either way, 64 KB + padding, so three CTAs of different clusters are resident per SM and their phases overlap.
// The transposition z lines <-> t lines crosses the cluster through distributed shared memory: after the forward z
// transform a thread stores its kz values into the tile of the CTA that owns them (st.shared::cluster), and before
// the inverse z transform it loads them from there (ld.shared::cluster); the t-line round trip (forward, scale,
// inverse) is local.  Element (xc, kz_local, t) of a CTA's part at t PITCH + kz_local XC + xc.
template <class R, int LZ, int XC, int NC>
struct Zt2ClusterShape {
    static constexpr int PHASE = 128 / (int)sizeof(C<R>);
    static constexpr int ROW = XC * LZ / NC;                                  // t-line lines of one CTA = elements per t
    static constexpr int PITCH = ROW + ((XC < PHASE && ROW % PHASE == 0) ? XC : 0);
    static constexpr int THREADS = 2 * ROW;
    static constexpr size_t SMEM = sizeof(C<R>) * (size_t)PITCH * LZ;         // (Lt = Lz)
    static constexpr int MINB = sizeof(R) == 8 ? 3 : 2;
    static_assert(ROW % 16 == 0 && (LZ / 2) % NC == 0, "16 lines per warp; whole kz ranges per thread half");
};

template <class R, int LZ, int XC, int NC>
__global__ void __cluster_dims__(NC, 1, 1)
    __launch_bounds__((Zt2ClusterShape<R, LZ, XC, NC>::THREADS), (Zt2ClusterShape<R, LZ, XC, NC>::MINB))
        k_fftr2_zt_cluster(C<R> *__restrict__ W, Geom g, const R *__restrict__ p2tab, R scale, const DevState *__restrict__ st) {
    pdl_enter();
    if (st->done) return;                                    // (the same decision in every CTA of a cluster)
    cluster_arrive();                                        // "I have started": waited for before the first remote store
    using Sh = Zt2ClusterShape<R, LZ, XC, NC>;
    constexpr int PITCH = Sh::PITCH, M = LZ / 2, LQ = LZ / NC;
    using S = SplitDft<LZ, PAIR_MASK, R>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C<R> *tile = reinterpret_cast<C<R> *>(smem_raw);
    const long long plane = g.S[2];
    const int q = (int)cluster_ctarank();
    const int lo0 = (blockIdx.x / NC) * XC;
    C<R> *Wc = W + (long long)blockIdx.y * g.V + lo0;
    const int tid = threadIdx.x;
    const int h = (tid >> 4) & 1;
    const int l = (tid >> 5) * 16 + (tid & 15);               // line number within this CTA's part
    const int xc = l % XC, r = l / XC;                        // z lines: t = q LQ + r;  t lines: kz = q LQ + r
    const int t = q * LQ + r;
    // shared::cluster address of (xc, kz = 2 j + h, t) in the part that owns kz -- part (2 j + h) / LQ = 2 j / LQ (LQ is
    // even), at kz_local = (2 j) % LQ + h: a per-part base for this thread plus a compile-time offset
    uint32_t tk[NC];
#pragma unroll
    for (int k = 0; k < NC; k++) tk[k] = dsmem_map(smem_u32(tile), k) + (uint32_t)((t * PITCH + h * XC + xc) * sizeof(C<R>));
    auto addr_of = [&](int j) { return tk[(2 * j) / LQ] + (uint32_t)(((2 * j) % LQ) * XC * sizeof(C<R>)); };

    C<R> v[M];
    C<R> *col = Wc + xc + plane * ((long long)LZ * t);
#pragma unroll
    for (int m = 0; m < M; m++) v[m] = col[plane * (m + M * h)];
    S::forward(v, h);                                         // -> kz = 2 j + h
    cluster_wait();                                           // every CTA of the cluster is resident
#pragma unroll
    for (int j = 0; j < M; j++) dsmem_st(addr_of(j), v[j].x, v[j].y);
    cluster_sync_all();                                       // the parts are complete
    {                                                         // t line at (xc, kz = q LQ + r): forward, scale, inverse
#pragma unroll
        for (int m = 0; m < M; m++) v[m] = tile[(m + M * h) * PITCH + l];
        S::forward(v, h);                                     // -> kt = 2 j + h
        const int lo = lo0 + xc, kx = lo / g.L[1], ky = lo % g.L[1];
        const R p2xyz = p2tab[kx] + p2tab[64 + ky] + p2tab[128 + t];       // (kz = q LQ + r, the same number as t)
#pragma unroll
        for (int j = 0; j < M; j++) {
            const R p2 = p2xyz + p2tab[192 + 2 * j + h];
            const R f = (p2 == (R)0) ? (R)0 : div_pos(scale, p2);     // Alg. 1 lines 5, 7; zero mode -> 0 (R6)
            v[j] = f * v[j];
        }
        S::inverse(v, h);                                     // -> t = m + M h
#pragma unroll
        for (int m = 0; m < M; m++) tile[(m + M * h) * PITCH + l] = v[m];
    }
    cluster_sync_all();
#pragma unroll
    for (int j = 0; j < M; j++) dsmem_ld(addr_of(j), v[j].x, v[j].y);
    S::inverse(v, h);                                         // -> z = m + M h   (the loads have landed: their values are used)
    cluster_arrive();                                         // "I no longer read anyone's part"
#pragma unroll
    for (int m = 0; m < M; m++) col[plane * (m + M * h)] = v[m];
    cluster_wait();                                           // nobody leaves while its part may still be read
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
template <> struct Xy2Cfg<float, 64> { static constexpr int P = 4, PF = 1; };    // (PF = 4: one CTA of 512 threads per SM; forward sweep at 64^4, ncu: 282 -> 160 us with 1)
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
    return fft_reg2_supported(g);                            // (64-point fp64 planes: by a 4-CTA cluster, k_fftr2_xy_gcluster)
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
    else {                                                   // one plane per CTA: the four components of a slice as a cluster
        constexpr size_t SM = sizeof(C<R>) * L * (L | 1);
        auto kern = k_fftr2_xy_gcluster<R, L>;
        if (cudaError_t e = ensure_dynamic_smem(kern, SM); e != cudaSuccess) return e;
        return launch_pdl(kern, dim3((unsigned)(4LL * g.L[2] * g.L[3])), dim3(2 * L), SM, stream, W, st, G, g.V, g.L[2] * g.L[3],
                          half_alpha);
    }
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

// the cluster-split (z, t) sweep: 64 x 64 (z, t) planes, NC = 2 or 4 CTAs per tile of XC = NC (fp64) / 2 NC (fp32)
// consecutive (kx, ky) indices -- 32 / 64 contiguous bytes per line element either way
template <class R, int NC> struct Zt2ClusterCfg { static constexpr int XC = (sizeof(R) == 8 ? 1 : 2) * NC; };
bool fft_reg2_zt_cluster_supported(const Geom &g, int nc) {
    return fft_reg2_supported(g) && g.L[2] == 64 && g.L[3] == 64 && (nc == 2 || nc == 4) && g.S[2] % 8 == 0;
}
template <class R, int NC>
static cudaError_t launch_zt2_cluster(const Geom &g, C<R> *W, const R *p2tab, R scale, const DevState *st, LaunchStream stream) {
    constexpr int XC = Zt2ClusterCfg<R, NC>::XC;
    using Sh = Zt2ClusterShape<R, 64, XC, NC>;
    auto kern = k_fftr2_zt_cluster<R, 64, XC, NC>;
    if (cudaError_t e = ensure_dynamic_smem(kern, Sh::SMEM); e != cudaSuccess) return e;
    dim3 grid((unsigned)(g.S[2] / XC * NC), 4);
    return launch_pdl(kern, grid, dim3(Sh::THREADS), Sh::SMEM, stream, W, g, p2tab, scale, st);
}

// which: 0 = (x, y) forward, 1 = (z, t) forward + scale + inverse, 2 = (x, y) inverse, 3 = (x, y) inverse + g
template <class R>
cudaError_t launch_fft_reg2(int which, const Geom &g, C<R> *W, const R *p2tab, R scale, const DevState *st,
                            LaunchStream stream, C<R> *G, R half_alpha, bool bulk, int comp, int zt_cluster) {
    t_xy_bulk = bulk;
    t_xy_comp = comp;
    if (which == 1) {
        if (zt_cluster > 0) {
            if (!fft_reg2_zt_cluster_supported(g, zt_cluster)) return cudaErrorInvalidValue;
            return zt_cluster == 2 ? launch_zt2_cluster<R, 2>(g, W, p2tab, scale, st, stream)
                                   : launch_zt2_cluster<R, 4>(g, W, p2tab, scale, st, stream);
        }
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
static std::string reg2_name(int which, const Geom &g, int zt_cluster) {
    const char *rn = sizeof(R) == 8 ? "double" : "float";
    char buf[96] = "";
    if (which == 1) {
        if (zt_cluster > 0) {
            snprintf(buf, sizeof buf, "k_fftr2_zt_cluster<%s, 64, %d, %d>", rn, (sizeof(R) == 8 ? 1 : 2) * zt_cluster, zt_cluster);
            return buf;
        }
#define LGF_GO(A, B) if (g.L[2] == A && g.L[3] == B) snprintf(buf, sizeof buf, "k_fftr2_zt<%s, %d, %d, %d>", rn, A, B, Zt2Cfg<R, A, B>::XC);
        LGF_REG2_ZT(LGF_GO)
#undef LGF_GO
        return buf;
    }
#define LGF_GO(LEN)                                                                                           \
    if (g.L[0] == LEN) {                                                                                       \
        if (which == 0) snprintf(buf, sizeof buf, "k_fftr2_xy<%s, %d, 0, %d, 0>", rn, LEN, Xy2Cfg<R, LEN>::PF);  \
        else if (which == 3 && Xy2Cfg<R, LEN>::P % 4 != 0) snprintf(buf, sizeof buf, "k_fftr2_xy_gcluster<%s, %d>", rn, LEN); \
        else snprintf(buf, sizeof buf, "k_fftr2_xy<%s, %d, 1, %d, %d>", rn, LEN, Xy2Cfg<R, LEN>::P, which == 3 ? 1 : 0); \
    }
    LGF_REG2_LEN(LGF_GO)
#undef LGF_GO
    return buf;
}
std::string fft_reg2_kernel_name(int which, const Geom &g, int prec, bool bulk, int zt_cluster) {
    std::string s = prec == 8 ? reg2_name<double>(which, g, zt_cluster) : reg2_name<float>(which, g, zt_cluster);
    if (bulk && which != 1 && s.size() > 10 && s.compare(0, 11, "k_fftr2_xy<") == 0) s.insert(10, "_bulk");      // k_fftr2_xy -> k_fftr2_xy_bulk
    return s;
}

template cudaError_t launch_fft_reg2<float>(int, const Geom &, C<float> *, const float *, float, const DevState *,
                                            LaunchStream, C<float> *, float, bool, int, int);
template cudaError_t launch_fft_reg2<double>(int, const Geom &, C<double> *, const double *, double, const DevState *,
                                             LaunchStream, C<double> *, double, bool, int, int);

}  // namespace lgf
