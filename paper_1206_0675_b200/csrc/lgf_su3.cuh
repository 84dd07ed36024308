// lgf_su3.cuh -- 3x3 complex matrices in registers: link load/store in the structure-of-arrays
// layout (18- or 12-real storage), the algebra part A_mu, packed hermitian-traceless fields and the
// Gram-Schmidt build of g(x).  Part of liblgf (CUDA path).  Shares nothing with oracle/.
//
// Internal link layout:  U[mu][e][s], e = 3*i + j over the stored rows
// (NR = 3 rows -> 9 complex planes per direction, NR = 2 rows -> 6), s = x + Lx*(y + Ly*(z + Lz*t)),
// each entry one interleaved complex number, so a warp reading one plane moves 32 consecutive
// 16-byte (fp64) or 8-byte (fp32) words.
//
// Packed hermitian traceless field (Delta and w; 8 reals per site instead of 18):
//   W[0][s] = M01, W[1][s] = M02, W[2][s] = M12 (complex), W[3][s] = (M00, M11) (two reals),
//   M22 = -M00 - M11, M10 = conj(M01), ...
#pragma once
#include "lgf_cplx.cuh"

namespace lgf {

// third row of an SU(3) matrix from the first two: c = (a x b)^*      (eq. 8)
template <class R>
__device__ __forceinline__ void reconstruct_row2(C<R> (&u)[9]) {
    u[6] = conj(u[1] * u[5] - u[2] * u[4]);
    u[7] = conj(u[2] * u[3] - u[0] * u[5]);
    u[8] = conj(u[0] * u[4] - u[1] * u[3]);
}

// Load link number mu of site s.  `links` is the base of the whole SoA array, V the plane length.
template <class R, int NR>
__device__ __forceinline__ void load_link(const C<R> *__restrict__ links, long long V, int mu, long long s,
                                          C<R> (&u)[9]) {
    const C<R> *p = links + (long long)mu * (3 * NR) * V + s;
#pragma unroll
    for (int e = 0; e < 3 * NR; e++) u[e] = p[(long long)e * V];
    if constexpr (NR == 2) reconstruct_row2(u);
}

template <class R, int NR>
__device__ __forceinline__ void store_link(C<R> *__restrict__ links, long long V, int mu, long long s,
                                           const C<R> (&u)[9]) {
    C<R> *p = links + (long long)mu * (3 * NR) * V + s;
#pragma unroll
    for (int e = 0; e < 3 * NR; e++) p[(long long)e * V] = u[e];
}

// Hermitian traceless 3x3 matrix in packed form: three complex off-diagonals and two real diagonals.
template <class R>
struct Herm {
    C<R> m01, m02, m12;
    R m00, m11;
};

template <class R>
__device__ __forceinline__ Herm<R> herm_zero() {
    Herm<R> h;
    h.m01 = h.m02 = h.m12 = mk<R>(0, 0);
    h.m00 = h.m11 = 0;
    return h;
}

// A = [(U - U^dag)/(2i)] - (1/3) tr[(U - U^dag)/(2i)] 1        (eq. 7 "- h.c. - trace")
//   off-diagonal: (U_ij - conj(U_ji))/(2i) = ( (Im U_ij + Im U_ji)/2 , -(Re U_ij - Re U_ji)/2 )
//   diagonal:     Im U_ii - (1/3) sum_k Im U_kk
template <class R>
__device__ __forceinline__ Herm<R> algebra_part(const C<R> (&u)[9]) {
    Herm<R> a;
    const R h = (R)0.5;
    a.m01 = mk<R>(h * (u[1].y + u[3].y), h * (u[3].x - u[1].x));
    a.m02 = mk<R>(h * (u[2].y + u[6].y), h * (u[6].x - u[2].x));
    a.m12 = mk<R>(h * (u[5].y + u[7].y), h * (u[7].x - u[5].x));
    const R tr3 = (u[0].y + u[4].y + u[8].y) * (R)(1.0 / 3.0);
    a.m00 = u[0].y - tr3;
    a.m11 = u[4].y - tr3;
    return a;
}

template <class R>
__device__ __forceinline__ void herm_add(Herm<R> &d, const Herm<R> &a) {
    d.m01 = d.m01 + a.m01; d.m02 = d.m02 + a.m02; d.m12 = d.m12 + a.m12;
    d.m00 += a.m00; d.m11 += a.m11;
}
template <class R>
__device__ __forceinline__ void herm_sub(Herm<R> &d, const Herm<R> &a) {
    d.m01 = d.m01 - a.m01; d.m02 = d.m02 - a.m02; d.m12 = d.m12 - a.m12;
    d.m00 -= a.m00; d.m11 -= a.m11;
}

// tr(M M^dag) = sum_ij |M_ij|^2 for a packed hermitian traceless M        (eq. 6)
template <class R>
__device__ __forceinline__ R herm_norm2(const Herm<R> &d) {
    const R m22 = -d.m00 - d.m11;
    return (R)2 * (norm2(d.m01) + norm2(d.m02) + norm2(d.m12)) + d.m00 * d.m00 + d.m11 * d.m11 + m22 * m22;
}

template <class R>
__device__ __forceinline__ Herm<R> load_herm(const C<R> *__restrict__ W, long long V, long long s) {
    Herm<R> h;
    h.m01 = W[s];
    h.m02 = W[V + s];
    h.m12 = W[2 * V + s];
    const C<R> d = W[3 * V + s];
    h.m00 = d.x;
    h.m11 = d.y;
    return h;
}
template <class R>
__device__ __forceinline__ void store_herm(C<R> *__restrict__ W, long long V, long long s, const Herm<R> &h) {
    W[s] = h.m01;
    W[V + s] = h.m02;
    W[2 * V + s] = h.m12;
    W[3 * V + s] = mk<R>(h.m00, h.m11);
}

// g = GS(1 + i*h*w): first-order expansion of exp[i (alpha/2) w] followed by the
// Gram-Schmidt projection on rows, third row from eq. 8 (reading R9).  h = alpha/2.
//   i*h*w_ij for hermitian w:  row 0 = (1 + i h w00, i h w01, i h w02),
//                              row 1 = (i h conj(w01), 1 + i h w11, i h w12)
template <class R>
__device__ __forceinline__ void build_g(const Herm<R> &w, R h, C<R> (&g)[9]) {
    C<R> a0 = mk<R>((R)1, h * w.m00), a1 = mk<R>(-h * w.m01.y, h * w.m01.x), a2 = mk<R>(-h * w.m02.y, h * w.m02.x);
    C<R> b0 = mk<R>(h * w.m01.y, h * w.m01.x), b1 = mk<R>((R)1, h * w.m11), b2 = mk<R>(-h * w.m12.y, h * w.m12.x);
    const R ia = inv_sqrt_pos(norm2(a0) + norm2(a1) + norm2(a2));
    a0 = ia * a0; a1 = ia * a1; a2 = ia * a2;
    // ab = sum_j conj(a_j) b_j ;  b -= ab * a
    C<R> ab = mk<R>(0, 0);
    ab = ab + mulc(b0, a0);
    ab = ab + mulc(b1, a1);
    ab = ab + mulc(b2, a2);
    b0 = b0 - ab * a0; b1 = b1 - ab * a1; b2 = b2 - ab * a2;
    const R ib = inv_sqrt_pos(norm2(b0) + norm2(b1) + norm2(b2));
    b0 = ib * b0; b1 = ib * b1; b2 = ib * b2;
    g[0] = a0; g[1] = a1; g[2] = a2;
    g[3] = b0; g[4] = b1; g[5] = b2;
    reconstruct_row2(g);
}

// out = a * b      (rows 0 .. NROWS-1 of the product only)
template <int NROWS, class R>
__device__ __forceinline__ void mat_mul(const C<R> (&a)[9], const C<R> (&b)[9], C<R> (&out)[9]) {
#pragma unroll
    for (int i = 0; i < NROWS; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            C<R> s = a[3 * i] * b[j];
            mad(s, a[3 * i + 1], b[3 + j]);
            mad(s, a[3 * i + 2], b[6 + j]);
            out[3 * i + j] = s;
        }
}
// out = a * b^dag  (rows 0 .. NROWS-1 of the product only)
template <int NROWS, class R>
__device__ __forceinline__ void mat_mul_dag(const C<R> (&a)[9], const C<R> (&b)[9], C<R> (&out)[9]) {
#pragma unroll
    for (int i = 0; i < NROWS; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            C<R> s = mulc(a[3 * i], b[3 * j]);
            madc(s, a[3 * i + 1], b[3 * j + 1]);
            madc(s, a[3 * i + 2], b[3 * j + 2]);
            out[3 * i + j] = s;
        }
}

// rows 0, 1 of g(x) are stored (G[e][s], e = 0..5); row 2 is (row0 x row1)^* by construction (eq. 8)
template <class R>
__device__ __forceinline__ void load_g(const C<R> *__restrict__ G, long long V, long long s, C<R> (&gx)[9]) {
#pragma unroll
    for (int e = 0; e < 6; e++) gx[e] = G[(long long)e * V + s];
    reconstruct_row2(gx);
}

// out = a * b * c^dag as it will be seen by whoever loads the stored link later: with 12-real storage
// only rows 0 and 1 are computed and row 2 is rebuilt from them (eq. 8), exactly as load_link does.
template <int NR, class R>
__device__ __forceinline__ void transform_link(const C<R> (&a)[9], const C<R> (&b)[9], const C<R> (&c)[9],
                                               C<R> (&out)[9]) {
    C<R> t[9];
    mat_mul<NR>(a, b, t);
    mat_mul_dag<NR>(t, c, out);
    if constexpr (NR == 2) reconstruct_row2(out);
}

// Opt-in (lgf_tune "reunit_every"): put a freshly transformed link back onto SU(3) -- Gram-Schmidt on rows 0, 1,
// row 2 = (row0 x row1)^* (eq. 8).  The method as the paper states it never does this (R13), and in
// fp64 it need not; in fp32 the links of a run of thousands of iterations drift far enough to move the
// gauge-invariant plaquette in the fourth digit.  Done inside the sweep, on every copy of the new link it
// computes, so Delta, F and theta stay those of the links that are stored and no extra pass is needed.
template <class R>
__device__ __forceinline__ void project_su3(C<R> (&u)[9]) {
    const R ia = (R)1 / sqrt(norm2(u[0]) + norm2(u[1]) + norm2(u[2]));
    u[0] = ia * u[0]; u[1] = ia * u[1]; u[2] = ia * u[2];
    C<R> ab = mulc(u[3], u[0]);
    ab = ab + mulc(u[4], u[1]);
    ab = ab + mulc(u[5], u[2]);
    u[3] = u[3] - ab * u[0]; u[4] = u[4] - ab * u[1]; u[5] = u[5] - ab * u[2];
    const R ib = (R)1 / sqrt(norm2(u[3]) + norm2(u[4]) + norm2(u[5]));
    u[3] = ib * u[3]; u[4] = ib * u[4]; u[5] = ib * u[5];
    reconstruct_row2(u);
}

// Order in which the CTAs of the sweep walk the lattice.  With the plain order (block b = sites
// 128 b .. 128 b + 127) the t-backward neighbour of a site was touched a whole t slice earlier: 43 MB of
// traffic at 32^3, 340 MB at 64^3 -- beyond L2, so U_t(x - t), g(x - t) and g(x) come from DRAM a second
// time (17 GB read instead of 11 at 64^4).  The tiled order walks (z, t) tiles of TZ z-planes: inside a
// tile t runs slower than z, so the t-neighbour is only TZ (x, y) planes of traffic away.
//   enumeration b' -> bxy = b' % nxy, zi = (b' / nxy) % TZ, t = (b' / (nxy TZ)) % Lt, ztile = b' / (nxy TZ Lt)
//   block base  = bxy + nxy * ((ztile TZ + zi) + Lz t)
struct BlockOrder {
    int nxy;      // CTAs per (x, y) plane; 0 = plain order
    int tz, Lz, Lt;
};
__device__ __forceinline__ long long block_base(const BlockOrder &bo, unsigned int b) {
    if (bo.nxy == 0) return b;
    const unsigned int bxy = b % bo.nxy; unsigned int r = b / bo.nxy;
    const unsigned int zi = r % bo.tz; r /= bo.tz;
    const unsigned int t = r % bo.Lt, ztile = r / bo.Lt;
    return (long long)bxy + (long long)bo.nxy * ((ztile * bo.tz + zi) + (long long)bo.Lz * t);
}

// ---- lattice geometry ----------------------------------------------------------------------------
struct Geom {
    int L[4];          // Lx, Ly, Lz, Lt
    long long S[4];    // strides 1, Lx, Lx*Ly, Lx*Ly*Lz
    long long V;
};

__device__ __forceinline__ void site_coords(const Geom &g, long long s, int (&c)[4]) {
    c[0] = (int)(s % g.L[0]); s /= g.L[0];
    c[1] = (int)(s % g.L[1]); s /= g.L[1];
    c[2] = (int)(s % g.L[2]);
    c[3] = (int)(s / g.L[2]);
}
// index of x - mu^ / x + mu^ (periodic)
__device__ __forceinline__ long long site_bwd(const Geom &g, long long s, const int (&c)[4], int mu) {
    return c[mu] == 0 ? s + (long long)(g.L[mu] - 1) * g.S[mu] : s - g.S[mu];
}
__device__ __forceinline__ long long site_fwd(const Geom &g, long long s, const int (&c)[4], int mu) {
    return c[mu] == g.L[mu] - 1 ? s - (long long)(g.L[mu] - 1) * g.S[mu] : s + g.S[mu];
}

// ---- block-wide sum of two doubles (warp shuffles, then one shared-memory hop) --------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// Every thread of the block must call this.  Result valid in thread 0.
__device__ __forceinline__ void block_sum2(double &a, double &b, double (*scratch)[2]) {
    a = warp_sum(a);
    b = warp_sum(b);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { scratch[wid][0] = a; scratch[wid][1] = b; }
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        a = lane < nw ? scratch[lane][0] : 0.0;
        b = lane < nw ? scratch[lane][1] : 0.0;
        a = warp_sum(a);
        b = warp_sum(b);
    }
}

}  // namespace lgf
