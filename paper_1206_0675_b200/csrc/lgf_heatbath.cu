// lgf_heatbath.cu -- thermalisation of the internal configuration with the Wilson action: Cabibbo-Marinari
// pseudo-heat-bath over the three SU(2) subgroups, Creutz / Kennedy-Pendleton sampling, checkerboard order
// (the producer of the paper's kind of input; the paper
// names no algorithm -- DESIGN.md readings R24-R27 fix this one).  Part of liblgf (CUDA path); shares nothing
// with oracle/: the uniform generator below is this side's own implementation of the written specification.
//
//   S = beta sum_p [1 - Re tr U_p / 3];  staple sum A_mu(x) = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
//       + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ]                                              (R24)
//   one launch per class (mu, parity): one thread per link (x, mu) with (x0+x1+x2+x3) mod 2 = parity; its
//   staples only contain links of other classes, so the update is done in place                      (R25)
//   W = U A; for (i, j) = (0,1), (0,2), (1,2): quaternion r of the 2x2 block of W, kk = |r|,
//   X ~ exp(a x0) sqrt(1 - x0^2), a = 2 beta kk / 3; alpha = X (r/kk)^dag; U <- E(alpha) U, W <- E(alpha) W  (R26)
//   then U is re-projected onto SU(3) (Gram-Schmidt rows 0, 1; row 2 = (row0 x row1)^*): without it the norm
//   error of rows 0, 1 grows exponentially over the sweeps in 12-real storage (overflow before 300 sweeps)  (R26)
//   overrelaxation (OVERRELAX): alpha = (V^dag)^2 instead of the draw -- alpha V = V^dag has the same x0 as V, the
//   action is unchanged by every step; no random numbers                                                    (R28)
//   uniforms u_n = ((mix64(key + (idx+1) G) >> 11) + 0.5) 2^-53, idx = ((((class V + site) 3 + k) 32 + t) 6 + n) (R27)
// The arithmetic is double precision whatever the storage precision of the links.
#include "lgf_state.cuh"
#include "lgf_pdl.cuh"

namespace lgf {

constexpr int HB_THREADS = 128;
constexpr int HB_MAXATT = 32;

using Z = C<double>;

__device__ __forceinline__ unsigned long long hb_mix64(unsigned long long z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__device__ __forceinline__ double hb_uniform(unsigned long long key, unsigned long long idx) {
    const unsigned long long z = hb_mix64(key + (idx + 1ULL) * 0x9E3779B97F4A7C15ULL);
    return ((double)(z >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

template <class R, int NR>
__device__ __forceinline__ void load_link_d(const C<R> *__restrict__ links, long long V, int mu, long long s, Z (&u)[9]) {
    C<R> t[9];
    load_link<R, NR>(links, V, mu, s, t);
#pragma unroll
    for (int e = 0; e < 9; e++) u[e] = mk<double>((double)t[e].x, (double)t[e].y);
}

// out = op(a) op(b) with compile-time dagger flags
template <bool DA, bool DB>
__device__ __forceinline__ void mm(const Z (&a)[9], const Z (&b)[9], Z (&out)[9]) {
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            Z s = mk<double>(0.0, 0.0);
#pragma unroll
            for (int k = 0; k < 3; k++) {
                const Z x = DA ? conj(a[3 * k + i]) : a[3 * i + k];
                const Z y = DB ? conj(b[3 * j + k]) : b[3 * k + j];
                mad(s, x, y);
            }
            out[3 * i + j] = s;
        }
}

__device__ __forceinline__ long long shifted(const Geom &g, const int (&c)[4], int mu, int d1, int nu, int d2) {
    int q[4] = {c[0], c[1], c[2], c[3]};
    q[mu] += d1;
    if (q[mu] < 0) q[mu] += g.L[mu]; else if (q[mu] >= g.L[mu]) q[mu] -= g.L[mu];
    q[nu] += d2;
    if (q[nu] < 0) q[nu] += g.L[nu]; else if (q[nu] >= g.L[nu]) q[nu] -= g.L[nu];
    return q[0] + g.S[1] * q[1] + g.S[2] * q[2] + g.S[3] * q[3];
}

// x0 = 1 - delta with density exp(a x0) sqrt(1 - x0^2): Creutz below a = 2, Kennedy-Pendleton above (R26)
__device__ __forceinline__ void hb_sample(double a, unsigned long long key, unsigned long long base, double (&x)[4]) {
    const double TWO_PI = 2.0 * 3.14159265358979323846264338327950288;
    double delta = 0.0;
    int t;
    for (t = 0; t < HB_MAXATT; t++) {
        const unsigned long long b = base + 6ULL * t;
        const double u0 = hb_uniform(key, b), u3 = hb_uniform(key, b + 3);
        if (a >= 2.0) {
            const double u1 = hb_uniform(key, b + 1), u2 = hb_uniform(key, b + 2);
            const double c = cos(TWO_PI * u1);
            delta = -(log(u0) + c * c * log(u2)) / a;
            if (u3 * u3 <= 1.0 - 0.5 * delta) break;
        } else {
            delta = -log(u0 + (1.0 - u0) * exp(-2.0 * a)) / a;
            const double x0 = 1.0 - delta;
            if (u3 * u3 <= 1.0 - x0 * x0) break;
        }
    }
    if (t == HB_MAXATT) {
        t = HB_MAXATT - 1;
        delta = fmin(fmax(delta, 0.0), 2.0);
    }
    const double u4 = hb_uniform(key, base + 6ULL * t + 4), u5 = hb_uniform(key, base + 6ULL * t + 5);
    const double x0 = 1.0 - delta;
    double rr = 1.0 - x0 * x0;
    rr = rr > 0.0 ? sqrt(rr) : 0.0;
    const double ct = 2.0 * u4 - 1.0;
    double st = 1.0 - ct * ct;
    st = st > 0.0 ? sqrt(st) : 0.0;
    const double phi = TWO_PI * u5;
    x[0] = x0;
    x[1] = rr * st * cos(phi);
    x[2] = rr * st * sin(phi);
    x[3] = rr * ct;
}

// One class (mu, parity) of one sweep.  class_id = sweep * 8 + mu * 2 + parity selects the random stream.
template <class R, int NR, bool OVERRELAX>
__global__ void __launch_bounds__(HB_THREADS) k_heatbath(LinkPair<R> lp, Geom g, const DevState *__restrict__ st,
                                                         double beta, unsigned long long key,
                                                         unsigned long long class_id, int mu, int parity, int tz) {
    pdl_enter();                                        // the eight class passes of a sweep are chained (lgf_pdl.cuh)
    C<R> *links = lp.buf[st->cur];                      // updated in place (no __restrict__: read and written)
    const long long h = (long long)blockIdx.x * HB_THREADS + threadIdx.x;
    if (h >= g.V / 2) return;
    // the h-th site of this parity: x = 2 xh + ((y + z + t + parity) & 1)   (all extents are even).  The threads
    // walk the lattice in (z, t) tiles of tz z-planes (inside a tile t runs slower than z), so that the staples'
    // t-neighbours are tz (x, y) planes of traffic away instead of a whole t slice (beyond L2 at 64^3); tz = Lz is
    // the plain order.  Which thread owns which site has no influence on the result.
    const int hx = g.L[0] / 2;
    int c[4];
    long long r = h / hx;
    c[1] = (int)(r % g.L[1]); r /= g.L[1];
    const int zi = (int)(r % tz); r /= tz;
    c[3] = (int)(r % g.L[3]);
    c[2] = (int)(r / g.L[3]) * tz + zi;
    c[0] = 2 * (int)(h % hx) + ((c[1] + c[2] + c[3] + parity) & 1);
    const long long s = c[0] + g.S[1] * c[1] + g.S[2] * c[2] + g.S[3] * c[3];

    Z A[9];
#pragma unroll
    for (int e = 0; e < 9; e++) A[e] = mk<double>(0.0, 0.0);
    const long long s_mu = shifted(g, c, mu, +1, mu, 0);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        Z a[9], b[9], t[9], p[9];
        // upper staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
        load_link_d<R, NR>(links, g.V, nu, s_mu, a);
        load_link_d<R, NR>(links, g.V, mu, shifted(g, c, nu, +1, nu, 0), b);
        mm<false, true>(a, b, t);
        load_link_d<R, NR>(links, g.V, nu, s, a);
        mm<false, true>(t, a, p);
#pragma unroll
        for (int e = 0; e < 9; e++) A[e] = A[e] + p[e];
        // lower staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu)
        const long long s_mnu = shifted(g, c, nu, -1, nu, 0);
        load_link_d<R, NR>(links, g.V, nu, shifted(g, c, mu, +1, nu, -1), a);
        load_link_d<R, NR>(links, g.V, mu, s_mnu, b);
        mm<true, true>(a, b, t);
        load_link_d<R, NR>(links, g.V, nu, s_mnu, a);
        mm<false, false>(t, a, p);
#pragma unroll
        for (int e = 0; e < 9; e++) A[e] = A[e] + p[e];
    }

    Z U[9], W[9];
    load_link_d<R, NR>(links, g.V, mu, s, U);
    mm<false, false>(U, A, W);
    const unsigned long long link_idx = class_id * (unsigned long long)g.V + (unsigned long long)s;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const int i = (k == 2) ? 1 : 0, j = (k == 0) ? 1 : 2;
        const Z a = W[3 * i + i], b = W[3 * i + j], cc = W[3 * j + i], d = W[3 * j + j];
        const double r0 = 0.5 * (a.x + d.x), r1 = 0.5 * (b.y + cc.y), r2 = 0.5 * (b.x - cc.x), r3 = 0.5 * (a.y - d.y);
        const double kk = sqrt(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3);
        if (!(kk > 1e-300)) continue;
        // alpha = X V^dag, V^dag = (r0, -r) / kk
        const double q0 = r0 / kk, q1 = -r1 / kk, q2 = -r2 / kk, q3 = -r3 / kk;
        double x[4];
        if constexpr (OVERRELAX) { x[0] = q0; x[1] = q1; x[2] = q2; x[3] = q3; }       // X = V^dag
        else hb_sample(2.0 * beta * kk / 3.0, key, ((link_idx * 3ULL + (unsigned long long)k) * HB_MAXATT) * 6ULL, x);
        const double al0 = x[0] * q0 - (x[1] * q1 + x[2] * q2 + x[3] * q3);
        const double al1 = x[0] * q1 + q0 * x[1] - (x[2] * q3 - x[3] * q2);
        const double al2 = x[0] * q2 + q0 * x[2] - (x[3] * q1 - x[1] * q3);
        const double al3 = x[0] * q3 + q0 * x[3] - (x[1] * q2 - x[2] * q1);
        const Z e_ii = mk<double>(al0, al3), e_ij = mk<double>(al2, al1), e_ji = mk<double>(-al2, al1),
                e_jj = mk<double>(al0, -al3);
#pragma unroll
        for (int col = 0; col < 3; col++) {
            const Z ui = U[3 * i + col], uj = U[3 * j + col];
            U[3 * i + col] = e_ii * ui + e_ij * uj;
            U[3 * j + col] = e_ji * ui + e_jj * uj;
            const Z wi = W[3 * i + col], wj = W[3 * j + col];
            W[3 * i + col] = e_ii * wi + e_ij * wj;
            W[3 * j + col] = e_ji * wi + e_jj * wj;
        }
    }
    {   // back onto SU(3): a <- row0 / |row0|; b <- row1 - (a^dag . row1) a, normalised; row2 = (a x b)^*
        const double ia = 1.0 / sqrt(norm2(U[0]) + norm2(U[1]) + norm2(U[2]));
        U[0] = ia * U[0]; U[1] = ia * U[1]; U[2] = ia * U[2];
        Z ab = mulc(U[3], U[0]);
        ab = ab + mulc(U[4], U[1]);
        ab = ab + mulc(U[5], U[2]);
        U[3] = U[3] - ab * U[0]; U[4] = U[4] - ab * U[1]; U[5] = U[5] - ab * U[2];
        const double ib = 1.0 / sqrt(norm2(U[3]) + norm2(U[4]) + norm2(U[5]));
        U[3] = ib * U[3]; U[4] = ib * U[4]; U[5] = ib * U[5];
        reconstruct_row2(U);
    }
    C<R> out[9];
#pragma unroll
    for (int e = 0; e < 9; e++) out[e] = mk<R>((R)U[e].x, (R)U[e].y);
    store_link<R, NR>(links, g.V, mu, s, out);
}

// a changed configuration: forget the history and the counters, keep which link buffer is current
__global__ void k_reset_counters(DevState *st) {
    st->n_hist = 0; st->n_updates = 0; st->done = 0; st->nan = 0; st->F = 0.0; st->theta = 0.0;
}

unsigned long long heatbath_key(unsigned long long seed) {
    unsigned long long z = seed ^ 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

template <class R>
cudaError_t launch_heatbath(int nr, LinkPair<R> links, const Geom &g, const DevState *st, double beta,
                            unsigned long long key, unsigned long long sweep, int mu, int parity, LaunchStream stream,
                            bool overrelax, int order_tz) {
    const int nb = (int)((g.V / 2 + HB_THREADS - 1) / HB_THREADS);
    // z-planes per (z, t) tile: automatic = plain order unless one t slice of a class pass's traffic (every link
    // once) exceeds L2, then about 24 MB per tile; a forced value must divide Lz.  Measured on B200, same
    // thermalised state and sweeps: 64^4 fp64/18 plain 49.2 ms per sweep, tz = 2 / 4 / 8 / 16: 46.0 / 44.6 / 45.0 /
    // 46.4 ms (automatic picks 4); 32^4, where a t slice fits L2: 2.88 ms either way.
    int tz = g.L[2];
    if (order_tz > 0 && g.L[2] % order_tz == 0) tz = order_tz;
    else if (order_tz <= 0) {
        const double per_plane = (double)g.L[0] * g.L[1] * 4.0 * 6.0 * nr * 2.0 * sizeof(R);
        if (per_plane * g.L[2] > 64.0e6) {
            tz = 1;
            while (tz * 2 <= g.L[2] && g.L[2] % (tz * 2) == 0 && per_plane * tz * 2 <= 24.0e6) tz *= 2;
        }
    }
    const unsigned long long class_id = sweep * 8ULL + (unsigned long long)(mu * 2 + parity);
#define LGF_HB(NRV, ORV) \
    return launch_pdl(k_heatbath<R, NRV, ORV>, dim3(nb), dim3(HB_THREADS), 0, stream, links, g, st, beta, key, class_id, mu, parity, tz)
    if (overrelax) {
        if (nr == 3) LGF_HB(3, true);
        LGF_HB(2, true);
    }
    if (nr == 3) LGF_HB(3, false);
    LGF_HB(2, false);
#undef LGF_HB
}
cudaError_t launch_reset_counters(DevState *st, LaunchStream stream) {
    k_reset_counters<<<1, 1, 0, stream>>>(st);
    return cudaGetLastError();
}

template cudaError_t launch_heatbath<float>(int, LinkPair<float>, const Geom &, const DevState *, double,
                                            unsigned long long, unsigned long long, int, int, LaunchStream, bool, int);
template cudaError_t launch_heatbath<double>(int, LinkPair<double>, const Geom &, const DevState *, double,
                                             unsigned long long, unsigned long long, int, int, LaunchStream, bool, int);

}  // namespace lgf
