/*
 * lgf_heatbath_oracle.c -- CPU ORACLE for the thermalisation of SU(3) Wilson-action configurations
 * (SURVEY.md section 8(f) NEXT-1): the producer of the paper's kind of input.  The paper only says the
 * ensembles were "generated via importance sampling using, for example, the Wilson action" at beta = 5.8,
 * 6.0, 6.2 (PAPER.md:50, :211, :237; generator cited as ref. [18], :270) and names no algorithm, so any exact
 * sampler of exp(-S) is admissible; the reading taken (R24-R27) is the textbook one:
 * Cabibbo-Marinari pseudo-heat-bath over the three SU(2) subgroups with Kennedy-Pendleton sampling.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT; plain double-precision C, no code shared with
 * paper_1206_0675_b200/csrc/.  Pins (tests/test_oracle_heatbath.py): staples against the pinned plaquette and
 * a numpy brute force, the Kennedy-Pendleton sampler against the closed form <x0> = I_2(a)/I_1(a), group
 * membership, the strong-coupling limit P = beta/18, the weak-coupling (equipartition) limit 1 - P = 2/beta,
 * and the counter-based stream (splitting a run does not change it).
 *
 * Definitions
 *   S = beta sum_p [1 - Re tr U_p / 3] over the 6V plaquettes                                  (R24)
 *   staple sum A_mu(x) = sum_{nu != mu} [ U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
 *                                       + U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) ],
 *     so that the plaquettes containing the link add up to Re tr[U_mu(x) A_mu(x)]
 *   sweep number n (counted from the first sweep applied to the loaded configuration): for mu = 0..3, for
 *     parity = 0, 1: every link (x, mu) with (x0+x1+x2+x3) mod 2 = parity is updated from the current
 *     neighbours (they all belong to other classes, so the order inside a class is irrelevant).  All
 *     extents must be even.                                                                    (R25)
 *   link update: W = U A; for the subgroups k = 0, 1, 2 acting on rows/columns (i, j) = (0,1), (0,2), (1,2):
 *     a = W_ii, b = W_ij, c = W_ji, d = W_jj;
 *     r0 = Re(a+d)/2, r1 = Im(b+c)/2, r2 = Re(b-c)/2, r3 = Im(a-d)/2, kk = |r|, V = r / kk  (an SU(2) element
 *     written as a unit quaternion q0 + i q.sigma = [[q0 + i q3, q2 + i q1], [-q2 + i q1, q0 - i q3]]);
 *     X ~ exp(a_kp x0) sqrt(1 - x0^2) dx0 dOmega with a_kp = 2 beta kk / 3 (Creutz / Kennedy-Pendleton, below);
 *     alpha = X V^dag; U <- E(alpha) U, W <- E(alpha) W with E the embedding of alpha in rows/columns i, j.  (R26)
 *   sampling x0, attempt t = 0, 1, ... (six uniforms u0..u5 per attempt):
 *     a_kp >= 2 (Kennedy-Pendleton): delta = -(ln u0 + cos^2(2 pi u1) ln u2) / a_kp; accept if u3^2 <= 1 - delta/2;
 *     a_kp <  2 (Creutz): delta = -ln(u0 + (1 - u0) exp(-2 a_kp)) / a_kp, i.e. x0 = 1 - delta drawn from
 *       exp(a_kp x0) on [-1, 1] by inverting its distribution function; accept if u3^2 <= 1 - x0^2;
 *     x0 = 1 - delta; direction cos(theta) = 2 u4 - 1, phi = 2 pi u5,
 *     x = sqrt(1 - x0^2) (sin(theta) cos(phi), sin(theta) sin(phi), cos(theta)).
 *     Both are exact; Kennedy-Pendleton alone is not usable at small a_kp with a bounded number of attempts
 *     (its acceptance falls like a_kp^(3/2): at a_kp = 0.2, 5 % of the draws exhaust 32 attempts and the
 *     strong-coupling pin P = beta/18 fails by 30 %), Creutz alone not at large a_kp.  With the switch at 2 the
 *     rejection probability per attempt stays below 0.5; after HB_MAXATT = 32 rejections (< 1e-9) the last
 *     delta, clipped to [0, 2], is used.
 *   overrelaxation sweep (microcanonical, no random numbers): same class order and subgroups, with
 *     alpha = (V^dag)^2 instead of the heat-bath draw: alpha V = V^dag has the same x0 as V, so Re tr[U A] -- and
 *     with it the action -- is unchanged by every single step; then the same re-projection.            (R28)
 *   uniforms: u_n = ((mix64(key + (idx + 1) G) >> 11) + 0.5) 2^-53, key = mix64(seed ^ G), G = 0x9E3779B97F4A7C15,
 *     mix64 = the splitmix64 finaliser, idx = (((((sweep 8 + mu 2 + parity) V + site) 3 + k) 32 + t) 6 + n).   (R27)
 *   After its three subgroup updates the link is re-projected onto SU(3): Gram-Schmidt on rows 0, 1, row 2 =
 *     (row0 x row1)^* (the same projection as the gauge fixer's, eq. 8).  On a unitary matrix this
 *     changes the last bits only, but it is needed: with 12-real link storage (row 2 rebuilt on every load) the
 *     norm error of rows 0, 1 is fed back through the rebuilt row by the (0,2) and (1,2) updates and grows
 *     exponentially -- 5e-13 after 25 sweeps, 7.5e-7 after 100, overflow before 300 on the CUDA side.      (R26)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define HB_PI 3.14159265358979323846264338327950288
#define HB_MAXATT 32

static long hb_volume(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }
static void hb_coords(const int L[4], long s, int c[4])
{
    c[0] = (int)(s % L[0]); s /= L[0];
    c[1] = (int)(s % L[1]); s /= L[1];
    c[2] = (int)(s % L[2]);
    c[3] = (int)(s / L[2]);
}
static long hb_index(const int L[4], const int c[4])
{
    return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3]));
}
/* site x + d1 mu^ + d2 nu^ (periodic), d = -1, 0, +1 */
static long hb_shift2(const int L[4], long s, int mu, int d1, int nu, int d2)
{
    int c[4];
    hb_coords(L, s, c);
    c[mu] = (c[mu] + d1 + L[mu]) % L[mu];
    c[nu] = (c[nu] + d2 + L[nu]) % L[nu];
    return hb_index(L, c);
}

/* out = op(a) op(b), dagger flags da, db */
static void hb_mul(const cplx *a, int da, const cplx *b, int db, cplx *out)
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0.0;
            for (int k = 0; k < 3; k++) {
                const cplx x = da ? conj(a[3 * k + i]) : a[3 * i + k];
                const cplx y = db ? conj(b[3 * j + k]) : b[3 * k + j];
                s += x * y;
            }
            out[3 * i + j] = s;
        }
}

static uint64_t hb_mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static double hb_uniform(uint64_t seed, uint64_t idx)
{
    const uint64_t G = 0x9E3779B97F4A7C15ULL;
    const uint64_t key = hb_mix64(seed ^ G);
    const uint64_t z = hb_mix64(key + (idx + 1) * G);
    return ((double)(z >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* ------------------------------------------------------------------------------------------ */
/* staples                                                                                    */
/* ------------------------------------------------------------------------------------------ */
/* A_mu(x) as defined in the header, for one link */
static void hb_staple(const int L[4], const cplx *U, long s, int mu, cplx *A)
{
    for (int e = 0; e < 9; e++) A[e] = 0.0;
    const long s_mu = hb_shift2(L, s, mu, +1, mu, 0);
    for (int nu = 0; nu < 4; nu++) {
        if (nu == mu) continue;
        cplx T[9], P[9];
        /* upper staple: U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag */
        const long s_nu = hb_shift2(L, s, nu, +1, nu, 0);
        hb_mul(U + (s_mu * 4 + nu) * 9, 0, U + (s_nu * 4 + mu) * 9, 1, T);
        hb_mul(T, 0, U + (s * 4 + nu) * 9, 1, P);
        for (int e = 0; e < 9; e++) A[e] += P[e];
        /* lower staple: U_nu(x+mu-nu)^dag U_mu(x-nu)^dag U_nu(x-nu) */
        const long s_mu_mnu = hb_shift2(L, s, mu, +1, nu, -1);
        const long s_mnu = hb_shift2(L, s, nu, -1, nu, 0);
        hb_mul(U + (s_mu_mnu * 4 + nu) * 9, 1, U + (s_mnu * 4 + mu) * 9, 1, T);
        hb_mul(T, 0, U + (s_mnu * 4 + nu) * 9, 0, P);
        for (int e = 0; e < 9; e++) A[e] += P[e];
    }
}

/* staple sums of every link: A[s][mu][3][3] */
void orc_hb_staples(const int L[4], const cplx *U, cplx *A)
{
    const long V = hb_volume(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        for (int mu = 0; mu < 4; mu++) hb_staple(L, U, s, mu, A + (s * 4 + mu) * 9);
}

/* ------------------------------------------------------------------------------------------ */
/* Kennedy-Pendleton                                                                          */
/* ------------------------------------------------------------------------------------------ */
/* X (unit quaternion x[0..3]) with density exp(a x0) sqrt(1 - x0^2) dx0 dOmega, a > 0; the uniforms are numbers
 * base + 6 t + n of stream `seed`, t = attempt.  Returns the number of attempts used. */
static int hb_kp(double a, uint64_t seed, uint64_t base, double x[4])
{
    double delta = 0.0;
    int t, used = HB_MAXATT;
    for (t = 0; t < HB_MAXATT; t++) {
        const double u0 = hb_uniform(seed, base + 6 * (uint64_t)t + 0);
        const double u1 = hb_uniform(seed, base + 6 * (uint64_t)t + 1);
        const double u2 = hb_uniform(seed, base + 6 * (uint64_t)t + 2);
        const double u3 = hb_uniform(seed, base + 6 * (uint64_t)t + 3);
        if (a >= 2.0) {                                        /* Kennedy-Pendleton */
            const double c = cos(2.0 * HB_PI * u1);
            delta = -(log(u0) + c * c * log(u2)) / a;
            if (u3 * u3 <= 1.0 - 0.5 * delta) { used = t + 1; break; }
        } else {                                               /* Creutz */
            delta = -log(u0 + (1.0 - u0) * exp(-2.0 * a)) / a;
            const double x0 = 1.0 - delta;
            if (u3 * u3 <= 1.0 - x0 * x0) { used = t + 1; break; }
        }
    }
    if (t == HB_MAXATT) {
        t = HB_MAXATT - 1;
        if (delta > 2.0) delta = 2.0;
        if (delta < 0.0) delta = 0.0;
    }
    const double u4 = hb_uniform(seed, base + 6 * (uint64_t)t + 4);
    const double u5 = hb_uniform(seed, base + 6 * (uint64_t)t + 5);
    const double x0 = 1.0 - delta;
    double rr = 1.0 - x0 * x0;
    rr = rr > 0.0 ? sqrt(rr) : 0.0;
    const double ct = 2.0 * u4 - 1.0;
    double st = 1.0 - ct * ct;
    st = st > 0.0 ? sqrt(st) : 0.0;
    const double phi = 2.0 * HB_PI * u5;
    x[0] = x0;
    x[1] = rr * st * cos(phi);
    x[2] = rr * st * sin(phi);
    x[3] = rr * ct;
    return used;
}

/* n independent draws at parameter a: X[n][4], attempts[n]; draw i uses the uniforms from index 192 i on */
void orc_hb_kp_sample(double a, unsigned long long seed, long n, double *X, int *attempts)
{
    for (long i = 0; i < n; i++) attempts[i] = hb_kp(a, seed, (uint64_t)i * 6 * HB_MAXATT, X + 4 * i);
}

/* ------------------------------------------------------------------------------------------ */
/* the sweep                                                                                  */
/* ------------------------------------------------------------------------------------------ */
void orc_gs(const cplx *M, cplx *G);      /* lgf_oracle.c: Gram-Schmidt projection onto SU(3), pinned there */

/* overrelax != 0: alpha = (V^dag)^2 (R28), beta / seed / link_idx unused */
static void hb_update_link(cplx *U, const cplx *A, double beta, uint64_t seed, uint64_t link_idx, int overrelax)
{
    static const int PAIR[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    cplx W[9];
    hb_mul(U, 0, A, 0, W);
    for (int k = 0; k < 3; k++) {
        const int i = PAIR[k][0], j = PAIR[k][1];
        const cplx a = W[3 * i + i], b = W[3 * i + j], c = W[3 * j + i], d = W[3 * j + j];
        const double r0 = 0.5 * creal(a + d), r1 = 0.5 * cimag(b + c), r2 = 0.5 * creal(b - c), r3 = 0.5 * cimag(a - d);
        const double kk = sqrt(r0 * r0 + r1 * r1 + r2 * r2 + r3 * r3);
        if (!(kk > 1e-300)) continue;                       /* degenerate staple: leave this subgroup alone */
        /* alpha = X V^dag, V^dag = (r0, -r) / kk; quaternion product (p0, p)(q0, q) = (p0 q0 - p.q, p0 q + q0 p - p x q) */
        const double q0 = r0 / kk, q1 = -r1 / kk, q2 = -r2 / kk, q3 = -r3 / kk;
        double x[4];
        if (overrelax) { x[0] = q0; x[1] = q1; x[2] = q2; x[3] = q3; }      /* X = V^dag: alpha = V^dag V^dag */
        else hb_kp(2.0 * beta * kk / 3.0, seed, ((link_idx * 3 + (uint64_t)k) * HB_MAXATT) * 6, x);
        const double al0 = x[0] * q0 - (x[1] * q1 + x[2] * q2 + x[3] * q3);
        const double al1 = x[0] * q1 + q0 * x[1] - (x[2] * q3 - x[3] * q2);
        const double al2 = x[0] * q2 + q0 * x[2] - (x[3] * q1 - x[1] * q3);
        const double al3 = x[0] * q3 + q0 * x[3] - (x[1] * q2 - x[2] * q1);
        const cplx e_ii = al0 + I * al3, e_ij = al2 + I * al1, e_ji = -al2 + I * al1, e_jj = al0 - I * al3;
        for (int col = 0; col < 3; col++) {                  /* rows i and j of U and of W */
            const cplx ui = U[3 * i + col], uj = U[3 * j + col];
            U[3 * i + col] = e_ii * ui + e_ij * uj;
            U[3 * j + col] = e_ji * ui + e_jj * uj;
            const cplx wi = W[3 * i + col], wj = W[3 * j + col];
            W[3 * i + col] = e_ii * wi + e_ij * wj;
            W[3 * j + col] = e_ji * wi + e_jj * wj;
        }
    }
    cplx P[9];
    orc_gs(U, P);                                            /* back onto SU(3) */
    memcpy(U, P, sizeof(P));
}

/* nsweeps sweeps, numbered sweep0, sweep0 + 1, ... (the number selects the random stream, so a run may be
 * split across calls).  Returns 0, or -1 if an extent is odd. */
int orc_heatbath(const int L[4], cplx *U, double beta, unsigned long long seed, long sweep0, long nsweeps)
{
    for (int mu = 0; mu < 4; mu++)
        if (L[mu] % 2) return -1;
    const long V = hb_volume(L);
    for (long sw = sweep0; sw < sweep0 + nsweeps; sw++)
        for (int mu = 0; mu < 4; mu++)
            for (int parity = 0; parity < 2; parity++) {
#pragma omp parallel for schedule(static)
                for (long s = 0; s < V; s++) {
                    int c[4];
                    hb_coords(L, s, c);
                    if (((c[0] + c[1] + c[2] + c[3]) & 1) != parity) continue;
                    cplx A[9];
                    hb_staple(L, U, s, mu, A);
                    const uint64_t link_idx = ((uint64_t)sw * 8 + (uint64_t)(mu * 2 + parity)) * (uint64_t)V + (uint64_t)s;
                    hb_update_link(U + (s * 4 + mu) * 9, A, beta, (uint64_t)seed, link_idx, 0);
                }
            }
    return 0;
}

/* nsweeps overrelaxation sweeps (R28).  Returns 0, or -1 if an extent is odd. */
int orc_overrelax(const int L[4], cplx *U, long nsweeps)
{
    for (int mu = 0; mu < 4; mu++)
        if (L[mu] % 2) return -1;
    const long V = hb_volume(L);
    for (long sw = 0; sw < nsweeps; sw++)
        for (int mu = 0; mu < 4; mu++)
            for (int parity = 0; parity < 2; parity++) {
#pragma omp parallel for schedule(static)
                for (long s = 0; s < V; s++) {
                    int c[4];
                    hb_coords(L, s, c);
                    if (((c[0] + c[1] + c[2] + c[3]) & 1) != parity) continue;
                    cplx A[9];
                    hb_staple(L, U, s, mu, A);
                    hb_update_link(U + (s * 4 + mu) * 9, A, 0.0, 0, 0, 1);
                }
            }
    return 0;
}
