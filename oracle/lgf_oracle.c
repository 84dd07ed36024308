/*
 * lgf_oracle.c -- CPU ORACLE for Fourier-accelerated Landau gauge fixing (arXiv:1206.0675).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, double-precision
 * restatement of the paper's Algorithm 1 and of eqs. (2)-(8) (PAPER.md:45-76,
 * :148), written step by step in the paper's order so that it can be checked against the paper by
 * eye.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares no code, header, table or helper with the CUDA path under
 * paper_1206_0675_b200/csrc/ and neither includes the other.
 *
 * What pins it (tests/test_oracle_*.py, run with -m "not gpu"): brute-force O(V^2) DFT on 2^4 and
 * 4^4, numpy.fft.fftn, the x-space lattice-Laplacian identity for the Fourier-acceleration operator,
 * hermiticity/tracelessness/zero-sum of Delta, hand-computed single-link case, the first-order
 * identity dF = (alpha/2)/(12V) sum tr[w Delta], the abelian contraction ratio (1-8 alpha)^2,
 * library QR for the Gram-Schmidt projection, plaquette invariance, the pure-gauge closed form
 * (F -> 1, theta -> 0); for orc_gluon_field the identity F[Delta](k) = sum_mu (exp(-2 pi i k_mu/L_mu) - 1) A_mu(k)
 * against the pinned Delta and DFT, hermiticity in k space and transversality after fixing; for the product of
 * the g fields the defining property G U0 G(x+mu)^dag = U_n.  Parity status: no function here is "parity unpinned" except the
 * iteration COUNTS on the synthetic configurations (the paper prints none for inputs we have).
 *
 * Conventions:
 *   - lattice dims L[4] = {Lx, Ly, Lz, Lt}, periodic, site index s = x + Lx*(y + Ly*(z + Lz*t));
 *   - canonical link array U[s][mu][i][j], mu = 0..3 = x,y,z,t, row-major 3x3, complex double
 *     (re, im interleaved) -- site-major array of structures;
 *   - A_mu(x) = [(U - U^dag)/(2i)] - (1/3) tr[.] 1            (hermitian traceless; R1, R4)
 *   - Delta(x) = sum_mu [A_mu(x - mu) - A_mu(x)]                (eq. 5, eq. 7)
 *   - F = sum_x sum_mu Re tr U_mu(x) / (4*3*V)                  (eq. 3 at g = 1)
 *   - theta = sum_x tr[Delta Delta^dag] / (3 V)                 (eq. 6)
 *   - w = F^-1 [ (p2max/p2) F Delta ], p2 = 4 sum_mu sin^2(pi k_mu/L_mu), p2max = 16, zero mode -> 0,
 *     forward sign e^{-i}, inverse e^{+i} with a single 1/V       (eq. 4; Alg. 1 lines 3-8; R5-R7)
 *   - g(x) = GS(1 + i (alpha/2) w(x)), Gram-Schmidt on rows, third row = (row0 x row1)^*  (R8, R9, eq. 8)
 *   - U_mu(x) <- g(x) U_mu(x) g(x+mu)^dag for all x, mu from one complete g field        (eq. 2, R10)
 *
 * Build: gcc -O2 -std=c11 -fopenmp -fcx-limited-range -shared -fPIC lgf_oracle.c -o liblgf_oracle.so -lm
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------------------------ */
/* lattice geometry                                                                           */
/* ------------------------------------------------------------------------------------------ */

static long volume(const int L[4]) { return (long)L[0] * L[1] * L[2] * L[3]; }

static void site_coords(const int L[4], long s, int c[4])
{
    c[0] = (int)(s % L[0]); s /= L[0];
    c[1] = (int)(s % L[1]); s /= L[1];
    c[2] = (int)(s % L[2]); s /= L[2];
    c[3] = (int)s;
}

static long site_index(const int L[4], const int c[4])
{
    return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3]));
}

/* index of the site x + dir*mu^ (dir = +1 or -1), periodic */
static long neighbour(const int L[4], long s, int mu, int dir)
{
    int c[4];
    site_coords(L, s, c);
    c[mu] = (c[mu] + dir + L[mu]) % L[mu];
    return site_index(L, c);
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* 3x3 complex matrices, row-major m[3*i+j]                                                   */
/* ------------------------------------------------------------------------------------------ */

static void mat_mul(const cplx *a, const cplx *b, cplx *out)          /* out = a b */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            out[3 * i + j] = s;
        }
}

static void mat_mul_dag(const cplx *a, const cplx *b, cplx *out)      /* out = a b^dag */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cplx s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * conj(b[3 * j + k]);
            out[3 * i + j] = s;
        }
}

/* A = [(U - U^dag)/(2i)] - (1/3) tr[(U - U^dag)/(2i)] 1      (eq. 7 "- h.c. - trace", R1, R4) */
static void algebra_part(const cplx *U, cplx *A)
{
    cplx B[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++)
            B[3 * i + j] = (U[3 * i + j] - conj(U[3 * j + i])) / (2.0 * I);
    cplx tr = B[0] + B[4] + B[8];
    for (int i = 0; i < 9; i++) A[i] = B[i];
    A[0] -= tr / 3.0;
    A[4] -= tr / 3.0;
    A[8] -= tr / 3.0;
}

/* third row of an SU(3) matrix from the first two: c = (a x b)^*    (eq. 8) */
void orc_reconstruct_row3(const cplx *rows01, cplx *row2)
{
    const cplx *a = rows01, *b = rows01 + 3;
    row2[0] = conj(a[1] * b[2] - a[2] * b[1]);
    row2[1] = conj(a[2] * b[0] - a[0] * b[2]);
    row2[2] = conj(a[0] * b[1] - a[1] * b[0]);
}

/* Gram-Schmidt projection to SU(3) on the rows of M (R9):
 *   a = row0 / |row0|;  b = row1 - (a^* . row1) a;  b /= |b|;  c = (a x b)^*  */
void orc_gs(const cplx *M, cplx *G)
{
    cplx a[3], b[3];
    double na = 0;
    for (int j = 0; j < 3; j++) na += creal(M[j]) * creal(M[j]) + cimag(M[j]) * cimag(M[j]);
    na = sqrt(na);
    for (int j = 0; j < 3; j++) a[j] = M[j] / na;
    cplx ab = 0;
    for (int j = 0; j < 3; j++) ab += conj(a[j]) * M[3 + j];
    for (int j = 0; j < 3; j++) b[j] = M[3 + j] - ab * a[j];
    double nb = 0;
    for (int j = 0; j < 3; j++) nb += creal(b[j]) * creal(b[j]) + cimag(b[j]) * cimag(b[j]);
    nb = sqrt(nb);
    for (int j = 0; j < 3; j++) b[j] /= nb;
    for (int j = 0; j < 3; j++) { G[j] = a[j]; G[3 + j] = b[j]; }
    orc_reconstruct_row3(G, G + 6);
}

/* ------------------------------------------------------------------------------------------ */
/* Algorithm 1 line 1 / 17: Delta(x), F, theta        (eqs. 3, 5, 6, 7)                       */
/* ------------------------------------------------------------------------------------------ */

/* Delta may be NULL.  Delta[s*9 + 3*i + j]. */
void orc_measure(const int L[4], const cplx *U, cplx *Delta, double *F, double *theta)
{
    const long V = volume(L);
    double sumF = 0.0, sumT = 0.0;
#pragma omp parallel for reduction(+ : sumF, sumT) schedule(static)
    for (long s = 0; s < V; s++) {
        cplx D[9];
        for (int i = 0; i < 9; i++) D[i] = 0;
        for (int mu = 0; mu < 4; mu++) {
            const cplx *Ux = U + (s * 4 + mu) * 9;
            const cplx *Ub = U + (neighbour(L, s, mu, -1) * 4 + mu) * 9;
            cplx Ax[9], Ab[9];
            algebra_part(Ux, Ax);
            algebra_part(Ub, Ab);
            for (int i = 0; i < 9; i++) D[i] += Ab[i] - Ax[i];      /* eq. 5: f(x - mu) - f(x) */
            sumF += creal(Ux[0] + Ux[4] + Ux[8]);                   /* eq. 3 */
        }
        double t = 0;                                               /* tr(D D^dag) = sum |D_ij|^2 */
        for (int i = 0; i < 9; i++) t += creal(D[i]) * creal(D[i]) + cimag(D[i]) * cimag(D[i]);
        sumT += t;
        if (Delta)
            for (int i = 0; i < 9; i++) Delta[s * 9 + i] = D[i];
    }
    *F = sumF / (4.0 * 3.0 * (double)V);
    *theta = sumT / (3.0 * (double)V);
}

/* ------------------------------------------------------------------------------------------ */
/* naive separable DFT (Alg. 1 lines 4, 6): one 1-D DFT of length L_mu per line and axis,      */
/* each output a plain sum over the line.  sign = -1 forward, +1 inverse.  No normalisation.  */
/* ------------------------------------------------------------------------------------------ */

static void dft_axis(const int L[4], int axis, int sign, const cplx *in, cplx *out)
{
    const long V = volume(L);
    const int n = L[axis];
    long stride = 1;
    for (int a = 0; a < axis; a++) stride *= L[a];
    cplx *tw = (cplx *)malloc(sizeof(cplx) * n);     /* tw[m] = exp(sign 2 pi i m / n), m = k*x mod n */
    for (int m = 0; m < n; m++) {
        double ang = 2.0 * ORC_PI * (double)m / (double)n;
        tw[m] = cos(ang) + I * (sign * sin(ang));
    }
    const long nlines = V / n;
#pragma omp parallel for schedule(static)
    for (long l = 0; l < nlines; l++) {
        long lo = l % stride, hi = l / stride;
        long base = lo + hi * stride * n;
        for (int k = 0; k < n; k++) {
            cplx s = 0;
            for (int x = 0; x < n; x++) s += in[base + x * stride] * tw[(int)(((long)k * x) % n)];
            out[base + k * stride] = s;
        }
    }
    free(tw);
}

/* 4-D DFT of one complex scalar field f[s] (V entries), out may alias in */
void orc_dft4d(const int L[4], const cplx *in, int sign, cplx *out)
{
    const long V = volume(L);
    cplx *a = (cplx *)malloc(sizeof(cplx) * V);
    cplx *b = (cplx *)malloc(sizeof(cplx) * V);
    memcpy(a, in, sizeof(cplx) * V);
    for (int axis = 0; axis < 4; axis++) {
        dft_axis(L, axis, sign, a, b);
        cplx *t = a; a = b; b = t;
    }
    memcpy(out, a, sizeof(cplx) * V);
    free(a);
    free(b);
}

/* Gluon field in momentum space (the quantity gauge-fixed configurations are
 * made for):  Ak[k][i][j] = sum_x exp(-2 pi i sum_nu k_nu x_nu / L_nu) A_mu(x)_ij  with A_mu(x) the
 * hermitian traceless algebra part of U_mu(x) (eq. 7 as read in R1, R4), k = kx + Lx (ky + Ly (kz + Lz kt)),
 * unnormalised, the link's field taken at the site x (no mid-point phase exp(-i pi k_mu / L_mu)).
 * With this convention eq. 5 reads  F[Delta](k) = sum_mu (exp(-2 pi i k_mu / L_mu) - 1) Ak_mu(k). */
void orc_gluon_field(const int L[4], const cplx *U, int mu, cplx *Ak)
{
    const long V = volume(L);
    cplx *f = (cplx *)malloc(sizeof(cplx) * V);
    cplx *g = (cplx *)malloc(sizeof(cplx) * V);
    cplx *A = (cplx *)malloc(sizeof(cplx) * V * 9);
    for (long s = 0; s < V; s++) algebra_part(U + (s * 4 + mu) * 9, A + s * 9);
    for (int e = 0; e < 9; e++) {
        for (long s = 0; s < V; s++) f[s] = A[s * 9 + e];
        orc_dft4d(L, f, -1, g);
        for (long s = 0; s < V; s++) Ak[s * 9 + e] = g[s];
    }
    free(f); free(g); free(A);
}

/* p^2(k) = 4 sum_mu sin^2(pi k_mu / L_mu): eigenvalues of the lattice -d^2 (R5) */
double orc_p2(const int L[4], const int k[4])
{
    double p2 = 0;
    for (int mu = 0; mu < 4; mu++) {
        double s = sin(ORC_PI * (double)k[mu] / (double)L[mu]);
        p2 += 4.0 * s * s;
    }
    return p2;
}

/* Alg. 1 lines 3-8: for every matrix element ij of Delta: FFT forward, times p2max/p2, FFT backward,
 * normalise by 1/V.  Delta, w: [s*9 + ij]. */
void orc_accelerate(const int L[4], const cplx *Delta, cplx *w)
{
    const long V = volume(L);
    const double p2max = 16.0;
    cplx *f = (cplx *)malloc(sizeof(cplx) * V);
    for (int ij = 0; ij < 9; ij++) {
        for (long s = 0; s < V; s++) f[s] = Delta[s * 9 + ij];
        orc_dft4d(L, f, -1, f);                                     /* line 4: FFT forward      */
#pragma omp parallel for schedule(static)
        for (long s = 0; s < V; s++) {                              /* line 5: apply p2max / p2 */
            int k[4];
            site_coords(L, s, k);
            double p2 = orc_p2(L, k);
            if (k[0] == 0 && k[1] == 0 && k[2] == 0 && k[3] == 0) f[s] = 0;   /* zero mode (R6) */
            else f[s] *= p2max / p2;
        }
        orc_dft4d(L, f, +1, f);                                     /* line 6: FFT backward     */
        for (long s = 0; s < V; s++) w[s * 9 + ij] = f[s] / (double)V;        /* line 7: normalise */
    }
    free(f);
}

/* Alg. 1 lines 9-11: g(x) = GS(1 + i (alpha/2) w(x))    (exp to first order, then reunitarise) */
void orc_build_g(const int L[4], const cplx *w, double alpha, cplx *g)
{
    const long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++) {
        cplx M[9];
        for (int i = 0; i < 9; i++) M[i] = I * (alpha / 2.0) * w[s * 9 + i];
        M[0] += 1.0; M[4] += 1.0; M[8] += 1.0;
        orc_gs(M, g + s * 9);
    }
}

/* Alg. 1 lines 12-16: U_mu(x) <- g(x) U_mu(x) g(x + mu)^dag   (eq. 2).  Each link depends only on
 * itself and on the (complete, fixed) g field, so the in-place loop is the simultaneous update. */
void orc_transform(const int L[4], cplx *U, const cplx *g)
{
    const long V = volume(L);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; s++)
        for (int mu = 0; mu < 4; mu++) {
            cplx *Ux = U + (s * 4 + mu) * 9;
            const cplx *gx = g + s * 9;
            const cplx *gf = g + neighbour(L, s, mu, +1) * 9;
            cplx T[9], R[9];
            mat_mul(gx, Ux, T);
            mat_mul_dag(T, gf, R);
            for (int i = 0; i < 9; i++) Ux[i] = R[i];
        }
}

/* One pass of the while-body of Alg. 1 given Delta of the current configuration. */
static void update_from_delta(const int L[4], cplx *U, const cplx *Delta, double alpha, cplx *w, cplx *g)
{
    orc_accelerate(L, Delta, w);
    orc_build_g(L, w, alpha, g);
    orc_transform(L, U, g);
}

/* n updates.  Fh[i], Th[i] = F, theta of the configuration after i updates, i = 0..n (n+1 entries;
 * R12: entry 0 is the input).  Fh / Th may be NULL. */
void orc_iterate(const int L[4], cplx *U, double alpha, long n, double *Fh, double *Th)
{
    const long V = volume(L);
    cplx *Delta = (cplx *)malloc(sizeof(cplx) * V * 9);
    cplx *w = (cplx *)malloc(sizeof(cplx) * V * 9);
    cplx *g = (cplx *)malloc(sizeof(cplx) * V * 9);
    double F, th;
    orc_measure(L, U, Delta, &F, &th);
    if (Fh) Fh[0] = F;
    if (Th) Th[0] = th;
    for (long it = 0; it < n; it++) {
        update_from_delta(L, U, Delta, alpha, w, g);
        orc_measure(L, U, Delta, &F, &th);
        if (Fh) Fh[it + 1] = F;
        if (Th) Th[it + 1] = th;
    }
    free(Delta); free(w); free(g);
}

/* Algorithm 1: measure; while theta >= tol (and it < max_iter): update, measure.
 * Returns the number of updates applied.  History entries 0..it are written while they fit in
 * hist_cap (Fh/Th may be NULL). */
long orc_fix(const int L[4], cplx *U, double alpha, double tol, long max_iter,
             double *Fh, double *Th, long hist_cap)
{
    const long V = volume(L);
    cplx *Delta = (cplx *)malloc(sizeof(cplx) * V * 9);
    cplx *w = (cplx *)malloc(sizeof(cplx) * V * 9);
    cplx *g = (cplx *)malloc(sizeof(cplx) * V * 9);
    double F, th;
    long it = 0;
    orc_measure(L, U, Delta, &F, &th);                                  /* line 1 */
    if (Fh && hist_cap > 0) Fh[0] = F;
    if (Th && hist_cap > 0) Th[0] = th;
    while (th >= tol && it < max_iter) {                                /* line 2 */
        update_from_delta(L, U, Delta, alpha, w, g);                    /* lines 3-16 */
        orc_measure(L, U, Delta, &F, &th);                              /* line 17 */
        it++;
        if (Fh && it < hist_cap) Fh[it] = F;
        if (Th && it < hist_cap) Th[it] = th;
    }
    free(Delta); free(w); free(g);
    return it;
}

/* Average plaquette P = (1/(6*3*V)) sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag]
 * (standard definition; gauge invariant -- used as an invariant of the link update). */
double orc_plaquette(const int L[4], const cplx *U)
{
    const long V = volume(L);
    double sum = 0.0;
#pragma omp parallel for reduction(+ : sum) schedule(static)
    for (long s = 0; s < V; s++)
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                const cplx *U1 = U + (s * 4 + mu) * 9;
                const cplx *U2 = U + (neighbour(L, s, mu, +1) * 4 + nu) * 9;
                const cplx *U3 = U + (neighbour(L, s, nu, +1) * 4 + mu) * 9;
                const cplx *U4 = U + (s * 4 + nu) * 9;
                cplx T1[9], T2[9], T3[9];
                mat_mul(U1, U2, T1);
                mat_mul_dag(T1, U3, T2);
                mat_mul_dag(T2, U4, T3);
                sum += creal(T3[0] + T3[4] + T3[8]);
            }
    return sum / (6.0 * 3.0 * (double)V);
}
