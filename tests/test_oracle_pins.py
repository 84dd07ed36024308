"""Pins of the CPU oracle (oracle/lgf_oracle.c) against facts fixed by the paper and by mathematics --
never against itself and never against the CUDA path.  Each test says which plausible mistake it is
meant to catch.  CPU only (-m "not gpu").

Citations: PAPER.md line numbers (arXiv:1206.0675) and SURVEY.md section 8(c) readings R1-R23.
"""
import itertools

import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

EYE = np.eye(3, dtype=np.complex128)


def dag(a):
    return np.conj(np.swapaxes(a, -1, -2))


def site_shape(dims):
    return (dims[3], dims[2], dims[1], dims[0])


def shift(f, mu, d):
    """f(x + d*mu^) on the (Lt, Lz, Ly, Lx, ...) grid."""
    return np.roll(f, -d, axis=3 - mu)


def rng_field(dims, seed, extra=()):
    r = np.random.default_rng(seed)
    shp = site_shape(dims) + tuple(extra)
    return r.normal(size=shp) + 1j * r.normal(size=shp)


# ------------------------------------------------------------------------------------------------
# separable DFT  (Alg. 1 lines 4 and 6)
# ------------------------------------------------------------------------------------------------

def brute_force_dft(dims, f, sign):
    """O(V^2) definition: F(k) = sum_x exp(sign 2 pi i sum_mu k_mu x_mu / L_mu) f(x), python loops."""
    Lx, Ly, Lz, Lt = dims
    out = np.zeros_like(f)
    pts = list(itertools.product(range(Lt), range(Lz), range(Ly), range(Lx)))
    for (kt, kz, ky, kx) in pts:
        s = 0j
        for (t, z, y, x) in pts:
            ph = kx * x / Lx + ky * y / Ly + kz * z / Lz + kt * t / Lt
            s += np.exp(sign * 2j * np.pi * ph) * f[t, z, y, x]
        out[kt, kz, ky, kx] = s
    return out


def test_dft_brute_force_2x2x2x2():
    dims = (2, 2, 2, 2)
    f = rng_field(dims, 1)
    for sign in (-1, +1):
        assert np.abs(oracle.dft4d(dims, f, sign) - brute_force_dft(dims, f, sign)).max() < 1e-13


def test_dft_brute_force_4x4x4x4_matrix():
    # full V x V DFT matrix (V = 256), built from the definition
    dims = (4, 4, 4, 4)
    f = rng_field(dims, 2)
    t, z, y, x = np.meshgrid(*[np.arange(4)] * 4, indexing="ij")
    X = np.stack([x.ravel(), y.ravel(), z.ravel(), t.ravel()], 1)  # site -> coords
    phase = (X[:, None, :] * X[None, :, :] / 4.0).sum(-1)          # sum_mu k_mu x_mu / L_mu
    for sign in (-1, +1):
        M = np.exp(sign * 2j * np.pi * phase)
        want = (M @ f.ravel()).reshape(f.shape)
        assert np.abs(oracle.dft4d(dims, f, sign) - want).max() < 1e-12


def test_dft_brute_force_asymmetric():
    # catches swapped axes / wrong strides: all four lengths differ, includes a radix-3 length
    dims = (2, 3, 4, 2)
    f = rng_field(dims, 3)
    assert np.abs(oracle.dft4d(dims, f, -1) - brute_force_dft(dims, f, -1)).max() < 1e-13


@pytest.mark.parametrize("dims", [(4, 6, 8, 12), (8, 8, 8, 8), (6, 4, 2, 3)])
def test_dft_matches_library_fft(dims):
    f = rng_field(dims, 4)
    V = np.prod(dims)
    assert np.abs(oracle.dft4d(dims, f, -1) - np.fft.fftn(f)).max() < 1e-11
    assert np.abs(oracle.dft4d(dims, f, +1) - np.fft.ifftn(f) * V).max() < 1e-11
    # round trip with the single 1/V of R7
    assert np.abs(oracle.dft4d(dims, oracle.dft4d(dims, f, -1), +1) / V - f).max() < 1e-13


# ------------------------------------------------------------------------------------------------
# Fourier acceleration operator  w = F^-1 (p2max/p2) F Delta   (eq. 4; R5-R7)
# ------------------------------------------------------------------------------------------------

def lattice_minus_laplacian(w):
    out = np.zeros_like(w)
    for mu in range(4):
        out -= shift(w, mu, +1) + shift(w, mu, -1) - 2 * w
    return out


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 12), (6, 6, 6, 12)])
def test_accelerate_inverts_lattice_laplacian(dims):
    """p^2 are the eigenvalues of -d^2: without any DFT, in x space,
    -sum_mu [w(x+mu) + w(x-mu) - 2 w(x)] = p2max * Delta(x) for zero-sum Delta.  Pins the p^2 formula,
    p2max = 16, the zero-mode choice and the 1/V normalisation in one go."""
    D = rng_field(dims, 5, (3, 3))
    D -= D.mean(axis=(0, 1, 2, 3), keepdims=True)        # zero mode removed (R6)
    w = oracle.accelerate(dims, D)
    assert np.abs(lattice_minus_laplacian(w) - 16.0 * D).max() < 1e-11
    # the zero mode of w itself is set to 0
    assert np.abs(w.mean(axis=(0, 1, 2, 3))).max() < 1e-13


def test_accelerate_zero_mode_is_dropped():
    dims = (4, 4, 4, 4)
    D = np.ones(site_shape(dims) + (3, 3), np.complex128) * (2.0 - 1.0j)
    assert np.abs(oracle.accelerate(dims, D)).max() < 1e-13


@pytest.mark.parametrize("k,factor", [((2, 2, 2, 2), 1.0),      # p2 = 16 = p2max
                                       ((2, 0, 0, 0), 4.0),      # p2 = 4
                                       ((1, 0, 0, 0), 8.0),      # p2 = 4 sin^2(pi/4) = 2
                                       ((1, 1, 1, 1), 2.0),      # p2 = 8
                                       ((3, 0, 2, 0), 16.0 / 6)])
def test_accelerate_plane_wave_closed_forms(k, factor):
    """A plane wave e^{2 pi i k.x/L} on 4^4 must come back multiplied by p2max/p2(k): closed-form values."""
    dims = (4, 4, 4, 4)
    t, z, y, x = np.meshgrid(*[np.arange(4)] * 4, indexing="ij")
    pw = np.exp(2j * np.pi * (k[0] * x + k[1] * y + k[2] * z + k[3] * t) / 4.0)
    D = np.zeros(site_shape(dims) + (3, 3), np.complex128)
    D[..., 0, 1] = pw
    D[..., 2, 2] = 3.0 * pw
    w = oracle.accelerate(dims, D)
    assert np.abs(w[..., 0, 1] - factor * pw).max() < 1e-13
    assert np.abs(w[..., 2, 2] - 3.0 * factor * pw).max() < 1e-13
    assert np.abs(w[..., 1, 0]).max() < 1e-14                     # components do not mix
    assert abs(oracle.p2(dims, k) - 16.0 / factor) < 1e-14


def test_accelerate_maps_hermitian_to_hermitian():
    # the multiplier is real and even in k, so hermitian traceless Delta gives hermitian traceless w
    dims = (4, 6, 4, 6)
    D = rng_field(dims, 6, (3, 3))
    D = D + dag(D)
    D -= np.trace(D, axis1=-2, axis2=-1)[..., None, None] * EYE / 3
    w = oracle.accelerate(dims, D)
    assert np.abs(w - dag(w)).max() < 1e-12
    assert np.abs(np.trace(w, axis1=-2, axis2=-1)).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# Delta, F, theta   (eqs. 3, 5, 6, 7; R1, R3, R4)
# ------------------------------------------------------------------------------------------------

def test_measure_unit_configuration():
    dims = (4, 4, 4, 4)
    U = np.broadcast_to(EYE, site_shape(dims) + (4, 3, 3)).copy()
    D, F, th = oracle.measure(dims, U)
    assert F == 1.0 and th == 0.0 and np.abs(D).max() == 0.0


def test_measure_constant_links():
    # x-independent U_mu: the lattice divergence vanishes identically, F is the mean trace
    dims = (4, 6, 4, 2)
    h = inputs.haar_su3(11, inputs.STREAM_HAAR, 0, 4)
    U = np.broadcast_to(h, site_shape(dims) + (4, 3, 3)).copy()
    D, F, th = oracle.measure(dims, U)
    assert np.abs(D).max() < 1e-15 and th < 1e-30
    assert abs(F - np.trace(h, axis1=-2, axis2=-1).real.sum() / 12.0) < 1e-15


def test_measure_delta_is_hermitian_traceless_zero_sum():
    dims = (4, 6, 4, 6)
    U = inputs.smooth_config(dims, 0.3, 21)
    D, F, th = oracle.measure(dims, U)
    assert np.abs(D - dag(D)).max() < 1e-15
    assert np.abs(np.trace(D, axis1=-2, axis2=-1)).max() < 1e-15
    assert np.abs(D.sum(axis=(0, 1, 2, 3))).max() < 1e-12        # telescoping over the periodic lattice
    # theta from the returned Delta (eq. 6) and F from the definition (eq. 3 at g = 1)
    V = np.prod(dims)
    assert abs(th - (np.abs(D) ** 2).sum() / (3 * V)) < 1e-14 * th
    assert abs(F - np.trace(U, axis1=-2, axis2=-1).real.sum() / (12 * V)) < 1e-15


@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_measure_single_link_hand_computed(mu):
    """All links 1 except U_mu(x0) = exp(i a lambda_2) = [[c, s, 0], [-s, c, 0], [0, 0, 1]].
    Then A_mu(x0) = sin(a) lambda_2, Delta(x0) = -A, Delta(x0 + mu) = +A, zero elsewhere.
    Catches: the sign of Delta (x - mu vs x + mu), a transposed operand in U - U^dag, a missing 1/(2i)."""
    dims = (4, 4, 4, 4)
    V = 256
    a = 0.37
    U = np.broadcast_to(EYE, site_shape(dims) + (4, 3, 3)).copy()
    x0 = [1, 2, 3, 0]                                   # (x, y, z, t)
    link = np.array([[np.cos(a), np.sin(a), 0], [-np.sin(a), np.cos(a), 0], [0, 0, 1]], complex)
    U[x0[3], x0[2], x0[1], x0[0], mu] = link
    lam2 = np.array([[0, -1j, 0], [1j, 0, 0], [0, 0, 0]])
    A = np.sin(a) * lam2
    D, F, th = oracle.measure(dims, U)
    x1 = list(x0)
    x1[mu] = (x1[mu] + 1) % 4
    want = np.zeros_like(D)
    want[x0[3], x0[2], x0[1], x0[0]] = -A
    want[x1[3], x1[2], x1[1], x1[0]] = +A
    assert np.abs(D - want).max() < 1e-16
    assert abs(th - 2 * 2 * np.sin(a) ** 2 / (3 * V)) < 1e-17   # tr(A A^dag) = 2 sin^2 a, two sites
    assert abs(F - (1 - (2 - 2 * np.cos(a)) / (12 * V))) < 1e-15


def test_algebra_part_is_first_order_field():
    # U = exp(i eps H): A = H eps + O(eps^3) -- pins the 1/(2i) and the overall sign (eq. 1, R1)
    dims = (2, 2, 2, 2)
    eps = 1e-4
    c = inputs.normals(5, inputs.STREAM_H, 0, 16 * 4 * 8).reshape(64, 8)
    H = np.einsum("na,aij->nij", c.astype(complex), inputs.gell_mann()).reshape(site_shape(dims) + (4, 3, 3))
    U = inputs.smooth_config(dims, eps, 5, haar=False)
    D, F, th = oracle.measure(dims, U)
    want = np.zeros_like(D)
    for mu in range(4):
        Amu = eps * H[..., mu, :, :]
        want += shift(Amu, mu, -1) - Amu
    assert np.abs(D - want).max() < 50 * eps ** 3


# ------------------------------------------------------------------------------------------------
# Gram-Schmidt reunitarisation and eq. (8)   (R9)
# ------------------------------------------------------------------------------------------------

def test_gs_equals_library_qr():
    r = np.random.default_rng(7)
    for _ in range(50):
        M = EYE + 0.3 * (r.normal(size=(3, 3)) + 1j * r.normal(size=(3, 3)))
        G = oracle.gs(M)
        Q, R = np.linalg.qr(M.T)                       # rows of M = columns of M^T
        d = np.diag(R)
        Q = Q * (d / np.abs(d))[None, :]               # M^T = (Q ph)(ph^* R) with positive diagonal
        # columns of Q with positive-diagonal R are the Gram-Schmidt vectors
        assert np.abs(G[0] - Q[:, 0]).max() < 1e-14
        assert np.abs(G[1] - Q[:, 1]).max() < 1e-14
        assert np.abs(G @ dag(G) - EYE).max() < 1e-15 * 8
        assert abs(np.linalg.det(G) - 1) < 1e-14
        # third row is the unique completion to det = 1: proportional to Q[:, 2]
        ph = G[2] @ np.conj(Q[:, 2])
        assert abs(abs(ph) - 1) < 1e-14


def test_gs_is_identity_on_su3():
    for g in inputs.haar_su3(3, inputs.STREAM_HAAR, 0, 20):
        assert np.abs(oracle.gs(g) - g).max() < 1e-14


def test_reconstruct_row3_eq8():
    for g in inputs.haar_su3(4, inputs.STREAM_HAAR, 0, 50):
        assert np.abs(oracle.reconstruct_row3(g[:2]) - g[2]).max() < 2e-15


def test_build_g_first_order_and_projection():
    # g = GS(1 + i (alpha/2) w): for tiny w equals exp(i (alpha/2) w) to second order; always in SU(3)
    dims = (2, 2, 2, 2)
    w = rng_field(dims, 8, (3, 3))
    w = w + dag(w)
    w -= np.trace(w, axis1=-2, axis2=-1)[..., None, None] * EYE / 3
    alpha = 0.08
    g = oracle.build_g(dims, w, alpha)
    assert np.abs(g @ dag(g) - EYE).max() < 1e-14
    assert np.abs(np.linalg.det(g) - 1).max() < 1e-14
    small = 1e-5 * w
    g2 = oracle.build_g(dims, small, alpha)
    assert np.abs(g2 - (EYE + 1j * (alpha / 2) * small)).max() < 1e-9   # O(|alpha w|^2)


# ------------------------------------------------------------------------------------------------
# link transform  U_mu(x) <- g(x) U_mu(x) g(x+mu)^dag   (eq. 2; Alg. 1 line 14)
# ------------------------------------------------------------------------------------------------

def test_transform_undoes_pure_gauge():
    """U = h(x) h(x+mu)^dag transformed with g = h^dag must give U = 1 exactly.  Catches g on the wrong
    side, a missing dagger, and a shift in the wrong direction (x - mu instead of x + mu)."""
    dims = (4, 2, 6, 4)
    V = int(np.prod(dims))
    U = inputs.pure_gauge_config(dims, 31)
    h = inputs.haar_su3(31, inputs.STREAM_HAAR, 0, V).reshape(site_shape(dims) + (3, 3))
    U1 = oracle.transform(dims, U, dag(h))
    assert np.abs(U1 - EYE).max() < 1e-14


def test_transform_preserves_plaquette_and_group():
    dims = (4, 4, 6, 2)
    V = int(np.prod(dims))
    U = inputs.smooth_config(dims, 0.4, 32)
    g = inputs.haar_su3(33, inputs.STREAM_HAAR, 0, V).reshape(site_shape(dims) + (3, 3))
    U1 = oracle.transform(dims, U, g)
    assert abs(oracle.plaquette(dims, U1) - oracle.plaquette(dims, U)) < 1e-14
    assert np.abs(U1 @ dag(U1) - EYE).max() < 1e-13
    assert np.abs(np.linalg.det(U1) - 1).max() < 1e-13
    # global (x-independent) g: tr U and tr(Delta Delta^dag) are invariant
    gc = np.broadcast_to(g[0, 0, 0, 0], g.shape).copy()
    _, F0, th0 = oracle.measure(dims, U)
    _, F1, th1 = oracle.measure(dims, oracle.transform(dims, U, gc))
    assert abs(F1 - F0) < 1e-14 and abs(th1 - th0) < 1e-13 * th0


def test_plaquette_closed_forms():
    dims = (4, 4, 4, 4)
    V = 256
    one = np.broadcast_to(EYE, site_shape(dims) + (4, 3, 3)).copy()
    assert oracle.plaquette(dims, one) == 1.0
    assert abs(oracle.plaquette(dims, inputs.pure_gauge_config(dims, 41)) - 1.0) < 1e-14
    # one link diag(e^{ia}, e^{-ia}, 1): it sits in 6 plaquettes, each with Re tr = 1 + 2 cos a
    a = 0.7
    one[1, 2, 3, 0, 2] = np.diag([np.exp(1j * a), np.exp(-1j * a), 1])
    assert abs(oracle.plaquette(dims, one) - (1 - 6 * (2 - 2 * np.cos(a)) / (18 * V))) < 1e-15


# ------------------------------------------------------------------------------------------------
# sign and size of the step   (eq. 4; R2, R3)
# ------------------------------------------------------------------------------------------------

def test_first_order_gain_in_F():
    """For g = exp(i omega): dF = (1/(12 V)) sum_x Re tr[omega(x) Delta(x)] + O(omega^2).
    With omega = (alpha/2) w this pins the sign of the exponent relative to Delta and the factor alpha/2:
    the literal reading of eq. (4) (R2) would give twice the slope."""
    dims = (4, 4, 4, 4)
    V = 256
    U = inputs.smooth_config(dims, 0.3, 51)
    D, F0, _ = oracle.measure(dims, U)
    w = oracle.accelerate(dims, D)
    slope = np.einsum("...ij,...ji->...", w, D).real.sum() / (12 * V) / 2.0   # dF/dalpha at 0
    assert slope > 0
    for alpha, tol in [(1e-4, 2e-3), (1e-5, 2e-4)]:
        g = oracle.build_g(dims, w, alpha)
        _, F1, _ = oracle.measure(dims, oracle.transform(dims, U, g))
        assert abs((F1 - F0) / alpha / slope - 1) < tol


def test_abelian_contraction_ratio():
    """Small diagonal (abelian) fields: the iteration is linear, Delta -> (1 - alpha p2max/2) Delta
    mode by mode, so theta_{n+1}/theta_n = (1 - 8 alpha)^2 = 0.1296 at alpha = 0.08."""
    dims = (4, 6, 4, 8)
    U = inputs.abelian_config(dims, 1e-4, 61)
    _, Fh, Th = oracle.iterate(dims, U, 0.08, 3)
    for n in range(3):
        assert abs(Th[n + 1] / Th[n] - (1 - 8 * 0.08) ** 2) < 1e-6
    # and for another alpha, to pin the alpha dependence
    _, Fh, Th = oracle.iterate(dims, U, 0.05, 2)
    assert abs(Th[1] / Th[0] - (1 - 8 * 0.05) ** 2) < 1e-6


# ------------------------------------------------------------------------------------------------
# whole iteration  (Algorithm 1)
# ------------------------------------------------------------------------------------------------

def test_pure_gauge_is_driven_to_unit_links():
    dims = (8, 8, 8, 8)
    U = inputs.pure_gauge_config(dims, 71)
    Uf, it, Fh, Th = oracle.fix(dims, U, 0.08, 1e-15, 500)
    assert it < 100 and Th[-1] < 1e-15
    assert abs(Fh[-1] - 1.0) < 1e-13
    # U -> z 1 with z in the centre of SU(3) is also F-maximal only for z = 1: links go to 1, error ~ sqrt(theta)
    assert np.abs(Uf - EYE).max() < 1e-6
    assert np.all(np.diff(Fh) > -1e-15)
    # late-stage contraction equals the linearised closed form (1 - 8 alpha)^2
    assert abs(Th[-1] / Th[-2] - 0.1296) < 2e-3


def test_fix_smooth_config_invariants():
    dims = (4, 6, 4, 6)
    U = inputs.smooth_config(dims, 0.2, 81)
    P0 = oracle.plaquette(dims, U)
    Uf, it, Fh, Th = oracle.fix(dims, U, 0.08, 1e-15, 2000)
    assert 0 < it < 2000 and Th[-1] < 1e-15 and Th[-2] >= 1e-15
    assert np.all(np.diff(Fh) > -1e-15)                            # F non-decreasing (R19)
    late = Th[Th < 0.5]
    assert np.all(np.diff(late) < 0)                               # theta decreasing once below 0.5 (R19)
    assert abs(oracle.plaquette(dims, Uf) - P0) < 1e-13            # gauge invariant
    tol_drift = 1e-15 * (it + 10) * 10                             # R13: links are never re-projected
    assert np.abs(Uf @ dag(Uf) - EYE).max() < tol_drift
    assert np.abs(np.linalg.det(Uf) - 1).max() < tol_drift
    # the returned history is the measure of the returned configuration
    _, F, th = oracle.measure(dims, Uf)
    # (OpenMP combines the per-thread partial sums in arbitrary order: equal up to rounding)
    assert abs(F - Fh[-1]) < 1e-14 and abs(th - Th[-1]) < 1e-12 * th


def test_theta_monotone_without_haar_dressing():
    # h(x) = 1: the start is already close to the gauge; theta falls from iteration 0 (R19 (i))
    dims = (4, 4, 4, 4)
    U = inputs.smooth_config(dims, 0.2, 82, haar=False)
    _, it, Fh, Th = oracle.fix(dims, U, 0.08, 1e-15, 2000)
    assert np.all(np.diff(Th) < 0) and np.all(np.diff(Fh) > -1e-15)


def test_iterate_and_fix_agree_and_count_updates():
    dims = (4, 4, 4, 4)
    U = inputs.smooth_config(dims, 0.2, 83)
    Uf, it, Fh, Th = oracle.fix(dims, U, 0.08, 1e-15, 2000)
    Ui, Fi, Ti = oracle.iterate(dims, U, 0.08, it)
    assert np.array_equal(Ui, Uf)
    assert np.allclose(Fi, Fh, rtol=1e-13, atol=0) and np.allclose(Ti, Th, rtol=1e-12, atol=0)
    # already fixed: zero updates (R11)
    _, it2, _, _ = oracle.fix(dims, Uf, 0.08, 1e-15, 2000)
    assert it2 == 0
    # max_iter cap
    _, it3, _, _ = oracle.fix(dims, U, 0.08, 1e-15, 5)
    assert it3 == 5


def test_accumulated_transformation_carries_U0_to_Un():
    """with G(x) = g_n(x) ... g_1(x) (left multiplication, newest factor first) the
    configuration after n updates is G(x) U0_mu(x) G(x+mu)^dag (eq. 2 composed).  Built here from the oracle's
    single steps; it must reproduce oracle.iterate's configuration, and G must stay in SU(3)."""
    dims = (4, 6, 4, 8)
    U0 = inputs.smooth_config(dims, 0.3, 31, haar=True)
    n = 6
    U = U0.copy()
    G = np.broadcast_to(np.eye(3, dtype=np.complex128), U0.shape[:4] + (3, 3)).copy()
    for _ in range(n):
        D, _, _ = oracle.measure(dims, U)
        g = oracle.build_g(dims, oracle.accelerate(dims, D), 0.08)
        U = oracle.transform(dims, U, g)
        G = g @ G
    U_n, _, _ = oracle.iterate(dims, U0, 0.08, n)
    assert np.max(np.abs(U - U_n)) < 1e-13
    assert np.max(np.abs(oracle.transform(dims, U0, G) - U_n)) < 1e-13
    # the other order of the product is NOT the transformation (the g_k do not commute)
    assert np.max(np.abs(G @ np.conj(np.swapaxes(G, -1, -2)) - np.eye(3))) < 1e-14
    assert np.max(np.abs(np.linalg.det(G) - 1)) < 1e-14


def _phase_minus_one(dims, mu):
    """exp(-2 pi i k_mu / L_mu) - 1 on the (kt, kz, ky, kx) grid."""
    L = dims[mu]
    ph = np.exp(-2j * np.pi * np.arange(L) / L) - 1.0
    shape = [1, 1, 1, 1]
    shape[3 - mu] = L
    return ph.reshape(shape + [1, 1])


def test_gluon_field_divergence_identity_and_symmetries():
    """NEXT-2: A_mu(k).  From eq. 5, F[Delta](k) = sum_mu (exp(-2 pi i k_mu/L_mu) - 1) A_mu(k) for ANY configuration
    -- it ties the new function to the pinned Delta and the pinned DFT (sign of the shift, site convention,
    normalisation).  A_mu(x) hermitian traceless  =>  A_mu(-k) = A_mu(k)^dag, tr A_mu(k) = 0."""
    dims = (4, 6, 2, 8)
    U = inputs.smooth_config(dims, 0.4, 58, haar=True)
    Delta, _, _ = oracle.measure(dims, U)
    lhs = np.stack([oracle.dft4d(dims, np.ascontiguousarray(Delta[..., i, j]), -1) for i in range(3) for j in range(3)],
                   axis=-1).reshape(Delta.shape)
    A = [oracle.gluon_field(dims, U, mu) for mu in range(4)]
    rhs = sum(_phase_minus_one(dims, mu) * A[mu] for mu in range(4))
    assert np.max(np.abs(lhs - rhs)) < 1e-11 * max(1.0, np.max(np.abs(lhs)))
    for mu in range(4):
        Am = A[mu]
        minus_k = np.roll(Am[::-1, ::-1, ::-1, ::-1], 1, axis=(0, 1, 2, 3))          # A(-k)
        assert np.max(np.abs(minus_k - np.conj(np.swapaxes(Am, -1, -2)))) < 1e-11
        assert np.max(np.abs(np.trace(Am, axis1=-2, axis2=-1))) < 1e-11
    # k = 0 is the plain lattice sum; constant links give a single non-zero mode
    const = np.broadcast_to(U[0, 0, 0, 0], U.shape).copy()
    Ac = oracle.gluon_field(dims, const, 1)
    assert np.max(np.abs(Ac.reshape(-1, 3, 3)[1:])) < 1e-10 and np.max(np.abs(Ac[0, 0, 0, 0])) > 1.0


def test_gluon_field_is_transverse_in_landau_gauge():
    """What the gauge fixing is for: after Algorithm 1 has driven theta below 1e-15 the lattice divergence of the
    gluon field vanishes mode by mode, sum_mu (exp(-2 pi i k_mu/L_mu) - 1) A_mu(k) = 0, while before it does not."""
    dims = (4, 4, 4, 8)
    U = inputs.smooth_config(dims, 0.3, 59, haar=True)
    V = int(np.prod(dims))

    def div(Ucfg):
        return sum(_phase_minus_one(dims, mu) * oracle.gluon_field(dims, Ucfg, mu) for mu in range(4))

    before = np.abs(div(U)).max()
    Ufix, it, F, th = oracle.fix(dims, U, 0.08, 1e-15, 2000)
    after = div(Ufix)
    assert th[-1] < 1e-15 and before > 1.0
    # Parseval: sum_k |F[Delta](k)|^2 = V sum_x |Delta(x)|^2 = V * 3 V theta
    assert abs(np.sum(np.abs(after) ** 2) - 3.0 * V * V * th[-1]) < 1e-3 * 3.0 * V * V * th[-1] + 1e-20
    assert np.abs(after).max() < np.sqrt(3.0 * V * V * 1e-15)
