"""Pins of the thermalisation oracle (oracle/lgf_heatbath_oracle.c; R24-R27)
against what the mathematics fixes -- none of them re-uses the oracle's own formulas:
  staples      : sum over links of Re tr[U A] = 4 x (sum over plaquettes), with the separately pinned plaquette;
                 one staple sum rebuilt with numpy from shifted link fields
  x0 sampler   : (Creutz below a = 2, Kennedy-Pendleton above) <x0> = I_2(a)/I_1(a) and <x0^2> = 1 - 3 I_2(a)/(a I_1(a)) for the density exp(a x0) sqrt(1-x0^2),
                 isotropy of the direction, unit norm
  heat bath    : links stay in SU(3); strong coupling <P> -> beta/18; weak coupling (equipartition over the
                 24V - ... quadratic modes) <1 - P> -> 2/beta; the stream is counter-based (a split run is the
                 same run); odd extents are refused
"""
import numpy as np
import pytest
from scipy.special import iv

import oracle
from paper_1206_0675_b200 import inputs


def _dag(M):
    return np.conj(np.swapaxes(M, -1, -2))


def _shift(F, mu, d):
    """F(x + d mu^) on the (Lt, Lz, Ly, Lx, ...) grid."""
    return np.roll(F, -d, axis=3 - mu)


def test_staples_sum_to_the_plaquette():
    dims = (4, 6, 2, 4)
    U = inputs.hot_config(dims, 11)
    A = oracle.hb_staples(dims, U)
    V = int(np.prod(dims))
    total = np.einsum("...ij,...ji->...", U, A).real.sum()
    assert abs(total / (4 * 18 * V) - oracle.plaquette(dims, U)) < 1e-14      # each plaquette has 4 links


@pytest.mark.parametrize("mu", [0, 1, 2, 3])
def test_staple_sum_numpy_brute_force(mu):
    dims = (4, 2, 6, 4)
    U = inputs.hot_config(dims, 12)
    A = oracle.hb_staples(dims, U)
    ref = np.zeros_like(U[..., 0, :, :])
    Um = U[..., mu, :, :]
    for nu in range(4):
        if nu == mu:
            continue
        Un = U[..., nu, :, :]
        ref += _shift(Un, mu, 1) @ _dag(_shift(Um, nu, 1)) @ _dag(Un)                       # upper staple
        ref += _dag(_shift(_shift(Un, mu, 1), nu, -1)) @ _dag(_shift(Um, nu, -1)) @ _shift(Un, nu, -1)   # lower
    assert np.max(np.abs(A[..., mu, :, :] - ref)) < 1e-13


@pytest.mark.parametrize("a", [0.05, 0.2, 0.7, 1.99, 2.0, 3.0, 12.0, 40.0])
def test_kennedy_pendleton_moments(a):
    n = 200000
    X, att = oracle.hb_kp_sample(a, 2024, n)
    assert np.max(np.abs((X ** 2).sum(axis=1) - 1.0)) < 1e-14
    m1 = iv(2, a) / iv(1, a)                       # <x0> for exp(a x) sqrt(1 - x^2) on [-1, 1]
    m2 = 1.0 - 3.0 * iv(2, a) / (a * iv(1, a))     # <x0^2>
    s1 = np.sqrt((m2 - m1 * m1) / n)
    assert abs(X[:, 0].mean() - m1) < 5 * s1
    assert abs((X[:, 0] ** 2).mean() - m2) < 5 * np.sqrt(np.var(X[:, 0] ** 2) / n)
    # direction uniform on the sphere of radius sqrt(1 - x0^2)
    r2 = 1.0 - (X[:, 0] ** 2).mean()
    for i in (1, 2, 3):
        assert abs(X[:, i].mean()) < 5 * np.sqrt(r2 / 3 / n)
        assert abs((X[:, i] ** 2).mean() - r2 / 3) < 5 * np.sqrt(np.var(X[:, i] ** 2) / n)
    # bounded attempts must not bias the draw: no draw may exhaust them (Creutz below a = 2, KP above)
    assert att.min() >= 1 and att.max() < 32 and att.mean() < 2.0


def test_heatbath_keeps_links_in_su3_and_is_counter_based():
    dims = (4, 4, 4, 4)
    U0 = inputs.hot_config(dims, 5)
    U2 = oracle.heatbath(dims, U0, 5.7, 99, 0, 2)
    U40 = oracle.heatbath(dims, U2, 5.7, 99, 2, 38)          # re-projected after every update (R26): no drift
    assert np.max(np.abs(U40 @ _dag(U40) - np.eye(3))) < 5e-15
    assert np.max(np.abs(U2 @ _dag(U2) - np.eye(3))) < 1e-14
    assert np.max(np.abs(np.linalg.det(U2) - 1)) < 1e-14
    assert not np.allclose(U2, U0)
    U1 = oracle.heatbath(dims, U0, 5.7, 99, 0, 1)
    assert np.array_equal(oracle.heatbath(dims, U1, 5.7, 99, 1, 1), U2)      # a split run is the same run
    assert not np.array_equal(oracle.heatbath(dims, U1, 5.7, 99, 0, 1), U2)  # the sweep number selects the stream
    assert not np.array_equal(oracle.heatbath(dims, U0, 5.7, 100, 0, 2), U2)
    with pytest.raises(ValueError):
        oracle.heatbath((4, 4, 3, 4), inputs.hot_config((4, 4, 3, 4), 5), 5.7, 1, 0, 1)


def _mean_plaquette(dims, U, beta, seed, therm, meas):
    U = oracle.heatbath(dims, U, beta, seed, 0, therm)
    vals = []
    for k in range(meas):
        U = oracle.heatbath(dims, U, beta, seed, therm + k, 1)
        vals.append(oracle.plaquette(dims, U))
    return float(np.mean(vals)), float(np.std(vals) / np.sqrt(meas))


def test_strong_coupling_limit():
    """<P> = beta/18 + O(beta^2) for SU(3) (leading order of the strong-coupling expansion)."""
    dims, beta = (6, 6, 6, 6), 0.3
    P, err = _mean_plaquette(dims, inputs.hot_config(dims, 1), beta, 17, 5, 40)
    assert abs(P - beta / 18.0) < 5 * max(err, 2e-4) + (beta / 18.0) ** 2 * 3      # room for the next order


def test_weak_coupling_limit():
    """<1 - P> = 2/beta at large beta: (8 x 4V - 8V gauge directions) quadratic modes at 1/2 each = 12V = beta 6V <1-P>."""
    dims, beta = (4, 4, 4, 4), 80.0
    cold = np.broadcast_to(np.eye(3, dtype=np.complex128), (4, 4, 4, 4, 4, 3, 3)).copy()
    P, err = _mean_plaquette(dims, cold, beta, 23, 40, 60)
    assert abs((1.0 - P) * beta / 2.0 - 1.0) < 0.06          # finite-volume zero modes and O(1/beta) terms: a few per cent


def test_overrelaxation_conserves_the_action_and_moves_the_links():
    """R28: every overrelaxation step leaves Re tr[U A] unchanged, so the plaquette is conserved to rounding by
    whole sweeps -- on a rough configuration, where the links move by O(1)."""
    dims = (4, 6, 4, 4)
    U0 = oracle.heatbath(dims, inputs.hot_config(dims, 8), 5.7, 3, 0, 3)
    P0 = oracle.plaquette(dims, U0)
    U1 = oracle.overrelax(dims, U0, 1)
    U3 = oracle.overrelax(dims, U1, 2)
    assert abs(oracle.plaquette(dims, U1) - P0) < 1e-14 and abs(oracle.plaquette(dims, U3) - P0) < 1e-14
    assert np.mean(np.abs(U1 - U0)) > 0.1                      # not a small move
    assert np.max(np.abs(U3 @ _dag(U3) - np.eye(3))) < 5e-15
    assert np.array_equal(oracle.overrelax(dims, U0, 3), U3)   # deterministic, no random numbers
    with pytest.raises(ValueError):
        oracle.overrelax((4, 4, 3, 4), inputs.hot_config((4, 4, 3, 4), 5), 1)


def test_heatbath_with_overrelaxation_keeps_the_equilibrium():
    """Mixing in microcanonical sweeps must not move the equilibrium: same weak-coupling limit 1 - P = 2/beta."""
    dims, beta = (4, 4, 4, 4), 80.0
    U = np.broadcast_to(np.eye(3, dtype=np.complex128), (4, 4, 4, 4, 4, 3, 3)).copy()
    vals = []
    for k in range(70):
        U = oracle.overrelax(dims, oracle.heatbath(dims, U, beta, 31, k, 1), 2)
        if k >= 25:
            vals.append(oracle.plaquette(dims, U))
    assert abs((1.0 - np.mean(vals)) * beta / 2.0 - 1.0) < 0.06
