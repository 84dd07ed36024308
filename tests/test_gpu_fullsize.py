"""Parity of the CUDA path with the oracle at BASELINE.json's FULL sizes, in the launch configuration
bench.py times (default plan, default tuning): C3 = 32^4 (the bench workload), C4 = 24^3 x 48, C5 = 64^4.
The oracle is affordable here: one 32^4 iteration takes it about a second, one 64^4 iteration about half a
minute.  Tolerances are north_star's (see tests/test_gpu_parity.py)."""
import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

ALPHA = 0.08
TOL = {8: dict(scalar=1e-12, links=1e-11), 4: dict(scalar=1e-5, links=2e-5)}


@pytest.fixture(scope="module")
def lgf():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_1206_0675_b200 import binding

    binding.load()
    return binding


def _run(lgf, dims, U, prec, storage, n):
    import torch

    cdt = torch.complex128 if prec == 8 else torch.complex64
    with lgf.Context(dims, prec, storage, stream=torch.cuda.current_stream()) as ctx:
        d = torch.from_numpy(U).to(cdt).cuda()
        ctx.set_links(d)
        ctx.iterate(ALPHA, n)
        Fh, Th = ctx.history()
        _, _, P = ctx.measure()
        out = ctx.get_links(torch.empty_like(d)).cpu().numpy().astype(np.complex128)
    return Fh, Th, P, out


@pytest.mark.parametrize("cfg", ["C3", "C4"])
def test_trajectory_20_full_size(lgf, config_cache, cfg):
    """(F_n, theta_n), n = 0..20, and ALL links after 20 iterations, every precision x storage variant."""
    dims = inputs.CONFIGS[cfg]["dims"]
    U = config_cache(cfg)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    P_o = oracle.plaquette(dims, U)
    for prec, storage in ((8, 18), (8, 12), (4, 18), (4, 12)):
        Fh, Th, P, out = _run(lgf, dims, U, prec, storage, 20)
        tol = TOL[prec]
        what = "%s prec=%d storage=%d" % (cfg, prec, storage)
        assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"], what
        assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"], what
        assert np.max(np.abs(out - U_o)) < tol["links"], what
        assert abs(P - P_o) < (1e-13 if prec == 8 else 1e-6), what


@pytest.mark.parametrize("cfg", ["C3", "C4"])
def test_iterations_to_convergence_full_size(lgf, config_cache, cfg):
    """Algorithm 1 to theta < 1e-15 (fp64): iteration count within 2 % of the oracle's, same final F, the
    plaquette unchanged, links still in SU(3) (R13 tolerance)."""
    import torch

    dims = inputs.CONFIGS[cfg]["dims"]
    U = config_cache(cfg)
    U_o, it_o, F_o, T_o = oracle.fix(dims, U, ALPHA, 1e-15, 2000)
    assert 0 < it_o < 2000 and T_o[-1] < 1e-15
    with lgf.Context(dims, 8, 18, stream=torch.cuda.current_stream()) as ctx:
        d = torch.from_numpy(U).to(torch.complex128).cuda()
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        Fh, Th = ctx.history()
        F, th, P = ctx.measure()
        out = d.cpu().numpy()
    assert abs(it - it_o) <= max(1, int(0.02 * it_o))
    assert len(Fh) == it + 1 and Th[-1] < 1e-15 and (it == 0 or Th[-2] >= 1e-15)
    n = min(it, it_o)
    assert np.max(np.abs(Fh[:n + 1] - F_o[:n + 1]) / np.abs(F_o[:n + 1])) < 1e-11
    assert np.all(np.diff(Fh) > -1e-14)                                   # F non-decreasing (R19)
    assert abs(P - oracle.plaquette(dims, U)) < 1e-13
    assert np.abs(out @ np.conj(np.swapaxes(out, -1, -2)) - np.eye(3)).max() < 1e-15 * (it + 10) * 10
    if it == it_o:
        assert np.max(np.abs(out - U_o)) < 1e-10


def test_c5_hot_start_one_iteration(lgf):
    """64^4 hot start (16.8 M sites, 9.7 GB of fp64 links): F and theta before and after one update and ALL
    links after it against the oracle; then a few more iterations for the invariants (F non-decreasing,
    plaquette unchanged)."""
    import torch

    dims = inputs.CONFIGS["C5"]["dims"]
    seed = inputs.CONFIGS["C5"]["seed"]
    d = inputs.hot_config_torch(dims, seed, device="cuda")
    U = d.cpu().numpy()
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 1)
    del U
    for prec, storage in ((8, 18), (8, 12), (4, 18), (4, 12)):      # every variant the bench times at 64^4
        cdt = torch.complex128 if prec == 8 else torch.complex64
        with lgf.Context(dims, prec, storage, stream=torch.cuda.current_stream()) as ctx:
            dd = d.to(cdt)
            ctx.set_links(dd)
            _, _, P0 = ctx.measure()
            ctx.iterate(ALPHA, 1)
            Fh, Th = ctx.history()
            out = ctx.get_links(torch.empty_like(dd))
            err = float((out.to(torch.complex128) - torch.from_numpy(U_o).cuda()).abs().max())
            del out
            ctx.iterate(ALPHA, 4)
            Fh5, Th5 = ctx.history()
            _, _, P5 = ctx.measure()
            del dd
        torch.cuda.empty_cache()
        tol = TOL[prec]
        assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
        assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
        assert err < tol["links"]
        assert np.all(np.diff(Fh5) > 0)
        assert abs(P5 - P0) < (1e-13 if prec == 8 else 1e-6)


def test_section_8f_rows_at_full_size(lgf, config_cache):
    """The SURVEY.md 8(f) rows at the bench lattice (32^4, fp64 / 18-real, default plan): two heat-bath sweeps and
    one overrelaxation sweep link by link against the thermalisation oracle; then, on the smooth C3 configuration,
    five updates with the accumulated transformation tracked -- G against the product of the oracle's g fields,
    G U0 G(x+mu)^dag against the CUDA path's own links -- and the gluon field A_t(k) against the oracle's."""
    import torch

    dims = inputs.CONFIGS["C3"]["dims"]
    V = int(np.prod(dims))
    # -- thermalisation (NEXT-1)
    hot = inputs.hot_config_torch(dims, 4242, device="cuda")
    U0 = hot.cpu().numpy()
    U1 = oracle.heatbath(dims, U0, 6.0, 55, 0, 1)
    U2 = oracle.overrelax(dims, oracle.heatbath(dims, U1, 6.0, 55, 1, 1), 1)
    with lgf.Context(dims, 8, 18, stream=torch.cuda.current_stream()) as ctx:
        ctx.set_links(hot)
        ctx.thermalize(6.0, 1, 55)
        e1 = np.abs(ctx.get_links(torch.empty_like(hot)).cpu().numpy() - U1)
        ctx.thermalize(6.0, 1, 55)
        ctx.overrelax(1)
        e2 = np.abs(ctx.get_links(torch.empty_like(hot)).cpu().numpy() - U2)
        _, _, P = ctx.measure()
    assert e1.max() < 1e-12
    assert np.quantile(e2, 0.999) < 1e-12 * 3.0 ** 2 and e2.max() < 1e-6        # see tests/test_gpu_heatbath.py
    assert abs(P - oracle.plaquette(dims, U2)) < 1e-12
    del hot, U0, U1, U2, e1, e2
    # -- accumulated transformation and gluon field (NEXT-2)
    U = config_cache("C3")
    Uo, G = U.copy(), np.broadcast_to(np.eye(3, dtype=np.complex128), U.shape[:4] + (3, 3)).copy()
    for _ in range(5):
        D, _, _ = oracle.measure(dims, Uo)
        g = oracle.build_g(dims, oracle.accelerate(dims, D), ALPHA)
        Uo = oracle.transform(dims, Uo, g)
        G = g @ G
    with lgf.Context(dims, 8, 18, stream=torch.cuda.current_stream()) as ctx:
        ctx.track_transform(True)
        d = torch.from_numpy(U).cuda()
        ctx.set_links(d)
        ctx.iterate(ALPHA, 5)
        Gd = ctx.get_transform(torch.empty(U.shape[:4] + (3, 3), dtype=torch.complex128, device="cuda")).cpu().numpy()
        out = ctx.get_links(torch.empty_like(d)).cpu().numpy()
        At = ctx.gluon_field(3, torch.empty(U.shape[:4] + (3, 3), dtype=torch.complex128, device="cuda")).cpu().numpy()
    assert np.max(np.abs(Gd - G)) < 1e-11 and np.max(np.abs(out - Uo)) < 1e-11
    assert np.max(np.abs(oracle.transform(dims, U, Gd) - out)) < 1e-11
    ref = oracle.gluon_field(dims, out, 3)
    assert np.max(np.abs(At - ref)) < 1e-12 * np.max(np.abs(ref))
    assert V == 32 ** 4
