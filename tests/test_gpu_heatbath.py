"""Parity of lgf_thermalize (csrc/lgf_heatbath.cu) with the thermalisation oracle on the same seeded inputs
(R24-R27).  The update is a deterministic function of the configuration and
of counter-based uniforms, so after a few sweeps the two sides agree link by link up to rounding; Monte-Carlo
dynamics amplifies rounding differences over many sweeps, so long runs are compared through the plaquette."""
import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

pytestmark = pytest.mark.gpu

# Tolerances (fp64).  One sweep from identical inputs: 1e-12 (staples are sums of 6 products of O(1) numbers,
# and the new link follows the DIRECTION r/|r| of a 2x2 block of U A, which divides the rounding error by |r|;
# measured max 7e-13 at beta = 0.3, 3e-14 at beta = 5.7, 9e-15 at beta = 80).  Each further sweep multiplies the
# difference of its inputs by the sensitivity of the Monte-Carlo map itself, measured on B200 against the oracle
# (8^4, whole error distribution, no link ever off by more than 1e-6, i.e. no accept/reject decision differs):
# x40 per sweep at beta = 0.3, where the links are nearly random and |r| is often small, x1.7 at beta >= 5.7.
# The amplification of a single link goes like 1/|r| and P(|r| < eps) ~ eps^4, so the MAXIMUM over 10^4-10^5
# links is a heavy-tailed extreme value with no fixed bound (5.05e-11 seen on 12 x 6 x 16 x 4); after the first
# sweep the tests therefore bound the 99.9 % quantile and the median, and require of the maximum only what
# separates rounding from a differing accept / reject decision (which changes a link by O(1)).
TOL1 = 1e-12
NO_FLIP = 1e-6


def growth(beta):
    return 50.0 if beta < 1.0 else 3.0


@pytest.fixture(scope="module")
def lgf():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_1206_0675_b200 import binding

    binding.load()
    return binding


def _dev(a, prec):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.complex128 if prec == 8 else torch.complex64).cuda()


def _links(ctx, like):
    import torch

    return ctx.get_links(torch.empty_like(like)).cpu().numpy().astype(np.complex128)


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 6, 16, 4), (4, 2, 2, 6)])
@pytest.mark.parametrize("beta", [0.3, 5.7, 80.0])          # Creutz branch, both branches, Kennedy-Pendleton branch
@pytest.mark.parametrize("storage", [18, 12])
def test_sweeps_match_the_oracle_fp64(lgf, dims, beta, storage):
    U0 = inputs.hot_config(dims, 321)
    U1 = oracle.heatbath(dims, U0, beta, 77, 0, 1)
    U2 = oracle.heatbath(dims, U1, beta, 77, 1, 1)
    with lgf.Context(dims, 8, storage) as ctx:
        d = _dev(U0, 8)
        ctx.set_links(d)
        ctx.thermalize(beta, 1, 77)
        assert np.max(np.abs(_links(ctx, d) - U1)) < 1e-12
        ctx.thermalize(beta, 1, 77)                           # continues the stream: sweep number 1
        out = _links(ctx, d)
        err = np.abs(out - U2)
        assert np.quantile(err, 0.999) < TOL1 * growth(beta)
        assert np.median(err) < 1e-12                           # the bulk stays at rounding level
        assert err.max() < NO_FLIP                              # no decision differs anywhere
        _, _, P = ctx.measure()
    assert abs(P - oracle.plaquette(dims, U2)) < 1e-12
    assert np.max(np.abs(out @ np.conj(np.swapaxes(out, -1, -2)) - np.eye(3))) < 1e-13


def test_one_sweep_matches_the_oracle_fp32(lgf):
    """fp32 link storage: the arithmetic is double, the links are rounded to float between class passes."""
    dims = (8, 8, 8, 8)
    U0 = inputs.hot_config(dims, 322).astype(np.complex64).astype(np.complex128)
    U1 = oracle.heatbath(dims, U0, 5.7, 78, 0, 1)
    with lgf.Context(dims, 4, 18) as ctx:
        d = _dev(U0, 4)
        ctx.set_links(d)
        ctx.thermalize(5.7, 1, 78)
        out = _links(ctx, d)
    err = np.abs(out - U1).max(axis=(-1, -2))
    # a link whose accept / reject decision sat within float rounding of the boundary would differ by O(1)
    assert (err > 1e-5).sum() == 0, "%d of %d links differ" % ((err > 1e-5).sum(), err.size)


def test_split_runs_and_state_reset(lgf):
    import torch

    dims = (8, 8, 8, 8)
    U0 = inputs.hot_config(dims, 323)
    with lgf.Context(dims, 8, 18) as ctx:
        d = _dev(U0, 8)
        ctx.set_links(d)
        ctx.thermalize(6.0, 3, 5)
        a = ctx.get_links(torch.empty_like(d)).clone()
        ctx.set_links(d)
        ctx.thermalize(6.0, 1, 5)
        ctx.thermalize(6.0, 2, 5)
        b = ctx.get_links(torch.empty_like(d))
        assert torch.equal(a, b)                                  # bit-identical whatever the split
        ctx.set_links(d)
        ctx.thermalize(6.0, 3, 6)
        assert not torch.equal(a, ctx.get_links(torch.empty_like(d)))
        # thermalising is loading a new configuration: history and counters start again
        ctx.iterate(0.08, 2)
        assert ctx.history_length() == 3
        ctx.thermalize(6.0, 1, 5)
        assert ctx.history_length() == 0 and ctx.iterations() == 0
        ctx.iterate(0.08, 1)
        Fh, Th = ctx.history()
        F, th, _ = ctx.measure(plaquette=False)
        assert len(Fh) == 2 and abs(Fh[-1] - F) < 1e-13 * abs(F)
    with lgf.Context((4, 4, 6, 4), 8, 18) as ctx:
        with pytest.raises(lgf.LgfError) as e:
            ctx.thermalize(6.0, 1, 1)
        assert e.value.code == lgf.LGF_ESTATE                      # nothing loaded
    with lgf.Context((4, 3, 4, 4), 8, 18) as ctx:
        ctx.set_links(_dev(inputs.hot_config((4, 3, 4, 4), 1), 8))
        with pytest.raises(lgf.LgfError) as e:
            ctx.thermalize(6.0, 1, 1)
        assert e.value.code == lgf.LGF_EINVAL                      # odd extent


def test_five_sweeps_and_plaquette(lgf):
    """Five sweeps from a cold start at beta = 6: still link-by-link agreement, and the same plaquette."""
    dims = (8, 8, 8, 8)
    cold = np.broadcast_to(np.eye(3, dtype=np.complex128), (8, 8, 8, 8, 4, 3, 3)).copy()
    U5 = oracle.heatbath(dims, cold, 6.0, 9, 0, 5)
    with lgf.Context(dims, 8, 18) as ctx:
        d = _dev(cold, 8)
        ctx.set_links(d)
        ctx.thermalize(6.0, 5, 9)
        out = _links(ctx, d)
        _, _, P = ctx.measure()
    err = np.abs(out - U5)
    assert np.quantile(err, 0.999) < TOL1 * growth(6.0) ** 4 and err.max() < NO_FLIP
    assert abs(P - oracle.plaquette(dims, U5)) < 1e-12
    assert 0.5 < P < 0.75                                          # between the hot and the cold start


@pytest.mark.parametrize("prec,storage", [(8, 12), (8, 18), (4, 12)])
def test_many_sweeps_stay_in_su3(lgf, prec, storage):
    """Regression: with 12-real storage the rebuilt third row fed the norm error of rows 0, 1 back through the
    (0,2) and (1,2) subgroup updates -- 7.5e-7 off SU(3) after 100 sweeps, overflow before 300.  The link is
    now re-projected after every update (R26): the deviation must stay at rounding level however long the run."""
    import torch

    dims = (8, 8, 8, 8)
    cdt = torch.complex128 if prec == 8 else torch.complex64
    cold = torch.zeros((8, 8, 8, 8, 4, 3, 3), dtype=cdt, device="cuda")
    for i in range(3):
        cold[..., i, i] = 1
    with lgf.Context(dims, prec, storage) as ctx:
        ctx.set_links(cold)
        ctx.thermalize(6.0, 400, 11)
        out = ctx.get_links(torch.empty_like(cold)).to(torch.complex128)
        _, _, P = ctx.measure()
    dev = float((out @ out.conj().transpose(-1, -2) - torch.eye(3, dtype=torch.complex128, device="cuda")).abs().max())
    assert bool(torch.isfinite(torch.view_as_real(out)).all())
    assert dev < (1e-14 if prec == 8 else 1e-6)
    assert 0.55 < P < 0.64            # thermalised at beta = 6 (8^4: large fluctuations around 0.594)


@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18)])
def test_overrelaxation_matches_the_oracle_and_conserves_the_action(lgf, prec, storage):
    """R28 on the CUDA side: one and two sweeps against the oracle, the plaquette conserved, history reset."""
    dims = (8, 4, 6, 8)
    U0 = oracle.heatbath(dims, inputs.hot_config(dims, 41), 5.7, 3, 0, 2)
    if prec == 4:
        U0 = U0.astype(np.complex64).astype(np.complex128)
    U1 = oracle.overrelax(dims, U0, 1)
    U2 = oracle.overrelax(dims, U1, 1)
    with lgf.Context(dims, prec, storage) as ctx:
        d = _dev(U0, prec)
        ctx.set_links(d)
        _, _, P0 = ctx.measure()
        ctx.iterate(0.08, 1)
        ctx.set_links(d)
        ctx.overrelax(1)
        assert ctx.history_length() == 0
        e1 = np.abs(_links(ctx, d) - U1)
        ctx.overrelax(1)
        e2 = np.abs(_links(ctx, d) - U2)
        _, _, P2 = ctx.measure()
        ctx.thermalize(5.7, 1, 3)                     # overrelaxation consumes no random numbers: this is sweep 0
        e3 = np.abs(_links(ctx, d) - oracle.heatbath(dims, U2, 5.7, 3, 0, 1))
    if prec == 8:
        assert e1.max() < TOL1 and np.quantile(e2, 0.999) < TOL1 * growth(5.7) and e2.max() < NO_FLIP
        assert np.quantile(e3, 0.999) < TOL1 * growth(5.7) ** 2 and e3.max() < NO_FLIP
        assert abs(P2 - P0) < 1e-13
    else:
        assert e1.max() < 1e-5 and e2.max() < 1e-4
        assert abs(P2 - P0) < 2e-6


@pytest.mark.parametrize("prec,storage", [(8, 18), (4, 12)])
def test_tiled_thread_order_is_bit_identical(lgf, prec, storage):
    """lgf_tune("hb_tz"): the (z, t)-tiled order in which the threads walk the lattice (used automatically when a
    t slice exceeds L2, i.e. at 64^4) only changes WHICH thread updates a site; sites, staples and random numbers
    are the same, so heat-bath and overrelaxation sweeps must come out bit for bit as in the plain order."""
    import torch

    dims = (8, 4, 8, 6)
    U0 = inputs.hot_config(dims, 77)
    res = []
    for tz in (8, 2, 4, 1):                                  # 8 = Lz: the plain order
        with lgf.Context(dims, prec, storage) as ctx:
            ctx.tune("hb_tz", tz)
            d = _dev(U0, prec)
            ctx.set_links(d)
            ctx.thermalize(5.9, 2, 13)
            ctx.overrelax(1)
            ctx.thermalize(5.9, 1, 13)
            res.append(ctx.get_links(torch.empty_like(d)).clone())
    for r in res[1:]:
        assert torch.equal(res[0], r)
    if prec == 8:
        ref = oracle.heatbath(dims, oracle.overrelax(dims, oracle.heatbath(dims, U0, 5.9, 13, 0, 2), 1), 5.9, 13, 2, 1)
        err = np.abs(res[1].cpu().numpy() - ref)
        assert np.quantile(err, 0.999) < TOL1 * growth(5.9) ** 3 and err.max() < NO_FLIP
