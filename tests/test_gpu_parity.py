"""Parity of the CUDA path (through the C ABI of liblgf.so) with the CPU oracle, element by element
on the same seeded inputs.  Tolerances are those BASELINE.json's north_star states:
  per-iteration F and theta over the first 20 iterations: relative 1e-12 (fp64) / 1e-5 (fp32)
  links after 20 iterations: max abs 1e-11 (fp64) / 2e-5 (fp32)
  iterations to theta < 1e-15 (fp64): within 2 % of the oracle's count
Every test here needs a GPU (-m gpu)."""
import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

pytestmark = pytest.mark.gpu

ALPHA = 0.08
TOL = {8: dict(scalar=1e-12, links=1e-11, field=1e-12), 4: dict(scalar=1e-5, links=2e-5, field=2e-5)}


@pytest.fixture(scope="module")
def lgf():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_1206_0675_b200 import binding

    binding.load()
    return binding


def to_dev(a, prec):
    import torch

    cdt = torch.complex128 if prec == 8 else torch.complex64
    return torch.from_numpy(np.ascontiguousarray(a)).to(cdt).cuda()


def to_np(t):
    return t.cpu().numpy().astype(np.complex128)


def site_shape(dims):
    return (dims[3], dims[2], dims[1], dims[0])


def random_herm_field(dims, seed):
    """Seeded hermitian traceless 3x3 field (input generator only: no method arithmetic)."""
    V = int(np.prod(dims))
    c = inputs.normals(seed, 7, 0, V * 8).reshape(V, 8).astype(np.complex128)
    H = np.einsum("na,aij->nij", c, inputs.gell_mann())
    return np.ascontiguousarray(H.reshape(site_shape(dims) + (3, 3)))


SMALL = [("C1", (8, 8, 8, 8)), ("mixed", (12, 6, 16, 4)), ("odd", (3, 24, 2, 48))]
VARIANTS = [(8, 18), (8, 12), (4, 18), (4, 12)]


def small_config(name, dims):
    if name == "C1":
        return inputs.make_config("C1")
    return inputs.smooth_config(dims, 0.25, 4242 + len(name), haar=True)


@pytest.mark.parametrize("name,dims", SMALL)
@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_delta_F_theta(lgf, name, dims, prec, storage):
    """a1: Delta(x) element by element, F and theta (eqs. 3, 5-7)."""
    import torch

    U = small_config(name, dims)
    D_o, F_o, th_o = oracle.measure(dims, U)
    with lgf.Context(dims, prec, storage) as ctx:
        ctx.set_links(to_dev(U, prec))
        F, th = ctx.step_delta()
        out = torch.empty(site_shape(dims) + (3, 3), dtype=torch.complex128 if prec == 8 else torch.complex64,
                          device="cuda")
        D = to_np(ctx.get_field(out))
    tol = TOL[prec]
    assert np.max(np.abs(D - D_o)) < tol["field"] * max(1.0, np.max(np.abs(D_o)))
    assert abs(F - F_o) <= tol["scalar"] * abs(F_o)
    assert abs(th - th_o) <= tol["scalar"] * abs(th_o)


ACC_DIMS = [(8, 8, 8, 8), (12, 6, 16, 4), (3, 24, 2, 48), (16, 16, 16, 16), (32, 8, 64, 4), (8, 8, 24, 48),
            (24, 24, 24, 48), (32, 32, 16, 16), (64, 64, 8, 8), (8, 8, 64, 64), (16, 16, 32, 32), (24, 24, 8, 8),
            (32, 32, 32, 32), (64, 64, 16, 16), (16, 16, 64, 64), (16, 16, 16, 32), (32, 32, 32, 64)]


@pytest.mark.parametrize("dims", ACC_DIMS)
@pytest.mark.parametrize("prec", [8, 4])
@pytest.mark.parametrize("plan", ["reg", "reg2", "reg2_bulk", "two_axis", "axis"])
def test_accelerate(lgf, dims, prec, plan):
    """a2-a4: w = F^-1 (16/p^2) F Delta / V against the oracle's naive separable DFT, with each FFT
    plan: register-line sweeps with one and with two threads per line, shared-memory two-axis sweeps
    (where the lattice allows them; the planner falls back otherwise) and one pass per axis."""
    import torch

    D = random_herm_field(dims, 99)
    D -= D.mean(axis=(0, 1, 2, 3), keepdims=True)        # like a real Delta: zero lattice sum
    w_o = oracle.accelerate(dims, D)
    with lgf.Context(dims, prec, 18) as ctx:
        ctx.tune("fft_reg", int(plan == "reg"))
        ctx.tune("fft_reg2", int(plan in ("reg2", "reg2_bulk")))
        ctx.tune("fft_bulk", int(plan == "reg2_bulk"))       # (x, y) planes on and off chip by cp.async.bulk + mbarrier
        ctx.tune("fft_two_axis", int(plan != "axis"))
        if plan == "axis":
            assert ctx.fft_passes() == 7
        ctx.set_field(to_dev(D, prec))
        ctx.step_accelerate()
        out = torch.empty(site_shape(dims) + (3, 3), dtype=torch.complex128 if prec == 8 else torch.complex64,
                          device="cuda")
        w = to_np(ctx.get_field(out))
    scale = np.max(np.abs(w_o))
    assert np.max(np.abs(w - w_o)) < (1e-12 if prec == 8 else 2e-5) * scale


@pytest.mark.parametrize("dims,passes", [((32, 32, 32, 32), 3), ((24, 24, 24, 48), 3), ((8, 8, 8, 8), 3), ((16, 16, 16, 32), 3),
                                         ((12, 6, 16, 4), 7), ((16, 16, 12, 6), 5), ((6, 12, 32, 32), 5)])
def test_fft_plan_and_tile_overrides(lgf, dims, passes):
    """The planner uses three sweeps where two-axis kernels exist; tile-size overrides change rounding only."""
    import torch

    D = random_herm_field(dims, 3)
    D -= D.mean(axis=(0, 1, 2, 3), keepdims=True)
    res = []
    with lgf.Context(dims, 8, 18) as ctx:
        assert ctx.fft_passes() == passes
        # default plan -> one-thread register lines -> shared-memory two-axis passes (with tile overrides) -> one
        # pass per axis
        for key, val in [(None, 0), ("fft_reg2", 0), ("fft_reg", 0), ("fft_xy_planes", 1), ("fft_xy_planes", 4),
                         ("fft_zt_xc", 2), ("fft_zt_xc", 8), ("fft_two_axis", 0)]:
            if key:
                ctx.tune(key, val)
            ctx.set_field(to_dev(D, 8))
            ctx.step_accelerate()
            out = torch.empty(site_shape(dims) + (3, 3), dtype=torch.complex128, device="cuda")
            res.append(to_np(ctx.get_field(out)))
        with pytest.raises(lgf.LgfError):
            ctx.tune("no_such_key", 1)
    w_o = oracle.accelerate(dims, D)
    for w in res:
        assert np.max(np.abs(w - w_o)) < 1e-12 * np.max(np.abs(w_o))


@pytest.mark.parametrize("name,dims", SMALL)
@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_update(lgf, name, dims, prec, storage):
    """a5 + a6: g = GS(1 + i alpha/2 w), U <- g U g^dag(x+mu), against the oracle on the same w."""
    import torch

    U = small_config(name, dims)
    w = 3.0 * random_herm_field(dims, 5)
    U_o = oracle.transform(dims, U, oracle.build_g(dims, w, ALPHA))
    with lgf.Context(dims, prec, storage) as ctx:
        d = to_dev(U, prec)
        ctx.set_links(d)
        ctx.set_field(to_dev(w, prec))
        ctx.step_update(ALPHA)
        out = to_np(ctx.get_links(torch.empty_like(d)))
    assert np.max(np.abs(out - U_o)) < (1e-13 if prec == 8 else 2e-6)


def run_trajectory(lgf, dims, U, prec, storage, n, tune=None):
    import torch

    with lgf.Context(dims, prec, storage, stream=torch.cuda.current_stream()) as ctx:
        for k, v in (tune or {}).items():
            ctx.tune(k, v)
        d = to_dev(U, prec)
        ctx.set_links(d)
        ctx.iterate(ALPHA, n)
        F, th, P = ctx.measure()
        Fh, Th = ctx.history()
        assert len(Fh) == n + 1 and ctx.iterations() == n        # entry k = after k updates (R12)
        # the fused sweep's (F, theta) of the last configuration agree with a fresh a1 pass on it
        rel = 1e-13 if prec == 8 else 1e-6
        assert abs(F - Fh[-1]) <= rel * abs(F) and abs(th - Th[-1]) <= rel * abs(th)
        out = to_np(ctx.get_links(torch.empty_like(d)))
    return Fh, Th, P, out


@pytest.mark.parametrize("cfg", ["C1", "C2"])
@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_20(lgf, config_cache, cfg, prec, storage):
    """north_star parity: (F_n, theta_n), n = 0..20, and the links after 20 iterations."""
    dims = inputs.CONFIGS[cfg]["dims"]
    U = config_cache(cfg)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, 20)
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]
    assert abs(P - oracle.plaquette(dims, U)) < (1e-13 if prec == 8 else 1e-6)      # gauge invariant


@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_two_thread_fft(lgf, config_cache, prec, storage):
    """20 iterations of C2 with the two-threads-per-line FFT sweeps (lgf_fft_reg2.cu), whose inverse
    (x, y) sweep ends with the g-build: the same parity bar as the default plan."""
    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, 20, tune={"fft_reg2": 1})
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]


@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_cluster_gbuild(lgf, prec, storage):
    """64-point planes: in fp64 (64 KB a plane, one per CTA) the inverse (x, y) sweep runs as clusters of four CTAs,
    one per packed component, and builds g out of the neighbours' shared memory (k_fftr2_xy_gcluster) -- no separate
    g-build pass; in fp32 the four planes share a CTA.  Four iterations of a 64 x 64 x 16 x 16 lattice against the
    oracle, and against the unfused plan."""
    dims, n = (64, 64, 16, 16), 4
    U = inputs.smooth_config(dims, 0.3, 6416, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, n)
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]
    Fh2, Th2, _, out2 = run_trajectory(lgf, dims, U, prec, storage, n, tune={"fuse_g": 0})
    assert np.max(np.abs(out2 - out)) < (1e-13 if prec == 8 else 1e-5)
    with lgf.Context(dims, prec, storage) as ctx:       # (fp32: four 32 KB planes fit one CTA, no cluster needed)
        last = "k_fftr2_xy_gcluster<double, 64>" if prec == 8 else "k_fftr2_xy_bulk<float, 64, 1, 4, 1>"
        assert ctx.kernel_names()["fft"][-1].startswith(last)


@pytest.mark.parametrize("name,dims", [("C2", (16, 16, 16, 16)), ("mixed", (12, 6, 16, 4))])
@pytest.mark.parametrize("storage", [18, 12])
@pytest.mark.parametrize("share", [0, 1])
@pytest.mark.parametrize("minb", [4, 5])
def test_trajectory_fp32_sweep_five_ctas(lgf, config_cache, name, dims, storage, share, minb):
    """lgf_tune("sweep_minb", 4 | 5): the fp32 register sweep compiled for four / five CTAs per SM (128 / 96 registers) --
    the automatic choices on lattices that fill them, forced here on small ones.  Same arithmetic in the same order as
    the three-CTA build: the oracle's parity bar, and bit-equal links."""
    U = config_cache("C2") if name == "C2" else small_config(name, dims)
    n = 12
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    tune = {"sweep_tma": 0, "sweep_share": share}
    Fh, Th, P, out = run_trajectory(lgf, dims, U, 4, storage, n, tune=dict(tune, sweep_minb=minb))
    tol = TOL[4]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]
    Fh3, Th3, _, out3 = run_trajectory(lgf, dims, U, 4, storage, n, tune=dict(tune, sweep_minb=3))
    assert np.array_equal(out, out3) and np.array_equal(Th, Th3)
    with lgf.Context(dims, 4, storage) as ctx:
        for k, v in dict(tune, sweep_minb=minb).items():
            ctx.tune(k, v)
        assert ctx.kernel_names()["update"][0].endswith(", %d>" % minb)


@pytest.mark.parametrize("nc", [2, 4])
@pytest.mark.parametrize("prec", [8, 4])
def test_trajectory_cluster_zt_tile(lgf, prec, nc):
    """lgf_tune("fft_zt_cluster", nc): a 64 x 64 (z, t) tile split over a cluster of nc CTAs, the z-line / t-line
    transposition going through distributed shared memory (k_fftr2_zt_cluster).  Three iterations of a
    16 x 16 x 64 x 64 lattice against the oracle; the kernel really is the one the context names."""
    dims, n = (16, 16, 64, 64), 3
    U = inputs.smooth_config(dims, 0.3, 1664, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, 18, n, tune={"fft_zt_cluster": nc})
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]
    with lgf.Context(dims, prec, 18) as ctx:
        ctx.tune("fft_zt_cluster", nc)
        assert any(k.startswith("k_fftr2_zt_cluster<") for k in ctx.kernel_names()["fft"])
        ctx.tune("fft_zt_cluster", 0)
        assert not any(k.startswith("k_fftr2_zt_cluster<") for k in ctx.kernel_names()["fft"])


@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_bulk_copy_fft(lgf, config_cache, prec, storage):
    """20 iterations of C2 with lgf_tune("fft_bulk", 1): the (x, y) sweeps -- the inverse one ending in the g-build --
    fed by bulk copies.  Same parity bar as the default plan."""
    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, 20, tune={"fft_reg2": 1, "fft_bulk": 1})
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]


@pytest.mark.parametrize("name,dims", SMALL + [("tiny", (2, 4, 2, 6)), ("C2", (16, 16, 16, 16))])
@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_shared_neighbour_sweep(lgf, config_cache, name, dims, prec, storage):
    """lgf_tune("sweep_share", 1): A'_x and A'_y of backward neighbours inside the same CTA come through shared
    memory, the others are recomputed.  Lattices whose x lines do not divide the CTA's 128 sites (12, 3, 2) mix
    both paths inside a warp.  Same parity bar as the default sweep."""
    U = config_cache("C2") if name == "C2" else small_config(name, dims)
    n = 12
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, n, tune={"sweep_share": 1})
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]


@pytest.mark.parametrize("name,dims", [("C1", (8, 8, 8, 8)), ("x24", (24, 12, 4, 6)), ("x16", (16, 8, 6, 4)), ("x64", (64, 4, 4, 2)),
                                       ("C2", (16, 16, 16, 16))])
@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_staged_sweep(lgf, config_cache, name, dims, prec, storage):
    """lgf_tune("sweep_tma", 1): the persistent sweep fed by TMA tensor copies through a shared-memory ring
    (lgf_sweep_tma.cu) in every precision x storage variant -- tiles of 2 x 64, 4 x 24, 8 x 16 and 8 x 8 sites, tiles
    that are a whole (x, y) plane, with and without the fp64 register split.  Same parity bar as the default sweep;
    and the run is repeated: the new links must be the same bit for bit (the kernel once handed a ring slot back
    while its loads were still in flight)."""
    import torch

    U = config_cache("C2") if name == "C2" else small_config(name, dims)
    n = 12
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    tol = TOL[prec]
    outs = []
    for rsplit in (1, 0, 1):
        Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, n, tune={"sweep_tma": 1, "sweep_rsplit": rsplit})
        assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
        assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
        assert np.max(np.abs(out - U_o)) < tol["links"]
        outs.append(out)
    assert np.array_equal(outs[0], outs[2])
    with lgf.Context(dims, prec, storage) as ctx:
        ctx.tune("sweep_tma", 1)
        assert ctx.kernel_names()["update"][0].startswith("k_sweep_tma<")     # the lattice does take the staged sweep


@pytest.mark.parametrize("prec,storage", VARIANTS)
def test_trajectory_time_extent_twice_the_spatial_one(lgf, prec, storage):
    """16^3 x 32 -- the usual shape of a lattice QCD volume (the paper tunes on 32^3 x n): 20
    iterations through the register-line sweeps with Lt = 2 Lz, every precision x storage variant."""
    dims = (16, 16, 16, 32)
    U = inputs.smooth_config(dims, 0.3, 3216, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, prec, storage, 20)
    tol = TOL[prec]
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]


def test_trajectory_asymmetric(lgf):
    """Radix-3 / mixed-length axes: 12 x 6 x 24 x 48, 10 iterations, fp64."""
    dims = (12, 6, 24, 48)
    U = inputs.smooth_config(dims, 0.3, 77, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 10)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, 8, 18, 10)
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < 1e-12
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12
    assert np.max(np.abs(out - U_o)) < 1e-11


@pytest.mark.parametrize("storage", [18, 12])
def test_fix_c1_iteration_count(lgf, config_cache, storage):
    """Algorithm 1 to theta < 1e-15 on C1: iteration count within 2 % of the oracle's, same final state."""
    import torch

    dims = inputs.CONFIGS["C1"]["dims"]
    U = config_cache("C1")
    U_o, it_o, F_o, T_o = oracle.fix(dims, U, ALPHA, 1e-15, 2000)
    with lgf.Context(dims, 8, storage) as ctx:
        d = to_dev(U, 8)
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        Fh, Th = ctx.history()
        F, th, P = ctx.measure()
    assert abs(it - it_o) <= max(1, round(0.02 * it_o))
    assert len(Fh) == it + 1 and Th[-1] < 1e-15 and th < 1e-15
    assert np.all(Th[:-1] >= 1e-15)
    n = min(it, it_o)
    assert np.max(np.abs(Fh[: n + 1] - F_o[: n + 1]) / np.abs(F_o[: n + 1])) < 1e-11
    if it == it_o:
        assert np.max(np.abs(to_np(d) - U_o)) < 1e-10
    assert abs(P - oracle.plaquette(dims, U)) < 1e-13


def test_fix_pure_gauge_reaches_F1(lgf, config_cache):
    """Closed form: U = h(x) h(x+mu)^dag is driven to F -> 1, theta -> 0, U -> 1 (C2 pure-gauge variant)."""
    dims = inputs.CONFIGS["C2pg"]["dims"]
    U = config_cache("C2pg")
    with lgf.Context(dims, 8, 18) as ctx:
        d = to_dev(U, 8)
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        F, th, P = ctx.measure()
    assert 0 < it < 200
    assert abs(F - 1.0) < 1e-12 and th < 1e-15 and abs(P - 1.0) < 1e-12
    eye = np.eye(3)
    assert np.max(np.abs(to_np(d) - eye)) < 1e-6


@pytest.mark.parametrize("storage", [18, 12])
def test_fix_c2_iteration_count(lgf, config_cache, storage):
    """BASELINE.json configs[1]: 16^4 fp64 to theta < 1e-15 -- the iteration count within 2 % of the oracle's
    (north_star), the oracle's whole (F, theta) history and its final links."""
    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    U_o, it_o, F_o, T_o = oracle.fix(dims, U, ALPHA, 1e-15, 2000)
    with lgf.Context(dims, 8, storage) as ctx:
        d = to_dev(U, 8)
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        Fh, Th = ctx.history()
    assert abs(it - it_o) <= max(1, round(0.02 * it_o))
    n = min(it, it_o, 40)                      # well above the rounding floor of theta
    assert np.max(np.abs(Fh[:n] - F_o[:n]) / np.abs(F_o[:n])) < 1e-12
    assert np.max(np.abs(Th[:n] - T_o[:n]) / np.abs(T_o[:n])) < 1e-11
    assert Th[it] < 1e-15 and np.all(Th[:it] >= 1e-15)
    if it == it_o:
        assert np.max(np.abs(to_np(d) - U_o)) < 1e-11


def test_c2pg_golden_trajectory(lgf, config_cache):
    """The CUDA path against the stored oracle trajectory of the pure-gauge C2 variant
    (tests/golden/c2pg_trajectory.txt, written by tests/golden/make_golden.py from oracle/ alone)."""
    from test_oracle_golden import read_trajectory

    it_g, plaq, rows, final = read_trajectory("c2pg_trajectory.txt")
    dims = inputs.CONFIGS["C2pg"]["dims"]
    U = config_cache("C2pg")
    with lgf.Context(dims, 8, 18) as ctx:
        d = to_dev(U, 8)
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        Fh, Th = ctx.history()
        _, _, P = ctx.measure()
    for n, F, th in rows:
        assert abs(Fh[n] - F) <= 1e-12 * abs(F) and abs(Th[n] - th) <= 1e-12 * abs(th)
    assert abs(it - it_g) <= 1 and abs(P - plaq) < 1e-12
    assert abs(Fh[-1] - final[1]) < 1e-12


def test_fix_fp32_c2(lgf, config_cache):
    """fp32 runs stop at theta < 1e-12 (BASELINE.json config C2); count close to the fp64 oracle's."""
    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    _, it_o, F_o, T_o = oracle.fix(dims, U, ALPHA, 1e-12, 2000)
    with lgf.Context(dims, 4, 18) as ctx:
        h = np.ascontiguousarray(U.astype(np.complex64))
        it = ctx.fix_host(h, ALPHA, 1e-12, 2000)
        F, th, _ = ctx.measure()
    assert abs(it - it_o) <= max(2, round(0.05 * it_o))
    assert th < 1e-12 and abs(F - F_o[-1]) < 1e-5 * abs(F_o[-1])
    # the returned host array is still SU(3) to fp32 accuracy
    UU = np.einsum("...ij,...kj->...ik", h.astype(np.complex128), h.astype(np.complex128).conj())
    assert np.max(np.abs(UU - np.eye(3))) < 1e-4


def test_edge_cases(lgf):
    import torch

    with pytest.raises(lgf.LgfError) as e:
        lgf.Context((8, 8, 8, 10), 8, 18)
    assert e.value.code == lgf.LGF_EINVAL
    with pytest.raises(lgf.LgfError):
        lgf.Context((8, 8, 8, 8), 2, 18)
    with pytest.raises(lgf.LgfError):
        lgf.Context((8, 8, 8, 8), 8, 8)
    dims = (4, 4, 4, 4)
    with lgf.Context(dims, 8, 18) as ctx:
        with pytest.raises(lgf.LgfError) as e:
            ctx.iterate(ALPHA, 1)
        assert e.value.code == lgf.LGF_ESTATE
        # unit links: already in Landau gauge, Delta = 0, F = 1, theta = 0 -> zero iterations
        U = np.broadcast_to(np.eye(3, dtype=np.complex128), site_shape(dims) + (4, 3, 3)).copy()
        d = to_dev(U, 8)
        assert ctx.fix(d, ALPHA, 1e-15, 100) == 0
        F, th, P = ctx.measure()
        assert F == 1.0 and th == 0.0 and P == 1.0
        assert np.array_equal(to_np(d), U)
        # max_iter = 0: measure only, nothing changes
        U2 = inputs.smooth_config(dims, 0.2, 5)
        d2 = to_dev(U2, 8)
        assert ctx.fix(d2, ALPHA, 1e-15, 0) == 0
        assert np.array_equal(to_np(d2), U2)
        assert ctx.history_length() == 1
        # max_iter reached before convergence: returns max_iter, history has max_iter + 1 entries
        assert ctx.fix(d2, ALPHA, 1e-15, 3) == 3
        assert ctx.history_length() == 4
        _, F_o, T_o = oracle.iterate(dims, U2, ALPHA, 3)
        Fh, Th = ctx.history()
        assert np.max(np.abs(Th - T_o) / T_o) < 1e-12


@pytest.mark.parametrize("probe", ["measure", "measure_no_plaquette", "step_delta", "none"])
def test_history_entry0_survives_a_measurement_before_iterate(lgf, config_cache, probe):
    """lgf_measure / lgf_step_delta fill W and the partial sums but record nothing; the first lgf_iterate
    after them must still record entry 0 = the loaded configuration (include/lgf.h, R12).  Found at 64^4:
    measure() before iterate() used to leave the history one entry short."""
    dims = inputs.CONFIGS["C1"]["dims"]
    U = config_cache("C1")
    _, F_o, T_o = oracle.iterate(dims, U, ALPHA, 3)
    with lgf.Context(dims, 8, 18) as ctx:
        ctx.set_links(to_dev(U, 8))
        if probe == "measure":
            ctx.measure()
        elif probe == "measure_no_plaquette":
            ctx.measure(plaquette=False)
        elif probe == "step_delta":
            ctx.step_delta()
        assert ctx.history_length() == 0
        ctx.iterate(ALPHA, 1)
        assert ctx.history_length() == 2 and ctx.iterations() == 1
        ctx.measure()                                   # between two iterate calls: no duplicate entry either
        ctx.iterate(ALPHA, 2)
        Fh, Th = ctx.history()
    assert len(Fh) == 4
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < 1e-12
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 6, 16, 4), (16, 16, 16, 16)])
@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18)])
def test_accumulated_transformation(lgf, dims, prec, storage):
    """NEXT-2: lgf_track_transform / lgf_get_transform.  G(x) = g_n(x) ... g_1(x) against the product of the
    oracle's g fields, and the defining property G U0 G(x+mu)^dag = U_n on the CUDA side's own output."""
    import torch

    U0 = inputs.smooth_config(dims, 0.3, 97, haar=True)
    n = 8
    U, G = U0.copy(), np.broadcast_to(np.eye(3, dtype=np.complex128), site_shape(dims) + (3, 3)).copy()
    for _ in range(n):
        D, _, _ = oracle.measure(dims, U)
        g = oracle.build_g(dims, oracle.accelerate(dims, D), ALPHA)
        U = oracle.transform(dims, U, g)
        G = g @ G
    tol = TOL[prec]["links"]
    cdt = torch.complex128 if prec == 8 else torch.complex64
    with lgf.Context(dims, prec, storage) as ctx:
        with pytest.raises(lgf.LgfError) as e:
            ctx.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda"))
        assert e.value.code == lgf.LGF_ESTATE
        ctx.track_transform(True)
        d = to_dev(U0, prec)
        ctx.set_links(d)
        ctx.iterate(ALPHA, 3)
        ctx.step_accelerate()                 # the single-step entry points accumulate too
        ctx.step_update(ALPHA)
        ctx.iterate(ALPHA, n - 4)
        Gd = to_np(ctx.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda")))
        out = to_np(ctx.get_links(torch.empty_like(d)))
        assert np.max(np.abs(Gd - G)) < tol
        assert np.max(np.abs(out - U)) < tol
        assert np.max(np.abs(oracle.transform(dims, U0, Gd) - out)) < tol
        # set_links resets G to the identity
        ctx.set_links(d)
        G1 = to_np(ctx.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda")))
        assert np.array_equal(G1, np.broadcast_to(np.eye(3), G1.shape))
        # a converged fix stops accumulating when the iteration stops
        it = ctx.fix(d, ALPHA, 1e-15 if prec == 8 else 1e-12, 500)
        Gf = to_np(ctx.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda")))
        assert 0 < it < 500
        assert np.max(np.abs(oracle.transform(dims, U0, Gf) - to_np(d))) < tol * (1 + it / 20)
        ctx.track_transform(False)


@pytest.mark.parametrize("storage", [18, 12])
def test_reunit_every_update_keeps_fp64_parity(lgf, config_cache, storage):
    """lgf_tune("reunit_every", 1): every new link is projected onto SU(3) inside the sweep -- on the stored copy
    and on the copy recomputed for the backward neighbour alike.  In fp64 the projection moves the last bits
    only, so the 20-iteration parity bar against the (never projecting) oracle must still hold; it would not
    if Delta were computed from differently projected copies."""
    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    Fh, Th, P, out = run_trajectory(lgf, dims, U, 8, storage, 20, tune={"reunit_every": 1})
    # ... and the same through the staged sweep wherever it applies (with and without the fp64 register split)
    for rsplit in (1, 0):
        Fh2, Th2, _, out2 = run_trajectory(lgf, dims, U, 8, storage, 20, tune={"reunit_every": 1, "sweep_tma": 1, "sweep_rsplit": rsplit})
        assert np.max(np.abs(Th2 - T_o) / np.abs(T_o)) < 1e-12 and np.max(np.abs(out2 - U_o)) < 1e-11
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < 1e-12
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12
    assert np.max(np.abs(out - U_o)) < 1e-11
    assert np.max(np.abs(out @ np.conj(np.swapaxes(out, -1, -2)) - np.eye(3))) < 2e-15      # tighter than R13's drift


@pytest.mark.parametrize("storage", [18, 12])
def test_reunit_holds_fp32_links_on_su3(lgf, storage):
    """fp32, 1500 updates of a rough (hot-start) 8^4 configuration: without projection the links drift and
    take the gauge-invariant plaquette with them; with reunit_every = 10 both stay at float rounding."""
    import torch

    dims = (8, 8, 8, 8)
    U = inputs.hot_config(dims, 4711)
    P0 = oracle.plaquette(dims, U.astype(np.complex64).astype(np.complex128))
    res = {}
    for every in (0, 10):
        with lgf.Context(dims, 4, storage) as ctx:
            ctx.tune("reunit_every", every)
            d = to_dev(U, 4)
            ctx.set_links(d)
            ctx.iterate(ALPHA, 1500)
            _, th, P = ctx.measure()
            out = to_np(ctx.get_links(torch.empty_like(d)))
        res[every] = (abs(P - P0), np.max(np.abs(out @ np.conj(np.swapaxes(out, -1, -2)) - np.eye(3))), th)
    assert res[10][1] < 2e-6 and res[10][0] < 5e-6
    assert res[0][1] > 5 * res[10][1]                # the drift the projection removes is real
    # the projection does not disturb the iteration: same theta as the unprojected run to within a factor 2
    # (a hot start converges slowly: theta ~ 1e-5 after 1500 updates, down from 3.6)
    assert res[10][2] < 1e-3 and 0.5 < res[10][2] / res[0][2] < 2.0


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 6, 16, 4), (3, 24, 2, 48), (16, 16, 16, 16), (6, 4, 32, 2)])
@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18)])
def test_gluon_field(lgf, dims, prec, storage):
    """lgf_gluon_field: A_mu(k) for every direction against the oracle (naive DFT of the algebra part), natural k
    order out of the permuted order the one-axis passes leave, both halves of the packed real fields."""
    import torch

    U = inputs.smooth_config(dims, 0.35, 808, haar=True)
    cdt = torch.complex128 if prec == 8 else torch.complex64
    with lgf.Context(dims, prec, storage) as ctx:
        d = to_dev(U, prec)
        ctx.set_links(d)
        ctx.iterate(ALPHA, 1)                                   # W holds Delta: the call must not depend on that
        U1 = to_np(ctx.get_links(torch.empty_like(d)))
        got = [to_np(ctx.gluon_field(mu, torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda")))
               for mu in range(4)]
        ctx.iterate(ALPHA, 1)                                   # ... and the iteration must still work after it
        assert ctx.history_length() == 3
        Fh, Th = ctx.history()
    _, F_o, T_o = oracle.iterate(dims, U, ALPHA, 2)
    rel = 1e-12 if prec == 8 else 1e-5
    assert np.max(np.abs(Th - T_o) / T_o) < rel and np.max(np.abs(Fh - F_o) / np.abs(F_o)) < rel
    for mu in range(4):
        ref = oracle.gluon_field(dims, U1, mu)
        scale = np.max(np.abs(ref))
        assert np.max(np.abs(got[mu] - ref)) < (1e-12 if prec == 8 else 2e-5) * scale, "mu = %d" % mu


def test_gluon_field_is_transverse_after_fixing(lgf, config_cache):
    """The point of it all, on the CUDA path's own output: fix C2 to theta < 1e-15, then
    sum_mu (exp(-2 pi i k_mu/L_mu) - 1) A_mu(k) = F[Delta](k) vanishes mode by mode (Parseval: 3 V^2 theta)."""
    import torch

    dims = inputs.CONFIGS["C2"]["dims"]
    V = int(np.prod(dims))
    U = config_cache("C2")

    def divergence(ctx):
        tot = 0
        for mu in range(4):
            A = to_np(ctx.gluon_field(mu, torch.empty(site_shape(dims) + (3, 3), dtype=torch.complex128, device="cuda")))
            ph = np.exp(-2j * np.pi * np.arange(dims[mu]) / dims[mu]) - 1.0
            shape = [1, 1, 1, 1, 1, 1]
            shape[3 - mu] = dims[mu]
            tot = tot + ph.reshape(shape) * A
        return tot

    with lgf.Context(dims, 8, 18) as ctx:
        d = to_dev(U, 8)
        ctx.set_links(d)
        before = np.abs(divergence(ctx)).max()
        it = ctx.fix(d, ALPHA, 1e-15, 2000)
        after = divergence(ctx)
        _, th, _ = ctx.measure(plaquette=False)
    assert 0 < it < 2000 and th < 1e-15 and before > 1.0
    assert abs(np.sum(np.abs(after) ** 2) - 3.0 * V * V * th) < 1e-3 * 3.0 * V * V * th
    assert np.abs(after).max() < np.sqrt(3.0 * V * V * 1e-15)


@pytest.mark.parametrize("dims", [(8, 8, 8, 8), (12, 6, 16, 4)])
@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18)])
def test_apply_transform(lgf, dims, prec, storage):
    """lgf_apply_transform: U <- G U G(x+mu)^dag for a given field G against the oracle's transform; G off SU(3)
    is projected first (row-wise Gram-Schmidt, the oracle's pinned orc_gs); history restarts; a tracked
    accumulated transformation picks the factor up."""
    import torch

    V = int(np.prod(dims))
    U = small_config("x", dims) if dims != (8, 8, 8, 8) else inputs.make_config("C1")
    h = inputs.haar_su3(606, inputs.STREAM_HAAR, 0, V).reshape(site_shape(dims) + (3, 3))
    noisy = h * (1.0 + 1e-3 * inputs.normals(607, 5, 0, V).reshape(site_shape(dims) + (1, 1)))      # off SU(3)
    h_proj = np.stack([oracle.gs(m) for m in noisy.reshape(-1, 3, 3)]).reshape(h.shape)
    U_o = oracle.transform(dims, U, h_proj)
    D_o, F_o, T_o = oracle.measure(dims, U_o)
    tol = 1e-13 if prec == 8 else 2e-6
    cdt = torch.complex128 if prec == 8 else torch.complex64
    with lgf.Context(dims, prec, storage) as ctx:
        ctx.track_transform(True)
        d = to_dev(U, prec)
        ctx.set_links(d)
        ctx.iterate(ALPHA, 2)
        ctx.set_links(d)
        _, _, P0 = ctx.measure()
        ctx.apply_transform(to_dev(noisy, prec))
        assert ctx.history_length() == 0 and ctx.iterations() == 0
        out = to_np(ctx.get_links(torch.empty_like(d)))
        Gt = to_np(ctx.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=cdt, device="cuda")))
        ctx.iterate(ALPHA, 0)                                   # records entry 0 from what the sweep left behind
        Fh, Th = ctx.history()
        _, _, P1 = ctx.measure()
    assert np.max(np.abs(out - U_o)) < tol
    assert np.max(np.abs(Gt - h_proj)) < tol
    assert len(Fh) == 1
    assert abs(Fh[0] - F_o) < (1e-12 if prec == 8 else 1e-5) * abs(F_o)
    assert abs(Th[0] - T_o) < (1e-12 if prec == 8 else 1e-5) * abs(T_o)
    assert abs(P1 - P0) < (1e-13 if prec == 8 else 1e-6)        # gauge invariant


def test_mixed_precision_workflow_preserves_the_orbit(lgf, config_cache):
    """Find G in fp32 (tracked), apply it to the ORIGINAL fp64 links, polish in fp64: theta < 1e-15 with the
    plaquette of the original configuration preserved to fp64 rounding, in far fewer fp64 iterations."""
    import torch

    dims = inputs.CONFIGS["C2"]["dims"]
    U = config_cache("C2")
    P_o = oracle.plaquette(dims, U)
    with lgf.Context(dims, 4, 18) as c32:
        c32.track_transform(True)
        l32 = to_dev(U, 4)
        it32 = c32.fix(l32, ALPHA, 1e-12, 2000)
        G32 = c32.get_transform(torch.empty(site_shape(dims) + (3, 3), dtype=torch.complex64, device="cuda"))
    with lgf.Context(dims, 8, 18) as c64:
        d = to_dev(U, 8)
        it_only = c64.fix(d.clone(), ALPHA, 1e-15, 2000)
        c64.set_links(d)
        c64.apply_transform(G32.to(torch.complex128))
        _, th_start, P_start = c64.measure()
        out = c64.get_links(torch.empty_like(d))
        it_polish = c64.fix(out, ALPHA, 1e-15, 2000)
        F, th, P = c64.measure()
    assert 0 < it32 < 2000 and 0 < it_only < 2000
    assert th_start < 1e-10                         # the float transformation already fixes the gauge to float accuracy
    assert abs(P_start - P_o) < 1e-13 and abs(P - P_o) < 1e-13
    assert th < 1e-15 and it_polish < it_only // 2


@pytest.mark.parametrize("prec", [8, 4])
def test_nan_input_stops_the_iteration(lgf, config_cache, prec):
    """include/lgf.h: theta NaN/Inf -> the device-side flag stops the loop, lgf_fix returns LGF_ENAN (at its next
    look at the flag, not after max_iter), lgf_iterate stops recording; nothing hangs or aborts."""
    import time

    import torch

    dims = inputs.CONFIGS["C1"]["dims"]
    U = config_cache("C1").copy()
    U[3, 2, 1, 0, 2, 1, 1] = np.nan
    with lgf.Context(dims, prec, 18) as ctx:
        d = to_dev(U, prec)
        t0 = time.perf_counter()
        with pytest.raises(lgf.LgfError) as e:
            ctx.fix(d, ALPHA, 1e-15, 10 ** 6)
        assert e.value.code == lgf.LGF_ENAN
        assert time.perf_counter() - t0 < 5.0                 # a million iterations would take half a minute
        ctx.set_links(to_dev(U, prec))
        ctx.iterate(ALPHA, 50)
        torch.cuda.synchronize()
        n = ctx.history_length()
        Fh, Th = ctx.history()
        assert 1 <= n <= 3 and not np.isfinite(Th[-1])        # the NaN reaches theta within an iteration or two
        # a clean configuration afterwards works as usual
        ctx.set_links(to_dev(config_cache("C1"), prec))
        ctx.iterate(ALPHA, 2)
        assert ctx.history_length() == 3 and np.all(np.isfinite(ctx.history()[1]))


def test_12_real_matches_18_real(lgf, config_cache):
    """Third-row reconstruction (eq. 8) changes rounding only."""
    dims = inputs.CONFIGS["C1"]["dims"]
    U = config_cache("C1")
    a = run_trajectory(lgf, dims, U, 8, 18, 8)
    b = run_trajectory(lgf, dims, U, 8, 12, 8)
    assert np.max(np.abs(a[3] - b[3])) < 1e-12
    assert np.max(np.abs(a[1] - b[1]) / a[1]) < 1e-12
