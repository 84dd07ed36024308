"""One configuration sharded over N ranks (t-slabs): parity with the CPU
oracle through the per-rank C entry points lgf_slab_*, with the N ranks emulated one after the other in ONE
process on the one GPU of the box (paper_1206_0675_b200.slab.LocalExchange: the exchanges are device copies, no
kernel waits on another rank).  The exchange over torch.distributed is covered on the CPU by
tests/test_slab_gloo.py (gloo, world_size 2) and here by a one-rank NCCL group.
Tolerances are the north_star's, as in tests/test_gpu_parity.py.  Every test here needs a GPU (-m gpu)."""
import numpy as np
import pytest

import oracle
from paper_1206_0675_b200 import inputs

pytestmark = pytest.mark.gpu

ALPHA = 0.08
TOL = {8: dict(scalar=1e-12, links=1e-11, field=1e-12), 4: dict(scalar=1e-5, links=2e-5, field=2e-5)}


@pytest.fixture(scope="module")
def slab():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_1206_0675_b200 import binding, slab

    binding.load()
    return slab


def to_dev(a, prec):
    import torch

    cdt = torch.complex128 if prec == 8 else torch.complex64
    return torch.view_as_real(torch.from_numpy(np.ascontiguousarray(a)).to(cdt).cuda())


def gathered(slabs):
    import torch

    t = torch.cat(list(slabs), dim=0).cpu().numpy().astype(np.float64)
    return t[..., 0] + 1j * t[..., 1]


# (dims, world): T = Lt / world from the whole lattice down to ONE slice per rank; Zl = Lz / world down to 1
CASES = [((8, 8, 8, 8), 1), ((8, 8, 8, 8), 2), ((8, 8, 8, 8), 4), ((8, 8, 8, 8), 8), ((12, 6, 16, 4), 2),
         ((12, 6, 16, 4), 4), ((16, 16, 12, 6), 3), ((16, 16, 12, 6), 6), ((3, 24, 2, 48), 2), ((32, 32, 8, 4), 4),
         ((64, 64, 4, 2), 2), ((16, 16, 16, 32), 8), ((32, 32, 16, 16), 4)]


@pytest.mark.parametrize("dims,world", CASES)
@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18), (4, 12)])
def test_slab_delta_and_accelerate(slab, dims, world, prec, storage):
    """a1 (with the U_t halo) and a2-a4 (with the two all-to-alls) element by element."""
    U = inputs.smooth_config(dims, 0.25, 977 + world, haar=True)
    D_o, F_o, th_o = oracle.measure(dims, U)
    w_o = oracle.accelerate(dims, D_o)
    fx = slab.SlabFixer(dims, prec, storage, slab.LocalExchange(world))
    fx.set_links_global(to_dev(U, prec))
    F, th = fx.measure()
    tol = TOL[prec]
    assert abs(F - F_o) <= tol["scalar"] * abs(F_o)
    assert abs(th - th_o) <= tol["scalar"] * abs(th_o)
    fx._step_delta(-1.0, False)
    D = gathered(fx.work_field())
    assert np.max(np.abs(D - D_o)) < tol["field"] * max(1.0, np.max(np.abs(D_o)))
    fx._step_accelerate()
    w = gathered(fx.work_field())
    assert np.max(np.abs(w - w_o)) < (1e-12 if prec == 8 else 2e-5) * np.max(np.abs(w_o))
    fx.destroy()


@pytest.mark.parametrize("dims,world", CASES)
@pytest.mark.parametrize("prec,storage", [(8, 18), (8, 12), (4, 18), (4, 12)])
def test_slab_trajectory(slab, dims, world, prec, storage):
    """north_star parity for the sharded path: (F_n, theta_n), n = 0..12, and the links after 12 iterations."""
    n = 12
    U = inputs.smooth_config(dims, 0.25, 4242 + world, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    fx = slab.SlabFixer(dims, prec, storage, slab.LocalExchange(world))
    fx.set_links_global(to_dev(U, prec))
    fx.iterate(ALPHA, n)
    Fh, Th = fx.history()
    out = gathered(fx.get_links())
    tol = TOL[prec]
    assert len(Fh) == n + 1
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(out - U_o)) < tol["links"]
    if world > 1:
        assert fx.exchanged_bytes > 0
    fx.destroy()


@pytest.mark.parametrize("dims,world", [((8, 8, 8, 8), 2), ((16, 16, 12, 6), 6), ((12, 6, 16, 4), 4)])
@pytest.mark.parametrize("prec,storage", [(8, 18), (4, 12)])
def test_slab_single_steps_make_the_same_trajectory(slab, dims, world, prec, storage):
    """The single-step entry points (delta / fft_inverse + gbuild / in-place update with the U_t halo re-exchanged
    every iteration) against the oracle, and a mix of both forms of a6 in one run."""
    n = 6
    U = inputs.smooth_config(dims, 0.25, 515 + world, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    fx = slab.SlabFixer(dims, prec, storage, slab.LocalExchange(world))
    fx.set_links_global(to_dev(U, prec))
    for k in range(n):
        fx._step_delta(-1.0, not fx._recorded)     # (the fused sweep has recorded its result itself)
        if k % 3 == 2:
            fx._step_iteration(ALPHA, -1.0)        # fused sweep in between: records the next entry itself
        else:
            fx._step_accelerate()
            fx._step_update(ALPHA)
    fx._step_delta(-1.0, not fx._recorded)
    Fh, Th = fx.history()
    tol = TOL[prec]
    assert len(Th) == n + 1
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < tol["scalar"]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(gathered(fx.get_links()) - U_o)) < tol["links"]
    fx.destroy()


def test_slab_sweep_refuses_a_stale_link_halo(slab):
    from paper_1206_0675_b200 import binding

    dims = (8, 8, 8, 8)
    fx = slab.SlabFixer(dims, 8, 18, slab.LocalExchange(2))
    fx.set_links_global(to_dev(inputs.make_config("C1"), 8))
    with pytest.raises(binding.LgfError):
        fx.ranks[0].sweep(fx._sums[0])         # no U_t halo yet
    fx._step_delta(-1.0, True)
    fx._step_accelerate()
    fx._step_update(ALPHA)                      # in-place update: the halo is stale again
    with pytest.raises(binding.LgfError):
        fx.ranks[0].sweep(fx._sums[0])
    fx.destroy()


@pytest.mark.parametrize("prec", [8, 4])
def test_slab_64_point_t_lines_in_registers(slab, prec):
    """Lt = 64: the t pass with 32 complex registers per thread (k_slab_fft_line2<64>), 3 iterations over 4 ranks."""
    dims, n = (16, 16, 16, 64), 3
    U = inputs.smooth_config(dims, 0.25, 6464, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    fx = slab.SlabFixer(dims, prec, 18, slab.LocalExchange(4))
    fx.set_links_global(to_dev(U, prec))
    fx.iterate(ALPHA, n)
    Fh, Th = fx.history()
    tol = TOL[prec]
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
    assert np.max(np.abs(gathered(fx.get_links()) - U_o)) < tol["links"]
    fx.destroy()


@pytest.mark.parametrize("world", [1, 2, 4])
@pytest.mark.parametrize("prec,storage", [(8, 18), (4, 12)])
def test_slab_component_pipelined_order_is_the_plain_order(slab, world, prec, storage):
    """The per-component entry points (fft_forward_comp / fft_t_comp / fft_zinv_comp / fft_xyinv) in the overlapped
    order against the plain order and the oracle: 16^3 x 32 over 1, 2, 4 emulated ranks."""
    dims, n = (16, 16, 16, 32), 5
    U = inputs.smooth_config(dims, 0.25, 1632, haar=True)
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, n)
    tol, outs = TOL[prec], []
    for overlap in (True, False):
        fx = slab.SlabFixer(dims, prec, storage, slab.LocalExchange(world), overlap=overlap)
        assert fx.overlap == overlap
        fx.set_links_global(to_dev(U, prec))
        fx.iterate(ALPHA, n)
        Fh, Th = fx.history()
        outs.append(gathered(fx.get_links()))
        assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < tol["scalar"]
        assert np.max(np.abs(outs[-1] - U_o)) < tol["links"]
        fx.destroy()
    assert np.array_equal(outs[0], outs[1])


def test_slab_equals_one_gpu_path_on_c2(slab):
    """16^4 (C2) over 4 ranks against the oracle over 20 iterations, and against the one-GPU path of liblgf."""
    import torch

    from paper_1206_0675_b200 import binding

    dims = inputs.CONFIGS["C2"]["dims"]
    U = inputs.make_config("C2")
    U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 20)
    d = to_dev(U, 8)
    fx = slab.SlabFixer(dims, 8, 18, slab.LocalExchange(4))
    fx.set_links_global(d)
    fx.iterate(ALPHA, 20)
    Fh, Th = fx.history()
    out = gathered(fx.get_links())
    assert np.max(np.abs(Fh - F_o) / np.abs(F_o)) < 1e-12
    assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12
    assert np.max(np.abs(out - U_o)) < 1e-11
    with binding.Context(dims, 8, 18) as ctx:
        ctx.set_links(d)
        ctx.iterate(ALPHA, 20)
        one = torch.empty_like(d)
        ctx.get_links(one)
        F1, T1 = ctx.history()
    one = one.cpu().numpy()
    assert np.max(np.abs(out - (one[..., 0] + 1j * one[..., 1]))) < 1e-11
    assert np.max(np.abs(Th - T1) / np.abs(T1)) < 1e-12
    fx.destroy()


def test_slab_fix_iteration_count(slab):
    """Algorithm 1 to theta < 1e-15 on C1 over 2 ranks: the oracle's iteration count within 2 %."""
    dims = inputs.CONFIGS["C1"]["dims"]
    U = inputs.make_config("C1")
    U_o, it_o, F_o, T_o = oracle.fix(dims, U, ALPHA, 1e-15, 2000)
    fx = slab.SlabFixer(dims, 8, 18, slab.LocalExchange(2))
    fx.set_links_global(to_dev(U, 8))
    it = fx.fix(ALPHA, 1e-15, 2000)
    Fh, Th = fx.history()
    assert abs(it - it_o) <= max(1, round(0.02 * it_o))
    assert len(Th) == it + 1 and Th[-1] < 1e-15 and np.all(Th[:-1] >= 1e-15)
    F, th = fx.measure()
    assert th < 1e-15 and abs(F - F_o[-1]) < 1e-11
    fx.destroy()


def test_slab_argument_validation(slab):
    from paper_1206_0675_b200 import binding

    with pytest.raises(binding.LgfError):
        binding.SlabContext((8, 8, 8, 8), 8, 18, 0, 3)            # 3 does not divide Lt
    with pytest.raises(binding.LgfError):
        binding.SlabContext((8, 8, 2, 8), 8, 18, 0, 4)            # 4 does not divide Lz
    with pytest.raises(binding.LgfError):
        binding.SlabContext((8, 8, 8, 8), 8, 18, 2, 2)            # rank out of range
    c = binding.SlabContext((8, 8, 8, 8), 8, 18, 1, 2)
    with pytest.raises(binding.LgfError):
        c.update()                                                # no links loaded
    assert c.halo_elems(binding.LGF_HALO_LINKS) == 512 * 18 and c.halo_elems(binding.LGF_HALO_G) == 512 * 12
    c.destroy()


def test_slab_over_a_one_rank_nccl_group(slab):
    """DistExchange on the device through an NCCL process group of one rank (the box has one GPU): the same
    driver code path torchrun ranks take, checked against the oracle."""
    import os

    import torch
    import torch.distributed as dist

    created = False
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29631")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
        created = True
    try:
        dims = (8, 8, 8, 8)
        U = inputs.make_config("C1")
        U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 5)
        fx = slab.SlabFixer(dims, 8, 18, slab.DistExchange(dist))
        fx.set_links_global(to_dev(U, 8))
        fx.iterate(ALPHA, 5)
        Fh, Th = fx.history()
        assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12
        assert np.max(np.abs(gathered(fx.get_links()) - U_o)) < 1e-11
        fx.destroy()
        # 16^4: every axis takes the register-line passes, so the exchanges run one component at a time on a second
        # stream (start / finish with events) while the main stream transforms the next component
        dims = inputs.CONFIGS["C2"]["dims"]
        U = inputs.make_config("C2")
        U_o, F_o, T_o = oracle.iterate(dims, U, ALPHA, 6)
        outs = []
        for overlap in (True, False):
            fx = slab.SlabFixer(dims, 8, 18, slab.DistExchange(dist), overlap=overlap)
            assert fx.overlap == overlap
            fx.set_links_global(to_dev(U, 8))
            fx.iterate(ALPHA, 6)
            Fh, Th = fx.history()
            outs.append(gathered(fx.get_links()))
            assert np.max(np.abs(Th - T_o) / np.abs(T_o)) < 1e-12
            assert np.max(np.abs(outs[-1] - U_o)) < 1e-11
            fx.destroy()
        assert np.array_equal(outs[0], outs[1])              # the same kernels on the same data, only ordered differently
    finally:
        if created:
            dist.destroy_process_group()
