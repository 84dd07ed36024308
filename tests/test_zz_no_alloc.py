"""lgf_measure_static (include/lgf.h, csrc/lgf_static.cu): the one entry point that allocates nothing -- its scratch
(per-block partial sums) is a fixed device array inside the library -- against the existing path (a context's
lgf_measure, whose scratch is cudaMalloc'ed) on two calls in a row.  Collected last on purpose (the file name): the
suite runs with `pytest -x`, and a failure here must not hide the parity tests."""
import numpy as np
import pytest

from paper_1206_0675_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {8: 1e-12, 4: 1e-5}          # the parity tests' relative tolerance on F and theta (tests/test_gpu_parity.py)


def _dev(a, prec):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).to(torch.complex128 if prec == 8 else torch.complex64).cuda()


@pytest.mark.parametrize("prec", [8, 4])
def test_measure_static_matches_the_context_path_on_two_calls_in_a_row(prec):
    import torch

    from paper_1206_0675_b200 import binding

    binding.load()
    # a 16^4 lattice first (256 blocks of partial sums), then an 8^4 one (16 blocks): the second call finds the first
    # one's partial sums in the shared scratch array and must not read them; then the first again
    cases = [("C2", inputs.CONFIGS["C2"]["dims"]), ("C1", inputs.CONFIGS["C1"]["dims"]), ("C2", inputs.CONFIGS["C2"]["dims"])]
    want = {}
    for name, dims in cases:
        if name not in want:
            d = _dev(inputs.make_config(name), prec)
            with binding.Context(dims, prec, 18, stream=torch.cuda.current_stream()) as ctx:      # the existing path
                ctx.set_links(d)
                F, th, _ = ctx.measure(plaquette=False)
            want[name] = (d, F, th)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for name, dims in cases:
        d, F, th = want[name]
        binding.measure_static(dims, prec, d, out, stream=torch.cuda.current_stream())
        got = out.cpu().numpy().copy()
        assert abs(got[0] - F) <= TOL[prec] * abs(F), (name, got[0], F)
        assert abs(got[1] - th) <= TOL[prec] * abs(th), (name, got[1], th)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0 - (1 << 20)        # the calls took no device memory


def test_measure_static_refuses_a_lattice_beyond_its_scratch():
    import torch

    from paper_1206_0675_b200 import binding

    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    dims = (64, 64, 32, 32)                                         # 4.2 M sites > LGF_STATIC_MAX_SITES
    assert int(np.prod(dims)) > binding.LGF_STATIC_MAX_SITES
    fake = torch.zeros(8, dtype=torch.float64, device="cuda")
    lib = binding.load()
    import ctypes

    rc = lib.lgf_measure_static((ctypes.c_int * 4)(*dims), 8, ctypes.c_void_p(fake.data_ptr()), ctypes.c_void_p(out.data_ptr()), None)
    assert rc == binding.LGF_EINVAL and b"LGF_STATIC_MAX_SITES" in lib.lgf_static_last_error()
    # the largest lattice it takes: 32^3 x 64 = 2^21 sites, unit links -> F = 1, theta = 0
    dims = (32, 32, 32, 64)
    U = torch.zeros(dims[::-1] + (4, 3, 3), dtype=torch.complex64, device="cuda")
    for i in range(3):
        U[..., i, i] = 1
    binding.measure_static(dims, 4, U, out)
    F, th = out.cpu().numpy()
    assert abs(F - 1.0) < 1e-12 and th == 0.0
