"""bench.py's multi-rank branch (NCCL barrier, max-over-ranks of the device time, whole-job rate) on a real
GPU.  The box has one GPU, so the process group has a single rank -- enough to execute every collective call
of that branch on device tensors; the arithmetic of the reductions is covered by tests/test_ensemble_gloo.py."""
import os
import socket

import pytest

pytestmark = pytest.mark.gpu


def test_time_variant_with_a_one_rank_nccl_group(config_cache):
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    import bench
    from paper_1206_0675_b200 import binding, ensemble, inputs

    binding.load()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        dims = inputs.CONFIGS["C1"]["dims"]
        U = config_cache("C1")
        r = bench.time_variant(binding, torch, U, dims, "fp64", 18, 20, 3, dist)
        assert r["ms_per_step"] > 0 and r["launches"] == 20 * 5 + 1 and r["remeasured"] is None
        assert 0 < r["theta"] < 1.0
        rate = ensemble.whole_job_rate(dist, 20, r["ms_total"])
        assert rate["units"] == 20 and abs(rate["ms"] - r["ms_total"]) < 1e-9
        e = bench.time_e2e(binding, torch, U, dims, "fp64", 18, 1e-15, 2000, dist)
        assert 0 < e["iterations"] < 2000 and e["theta"] < 1e-15
    finally:
        dist.destroy_process_group()
