"""The N > 1 path is "replicas only": whole configurations are sharded over the
ranks, no data-path collective.  These CPU tests run the host-side bookkeeping with world_size 2 on the
gloo backend: member sharding, distinct seeded inputs per member, max-over-ranks timing, whole-job rate
and the gather of per-member results on rank 0."""
import os
import socket

import numpy as np
import pytest

from paper_1206_0675_b200 import ensemble, inputs


def test_member_indices_partition():
    for n in (0, 1, 2, 5, 8, 13):
        for world in (1, 2, 3, 8):
            parts = [ensemble.member_indices(n, r, world) for r in range(world)]
            flat = sorted(m for p in parts for m in p)
            assert flat == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        ensemble.member_indices(4, 2, 2)


def test_no_dist_is_identity():
    assert ensemble.max_over_ranks(None, 3.5) == 3.5
    assert ensemble.sum_over_ranks(None, 7) == 7.0
    r = ensemble.whole_job_rate(None, 200, 100.0)
    assert r["per_s"] == pytest.approx(2000.0)
    assert ensemble.gather_results(None, [{"member": 1}, {"member": 0}]) == [{"member": 0}, {"member": 1}]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        members = ensemble.member_indices(5, rank, world)
        local = []
        for m in members:
            U = inputs.smooth_config((4, 4, 4, 4), 0.2, 77 + 7919 * ensemble.member_seed_offset(m), haar=True)
            local.append({"member": m, "rank": rank, "checksum": float(np.abs(U).sum()), "first": complex(U.flat[0])})
        ms_local = 10.0 * (rank + 1)                      # rank 1 is the slow one
        rate = ensemble.whole_job_rate(dist, units_local=len(members) * 20, ms_local=ms_local)
        dist.barrier()
        res = ensemble.gather_results(dist, local)
        q.put((rank, rate, res))
    finally:
        dist.destroy_process_group()


def test_replicas_world2_gloo():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(2):
        rank, rate, res = q.get(timeout=120)
        got[rank] = (rate, res)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # timing: max over ranks (20 ms), units: all 5 members x 20 iterations, on every rank
    for rank in (0, 1):
        rate = got[rank][0]
        assert rate["ms"] == pytest.approx(20.0)
        assert rate["units"] == pytest.approx(100.0)
        assert rate["per_s"] == pytest.approx(100.0 / 0.020)
    assert got[1][1] is None
    res = got[0][1]
    assert [r["member"] for r in res] == [0, 1, 2, 3, 4]
    assert [r["rank"] for r in res] == [0, 1, 0, 1, 0]
    # every member is a different configuration (distinct seeds), reproducible from its index alone
    firsts = {r["first"] for r in res}
    assert len(firsts) == 5
    U2 = inputs.smooth_config((4, 4, 4, 4), 0.2, 77 + 7919 * 2, haar=True)
    assert res[2]["checksum"] == pytest.approx(float(np.abs(U2).sum()), rel=0, abs=0)
