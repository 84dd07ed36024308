"""The exchanges of the sharded path (paper_1206_0675_b200/slab.py) on the CPU:
world_size 2 and 3 over gloo against the in-process LocalExchange, and the all-to-all against the buffer layout
include/lgf.h documents for lgf_slab_fft_forward / _t / _inverse ([q][c][tl][zl][y][x], chunk q <-> rank q), modelled here as
plain numpy index shuffles -- data movement only, none of the method's arithmetic.  The kernels that fill and
read those buffers are checked on the GPU (tests/test_gpu_slab.py, with LocalExchange); this file checks that
the torch.distributed plumbing delivers the same chunks to the same places."""
import os
import socket

import numpy as np
import pytest

from paper_1206_0675_b200 import slab


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


# ---- the documented layouts, as numpy ------------------------------------------------------------------
def pack_stage0(Wslab, n):
    """t-slab field [c][T][Lz][Sxy] -> send buffer [c][q][tl][zl][xy], z = q Zl + zl."""
    C, T, Lz, S = Wslab.shape
    Zl = Lz // n
    return np.ascontiguousarray(Wslab.reshape(C, T, n, Zl, S).transpose(0, 2, 1, 3, 4)).reshape(-1)


def unpack_stage1(buf, n, C, T, Zl, S):
    """receive buffer [c][q][tl][zl][xy] -> z-slab field [c][t = q T + tl][zl][xy]."""
    return buf.reshape(C, n * T, Zl, S).copy()              # (a copy: the buffer is reused by the next exchange)


def pack_stage2(Wz, n):
    C, Lt, Zl, S = Wz.shape
    T = Lt // n
    return Wz.reshape(-1).copy()                               # [c][q][tl][zl][xy] with t = q T + tl: the field as it stands


def unpack_stage3(buf, n, C, T, Zl, S):
    return np.ascontiguousarray(buf.reshape(C, n, T, Zl, S).transpose(0, 2, 1, 3, 4)).reshape(C, T, n * Zl, S)


def global_field(C, Lt, Lz, S):
    return np.arange(C * Lt * Lz * S, dtype=np.float64).reshape(C, Lt, Lz, S) * 0.5 + 1.0


def test_slab_of_is_a_contiguous_t_slice():
    import torch

    U = torch.arange(8 * 2 * 3).reshape(8, 2, 3)
    parts = [slab.slab_of(U, r, 4) for r in range(4)]
    assert all(p.is_contiguous() and p.shape[0] == 2 for p in parts)
    assert torch.equal(torch.cat(parts), U)
    with pytest.raises(ValueError):
        slab.slab_of(U, 0, 3)


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_local_exchange_round_trip(n):
    """t-slabs -> z-slabs -> t-slabs through LocalExchange and the documented layouts is the identity, and the
    z-slab a rank holds in between is the right piece of the global field."""
    import torch

    C, Lt, Lz, S = 4, 2 * n, 3 * n, 5
    T, Zl = Lt // n, Lz // n
    W = global_field(C, Lt, Lz, S)
    ex = slab.LocalExchange(n)
    send = [torch.from_numpy(pack_stage0(W[:, r * T:(r + 1) * T], n)) for r in range(n)]
    recv = [torch.empty_like(s) for s in send]
    ex.all_to_all(send, recv)
    Wz = [unpack_stage1(recv[r].numpy(), n, C, T, Zl, S) for r in range(n)]
    for r in range(n):
        assert np.array_equal(Wz[r], W[:, :, r * Zl:(r + 1) * Zl])
    send = [torch.from_numpy(pack_stage2(Wz[r], n)) for r in range(n)]
    for c in (2, 0, 3, 1):                     # the overlapped form, one component at a time, in any order
        ex.finish(ex.start_all_to_all_comp(send, recv, c))
    for r in range(n):
        assert np.array_equal(unpack_stage3(recv[r].numpy(), n, C, T, Zl, S), W[:, r * T:(r + 1) * T])
    # halos: +1 sends to the rank above (U_t of the last slice), -1 to the rank below (g of the first slice)
    tag = [torch.full((3,), float(r)) for r in range(n)]
    got = [torch.empty(3) for _ in range(n)]
    ex.shift(tag, got, +1)
    assert [int(g[0]) for g in got] == [(r - 1) % n for r in range(n)]
    ex.shift(tag, got, -1)
    assert [int(g[0]) for g in got] == [(r + 1) % n for r in range(n)]
    vals = [torch.tensor([1.0 + r, 10.0 * r], dtype=torch.float64) for r in range(n)]
    ex.all_reduce_sum(vals)
    assert all(v.tolist() == [n + n * (n - 1) / 2, 10.0 * n * (n - 1) / 2] for v in vals)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ex = slab.DistExchange(dist)
        assert ex.world == world and ex.local_ranks == [rank]
        C, Lt, Lz, S = 4, 2 * world, 3 * world, 5
        T, Zl = Lt // world, Lz // world
        W = global_field(C, Lt, Lz, S)
        send = [torch.from_numpy(pack_stage0(W[:, rank * T:(rank + 1) * T], world))]
        recv = [torch.empty_like(send[0])]
        ex.all_to_all(send, recv)
        Wz = unpack_stage1(recv[0].numpy(), world, C, T, Zl, S)
        ok_fwd = bool(np.array_equal(Wz, W[:, :, rank * Zl:(rank + 1) * Zl]))
        send = [torch.from_numpy(pack_stage2(Wz, world))]
        for c in (2, 0, 3, 1):                 # the overlapped form, one component at a time (synchronous on the CPU)
            ex.finish(ex.start_all_to_all_comp(send, recv, c))
        ok_back = bool(np.array_equal(unpack_stage3(recv[0].numpy(), world, C, T, Zl, S), W[:, rank * T:(rank + 1) * T]))
        tag, got = [torch.full((3,), float(rank))], [torch.empty(3)]
        ex.shift(tag, got, +1)
        up = int(got[0][0])
        ex.shift(tag, got, -1)
        down = int(got[0][0])
        vals = [torch.tensor([1.0 + rank, 10.0 * rank], dtype=torch.float64)]
        ex.all_reduce_sum(vals)
        dist.barrier()
        q.put((rank, ok_fwd, ok_back, up, down, vals[0].tolist()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_dist_exchange_gloo(world):
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n = world
    for rank, ok_fwd, ok_back, up, down, sums in res:
        assert ok_fwd and ok_back
        assert up == (rank - 1) % n and down == (rank + 1) % n
        assert sums == [n + n * (n - 1) / 2, 10.0 * n * (n - 1) / 2]
