"""Multi-GPU plumbing: replicas only.

Gauge fixing is done a posteriori on each configuration of an ensemble, so the units of
work are whole configurations and they are independent: rank r of N fixes the ensemble members
r, r + N, r + 2N, ...  There is no data-path collective.  The only communication is the bookkeeping
below (barrier, max-over-ranks of the device time, sum of the units processed), which works on any
torch.distributed backend (nccl on the GPUs, gloo in the CPU tests).

This module holds none of the method's arithmetic and never touches liblgf or the oracle.
"""
from __future__ import annotations

from typing import List, Optional, Sequence


def member_indices(n_members: int, rank: int, world: int) -> List[int]:
    """Ensemble members owned by `rank` of `world` (round robin: balanced to within one member)."""
    if world < 1 or not (0 <= rank < world) or n_members < 0:
        raise ValueError("bad (n_members, rank, world) = (%r, %r, %r)" % (n_members, rank, world))
    return list(range(rank, n_members, world))


def member_seed_offset(member: int) -> int:
    """`seed_offset` argument of inputs.make_config for ensemble member `member` (member 0 = the
    configuration BASELINE.json names)."""
    if member < 0:
        raise ValueError("negative ensemble member")
    return int(member)


def _device_of(dist, device=None):
    if device is not None:
        return device
    import torch

    return torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")


def max_over_ranks(dist, value: float, device=None) -> float:
    """Max of a per-rank scalar (the device-timed milliseconds of the timed region).  dist=None: identity."""
    if dist is None:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_of(dist, device))
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(dist, value: float, device=None) -> float:
    """Sum of a per-rank count (units processed).  dist=None: identity."""
    if dist is None:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=_device_of(dist, device))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_results(dist, local: Sequence[dict]) -> Optional[List[dict]]:
    """Collect the per-member result records (member index, iterations, F, theta, ...) of every rank on
    rank 0, sorted by member index; other ranks get None.  dist=None: the local list, sorted."""
    if dist is None:
        return sorted(local, key=lambda r: r["member"])
    world, rank = dist.get_world_size(), dist.get_rank()
    bucket = [None] * world if rank == 0 else None
    dist.gather_object(list(local), bucket, dst=0)
    if rank != 0:
        return None
    out = [r for part in bucket for r in part]
    return sorted(out, key=lambda r: r["member"])


def whole_job_rate(dist, units_local: float, ms_local: float, device=None) -> dict:
    """Whole-job throughput = units all ranks processed / max-over-ranks time (bench.py contract)."""
    ms = max_over_ranks(dist, ms_local, device)
    units = sum_over_ranks(dist, units_local, device)
    return {"units": units, "ms": ms, "per_s": units / (ms * 1e-3) if ms > 0 else float("nan")}
