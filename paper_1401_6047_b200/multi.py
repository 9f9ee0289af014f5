"""One process per GPU: how the path is spread over ranks.

The hot path has no exchange step between independent systems, so N ranks run N independent shards with NO
data-path collective.  torch.distributed carries only the measurement plumbing: a barrier on both sides of
the timed region and the max over ranks of the device-side time.  Everything here works with the gloo
backend on CPU as well (tests/test_multirank_cpu.py) -- it holds none of the method's arithmetic.
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple

from . import workloads as W


def dist_env() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) without it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_workload(index: int, rank: int) -> W.Workload:
    """Weak scaling: every rank advances its own full-size copy of BASELINE config `index`; rank r shifts
    E_dc by 0.01 r so the replicas are distinct parameter points of a sweep."""
    w = W.get(index)
    if rank > 0:
        for p in w.params:
            p.E_dc = p.E_dc + 0.01 * rank
    return w


def shard_systems(n_batch: int, rank: int, world: int) -> range:
    """Strong scaling of a batch: the contiguous block of system indices rank `rank` owns (sizes differ by at
    most one; empty when there are more ranks than systems)."""
    base, extra = divmod(n_batch, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def shard_workload(w: W.Workload, rank: int, world: int) -> W.Workload:
    """The sub-batch of `w` owned by `rank` (same lattice and dt; per-system parameters untouched)."""
    idx = shard_systems(w.grid.n_batch, rank, world)
    ps = [w.params[i] for i in idx]
    longest = max([p.n_steps_total for p in ps], default=0)
    return W.Workload(name=f"{w.name}[{idx.start}:{idx.stop}]",
                      grid=W.Grid(w.grid.n_harm, w.grid.n_phiy, len(ps), w.grid.dt), params=ps,
                      n_steps=longest if longest > 0 else w.n_steps, note=w.note, extra=dict(w.extra))


def barrier(sync_device=None) -> None:
    """dist.barrier() (if a process group exists) followed by a device synchronise."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
    if sync_device is not None:
        import torch
        torch.cuda.synchronize(sync_device)


def max_over_ranks(x: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_rate(units_this_rank: float, seconds_this_rank: float, device="cpu") -> Tuple[float, float]:
    """(units of all ranks / max-over-ranks time, that time): the aggregate throughput bench.py reports."""
    t = max_over_ranks(seconds_this_rank, device)
    return sum_over_ranks(units_this_rank, device) / t, t
