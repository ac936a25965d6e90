"""Multi-GPU plumbing of bench.py.

The hot path has no exchange step: with N ranks every rank grids one independent,
identically shaped problem (weak scaling) and torch.distributed is used only to line the
ranks up and to take the maximum of their timings.  Nothing here touches the method's
arithmetic; the same helpers run on CPU with the gloo backend (tests/test_dist_cpu.py).
"""
from __future__ import annotations

import os
from typing import Sequence


def env_world():
    """(world_size, rank, local_rank) from the torchrun environment (1, 0, 0 without it)."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def barrier(world: int, device_sync=None):
    """Rendezvous of all ranks, then (on a GPU) a device synchronise."""
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    if device_sync is not None:
        device_sync()


def max_over_ranks(values: Sequence[float], world: int, device=None) -> list:
    """Element-wise maximum of `values` over the ranks (a job is as slow as its slowest rank)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_rate(units_per_rank: int, world: int, steps: int, ms_total_max: float) -> float:
    """Units all ranks processed divided by the slowest rank's time."""
    return units_per_rank * world * steps / (ms_total_max * 1e-3)
