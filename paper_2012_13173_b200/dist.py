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


# ---------------------------------------------------------------------------------------------
# One problem over several GPUs (SURVEY.md 8e i / 8f NEXT-4): every rank owns a band of target
# rows and the samples that can reach it.  Outputs of the bands are disjoint, so there is no
# collective on the data path -- only the samples within the support radius of a band edge are
# seen by two ranks (the halo).  The selection below is by latitude only and is a SUPERSET of
# what the band needs; the library drops what cannot reach its target anyway (step a2).
def row_band(ny: int, world: int, rank: int, align: int = 1):
    """Rows [iy0, iy1) of rank `rank`: contiguous bands, sizes differing by at most `align` rows,
    boundaries on multiples of `align` (the tile height, so every band is tiled like the whole)."""
    units = (ny + align - 1) // align
    lo = (units * rank) // world
    hi = (units * (rank + 1)) // world
    return min(lo * align, ny), min(hi * align, ny)


def band_target(target, iy0: int, iy1: int):
    """The plate-carree target restricted to rows [iy0, iy1): same columns, same cell centres."""
    from .workloads import CarTarget
    return CarTarget(target.nx, iy1 - iy0, target.lon0, target.lat0 + iy0 * target.dlat, target.dlon, target.dlat)


def band_sample_mask(lat_deg, target, iy0: int, iy1: int, radius_deg: float, margin_deg: float = 0.0):
    """Boolean mask (numpy or torch, like `lat_deg`) of the samples whose latitude lies within
    radius + margin of the band's rows: every sample that can contribute to the band is kept
    (great-circle distance >= latitude difference)."""
    a = target.lat0 + iy0 * target.dlat
    b = target.lat0 + (iy1 - 1) * target.dlat
    lo, hi = min(a, b) - radius_deg - margin_deg, max(a, b) + radius_deg + margin_deg
    return (lat_deg >= lo) & (lat_deg <= hi)
