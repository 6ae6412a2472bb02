"""Rank plumbing for `bench.py --gpus N` (torch.distributed; NCCL on GPUs, gloo in the CPU tests).

The hot path shards by simplex: rank r owns a contiguous block of M (simplex_block), the sites
and their index are replicated, and one all-reduce of per-cell (measure, first moment) combines the partial
cells (combine_partial_cells).  Measurement: the slowest rank's device time (max) and the units each rank
processed (sum); rank 0 reports units / max time.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def whole_job_rate(units_local: float, ms_local: float, device=None) -> tuple[float, float]:
    """(units per second of the whole job, max-over-ranks ms).  Works without an initialised group."""
    if not (dist.is_available() and dist.is_initialized()):
        return units_local / (ms_local * 1e-3), ms_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()) / (float(t.item()) * 1e-3), float(t.item())


def shard_of_replicas(n_units: int, rank: int, world: int) -> range:
    """Simple domains (one piece per cell, nothing to partition): every rank owns all units of its own copy."""
    del rank, world
    return range(n_units)


def simplex_block(m: int, rank: int, world: int) -> tuple[int, int]:
    """Rank's contiguous block [begin, end) of the m simplices (vd_options.simplex_begin / simplex_end).

    The path shards by simplex: every piece P_{a,i} is found from seeds inside T_a and positive
    flags on T_a's own pieces, so a rank that owns T_a produces all of its pieces and no pair ever
    migrates.  Sites and their index are replicated.  Blocks differ by at most one simplex."""
    base, extra = divmod(int(m), int(world))
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def combine_partial_cells(measure, centroid, sites):
    """The one exchange step of the sharded path: per-cell partial measure and first moment (measure x centroid)
    summed over ranks (all_reduce: NCCL over NVLink on GPUs, gloo in the CPU tests); centroid = moment / measure,
    the site itself for an empty cell (vd.h).  Tensors [n], [n][dim], [n][dim] on the rank's device; returns the
    combined (measure, centroid).  Without an initialised group it returns its inputs' own combination."""
    moment = centroid * measure[:, None]
    total = measure.clone()
    if dist.is_available() and dist.is_initialized():
        packed = torch.cat([total[:, None], moment], dim=1).contiguous()
        dist.all_reduce(packed, op=dist.ReduceOp.SUM)
        total, moment = packed[:, 0].contiguous(), packed[:, 1:]
    safe = torch.where(total > 0, total, torch.ones_like(total))
    cen = torch.where((total > 0)[:, None], moment / safe[:, None], sites)
    return total, cen
