"""Rank plumbing for `bench.py --gpus N` (torch.distributed; NCCL on GPUs, gloo in the CPU tests).

The hot path does not shard in this round ("replicas only"): every rank runs the whole
workload on its own GPU.  What the ranks exchange is measurement only: the slowest rank's device time
(max) and the units each rank processed (sum); rank 0 reports units / max time.
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
    """Replicas only: every rank owns all units of its own copy of the workload."""
    del rank, world
    return range(n_units)
