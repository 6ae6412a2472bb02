"""Rank plumbing for `bench.py --gpus N` (torch.distributed; NCCL on GPUs, gloo in the CPU tests).

The hot path shards by simplex: rank r owns a contiguous block of M (simplex_block), the sites
and their index are replicated, and one all-reduce of per-cell (measure, first moment) combines the partial
cells (combine_partial_cells: the packing and the division run in the library's kernels -- vd_partial_moments /
vd_finish_centroids --, this module only calls all_reduce).  Measurement: the slowest rank's device time (max) and the units each rank
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


def simplex_block(m: int, rank: int, world: int) -> tuple[int, int]:
    """Rank's contiguous block [begin, end) of the m simplices (vd_options.simplex_begin / simplex_end).

    The path shards by simplex: every piece P_{a,i} is found from seeds inside T_a and positive
    flags on T_a's own pieces, so a rank that owns T_a produces all of its pieces and no pair ever
    migrates.  Sites and their index are replicated.  Blocks differ by at most one simplex."""
    base, extra = divmod(int(m), int(world))
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def all_reduce_sums(packed):
    """The one exchange step of the sharded path: per-cell (measure, first moment) rows [n][1 + dim], summed over
    the ranks in place (all_reduce: NCCL over NVLink on GPUs, gloo in the CPU tests).  No group: unchanged."""
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(packed, op=dist.ReduceOp.SUM)
    return packed


def combine_partial_cells(ctx, buf=None):
    """After ctx.compute() on this rank's block of M: vd_partial_moments packs (measure, measure x centroid) per cell
    into a device buffer, one all-reduce sums it over the ranks, vd_finish_centroids rewrites the context's measure /
    centroid arrays from the sums (centroid = moment / measure, the site itself for an empty cell) -- every rank then
    holds the whole diagram's measures and centroids.  Returns the buffer (pass it back in to reuse it)."""
    if buf is None:
        buf = torch.empty((ctx.n, 1 + ctx.dim), dtype=torch.float64, device=torch.device("cuda", torch.cuda.current_device()))
    ctx.partial_moments(buf.data_ptr())
    all_reduce_sums(buf)
    ctx.finish_centroids(buf.data_ptr())
    return buf


def simplex_blocks_balanced(sites, verts, simplices, world: int, grid: int = 0):
    """Contiguous blocks of M with about equal WORK instead of equal simplex count ("balanced by an
    estimate of pairs (sites per simplex + 1)").  The number of pieces of T_a is about 1 + the number of sites
    near it; that is estimated from a coarse histogram of the sites (grid^d bins of ~64 sites over the joint bounding box):
    density at the simplex's centroid times the simplex's measure, plus a fringe term.  Returns [(begin, end)] * world, the
    same on every rank (numpy only, deterministic).  Clustered sites (BASELINE config 3) make equal-count blocks
    differ several-fold in pairs."""
    import numpy as np
    s = np.asarray(sites, np.float64)
    v = np.asarray(verts, np.float64)
    t = np.asarray(simplices)
    m, d = t.shape[0], s.shape[1]
    if grid <= 0:   # ~64 sites per bin: a density estimate, not noise
        grid = int(min(64, max(2, round((s.shape[0] / 64.0) ** (1.0 / d)))))
    lo = np.minimum(s.min(0), v.min(0))
    hi = np.maximum(s.max(0), v.max(0))
    ext = np.where(hi > lo, hi - lo, 1.0)
    bins = np.minimum((np.clip((s - lo) / ext, 0.0, 1.0) * grid).astype(np.int64), grid - 1)
    flat = np.ravel_multi_index(tuple(bins.T), (grid,) * d)
    hist = np.bincount(flat, minlength=grid ** d).astype(np.float64)
    cell_vol = float(np.prod(ext / grid))
    corners = v[t]                                            # [m][k][d]
    cen = corners.mean(1)
    cb = np.minimum((np.clip((cen - lo) / ext, 0.0, 1.0) * grid).astype(np.int64), grid - 1)
    dens = hist[np.ravel_multi_index(tuple(cb.T), (grid,) * d)] / cell_vol
    k = t.shape[1]
    if k == d + 1:      # a d-simplex in R^d: its measure
        e = corners[:, 1:, :] - corners[:, :1, :]
        meas = np.abs(np.linalg.det(e)) / float(np.prod(np.arange(1, d + 1)))
    else:               # a triangle in R^3 (surface): its area times one bin's thickness -- the slab of sites it meets
        e1, e2 = corners[:, 1] - corners[:, 0], corners[:, 2] - corners[:, 0]
        meas = 0.5 * np.linalg.norm(np.cross(e1, e2), axis=1) * float(np.mean(ext / grid))
    inside = dens * meas                                      # expected sites inside T_a
    # cells meeting T_a: the sites inside, a fringe of cells cut by its boundary (~ inside^((d-1)/d)), at least one
    work = 1.0 + inside + 3.0 * inside ** ((d - 1.0) / d)
    cum = np.cumsum(work)
    cuts = [0]
    for r in range(1, world):
        cuts.append(int(np.searchsorted(cum, cum[-1] * r / world)))
    cuts.append(m)
    cuts = [min(max(c, 0), m) for c in cuts]
    for k in range(1, len(cuts)):
        cuts[k] = max(cuts[k], cuts[k - 1])
    return [(cuts[r], cuts[r + 1]) for r in range(world)]
