"""Multi-GPU plumbing of the CE search: one process per GPU, torch.distributed.

The path has no exchange step: light curves are independent problems (PAPER.md:232-234 batches them for memory
only), so a job is partitioned BY LIGHT CURVE, every rank runs the same gce_ce_search on its own contiguous
slice, and the per-light-curve outputs are concatenated.  No data-path collective exists; the only collectives
are the result gather and the max-over-ranks timing reduction of the benchmark.  This module holds that host
logic and nothing of the method's arithmetic, so it is importable (and tested, world_size 2, gloo) without a
GPU or the CUDA library.
"""
from __future__ import annotations

import numpy as np


def partition_light_curves(lc_offsets, world_size: int):
    """Contiguous light-curve ranges [lo, hi) per rank, balanced by point count (the work of a light curve is
    N x n_p x n_pdot point-folds and the grid is shared, so points are the weight).  Every light curve goes to
    exactly one rank; ranks may be empty when there are fewer light curves than ranks."""
    offs = np.asarray(lc_offsets, dtype=np.int64)
    n_lc = int(offs.shape[0] - 1)
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    total = int(offs[-1]) if n_lc > 0 else 0
    bounds = [0]
    for r in range(1, world_size):
        # first light curve whose start offset reaches r/world of the points, never before the previous bound
        target = total * r / world_size
        b = int(np.searchsorted(offs[:-1], target, side="left")) if n_lc > 0 else 0
        bounds.append(min(max(b, bounds[-1]), n_lc))
    bounds.append(n_lc)
    return [(bounds[r], bounds[r + 1]) for r in range(world_size)]


def shard_arrays(times, mags, lc_offsets, lo: int, hi: int):
    """The CSR slice of light curves [lo, hi): (times, mags, lc_offsets rebased to 0).  Views, no copy."""
    offs = np.asarray(lc_offsets, dtype=np.int64)
    a, b = int(offs[lo]), int(offs[hi])
    return times[a:b], mags[a:b], offs[lo:hi + 1] - a


def gather_per_light_curve(local, n_lc_total: int, ranges, rank: int, dist=None):
    """Concatenate per-light-curve result rows (numpy [n_local, ...]) from all ranks in light-curve order.
    `dist` is torch.distributed (initialised) or None for a single process."""
    local = np.ascontiguousarray(local)
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local
    parts = [None] * dist.get_world_size()
    dist.all_gather_object(parts, local)
    out = np.concatenate([p for p in parts if p.shape[0] > 0], axis=0) if n_lc_total > 0 else local
    assert out.shape[0] == n_lc_total, (out.shape, n_lc_total)
    return out


def reduce_timing(total_ms: float, point_folds: float, dist=None, device=None):
    """Whole-job accounting of the benchmark: (max over ranks of the timed milliseconds, sum over ranks of the
    point-folds processed).  Uses all_reduce MAX / SUM on `device` (the rank's GPU under NCCL, CPU under gloo)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(total_ms), float(point_folds)
    import torch
    t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    pf = torch.tensor([float(point_folds)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(pf, op=dist.ReduceOp.SUM)
    return float(t.item()), float(pf.item())
