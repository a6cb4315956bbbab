"""Multi-GPU plumbing: views are independent units, so rank r of a job takes
a contiguous range of views, runs the three C-ABI calls on it, and the only exchanges are the reduction of the
timing / counters and (optionally) a gather of the per-view track counts so that every rank can index the global
track list.  No data-path collective exists.  Works with any torch.distributed backend (nccl on GPUs, gloo in the
CPU tests); without an initialised process group every function is the identity.
"""
from __future__ import annotations

import numpy as np


def view_range(rank: int, world: int, views_per_rank: int):
    """Views [first, first + n) of rank `rank` under weak scaling (every rank owns `views_per_rank` views)."""
    if not (0 <= rank < world) or views_per_rank < 0:
        raise ValueError("bad rank / world / views_per_rank")
    return rank * views_per_rank, views_per_rank


def split_views(n_views: int, world: int, grains_per_view=None):
    """Strong-scaling split of n_views over `world` ranks: contiguous ranges, returned as the list of (first, n) per
    rank.  Without grain counts the sizes differ by at most one.  With `grains_per_view` (length n_views) the ranges
    are balanced by sum N^2 instead (the work of a view goes with its seeds, i.e. with N times the grain
    density): the cut after rank r is placed where the running sum of N^2 comes closest to (r + 1) / world of the total,
    every rank keeping at least one view while views are left."""
    if world < 1 or n_views < 0:
        raise ValueError("bad world / n_views")
    if grains_per_view is None:
        base, extra = divmod(n_views, world)
        out, first = [], 0
        for r in range(world):
            n = base + (1 if r < extra else 0)
            out.append((first, n))
            first += n
        return out
    w = np.asarray(grains_per_view, np.float64) ** 2
    if len(w) != n_views:
        raise ValueError("grains_per_view must have one entry per view")
    cum = np.concatenate(([0.0], np.cumsum(w)))          # cum[k] = weight of views 0..k-1
    cuts = [0]
    for r in range(1, world):
        # the cut closest to r / world of the total weight ...
        target = cum[-1] * r / world
        k = int(np.searchsorted(cum, target))
        if k > 0 and (k > n_views or target - cum[k - 1] <= cum[k] - target):
            k -= 1
        # ... but at least one view for every rank before and after it while views are left
        lo = min(cuts[-1] + 1, n_views)
        hi = max(lo, n_views - (world - r))
        cuts.append(min(max(k, lo), hi))
    cuts.append(n_views)
    return [(cuts[r], cuts[r + 1] - cuts[r]) for r in range(world)]


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def reduce_step(ms_local: float, counters_local, device="cpu"):
    """(max over ranks of the step time, sum over ranks of the integer counters)."""
    import torch
    dist = _dist()
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    c = torch.as_tensor(np.asarray(counters_local, np.int64), device=device).clone()
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), [int(x) for x in c.cpu().tolist()]


def gather_track_off(track_off_local, device="cpu"):
    """Global track_off over all ranks' views (rank order = view order) from every rank's local track_off:
    one all_gather of the per-view track counts (4 B per view).  Every rank must own the same number of views."""
    import torch
    dist = _dist()
    counts = np.diff(np.asarray(track_off_local, np.int64)).astype(np.int32)
    if dist is None:
        allc = counts
    else:
        mine = torch.as_tensor(counts, device=device)
        parts = [torch.empty_like(mine) for _ in range(dist.get_world_size())]
        dist.all_gather(parts, mine)
        allc = np.concatenate([p.cpu().numpy() for p in parts])
    off = np.zeros(len(allc) + 1, np.int64)
    off[1:] = np.cumsum(allc)
    return off
