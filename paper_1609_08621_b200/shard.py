"""Multi-GPU sharding of the list-evaluation path.

Buckets are independent units of work: they read shared read-only arrays (particles, cells) and
write disjoint output rows (PAPER.md:L65 sinks are walked independently; L99 GPU work packages are
independent).  So N ranks shard the bucket range; no data-path collective is needed.  This module
holds the HOST logic only (numpy): where to cut, and how to cut the CSR lists.  Each rank then calls
``Context.gravity_eval`` on its piece.
"""
from __future__ import annotations

import numpy as np

# cost model: flops per (sink, list entry) as executed by the default kernel
W_PP = 19
W_PC = 187


def bucket_cost(count, pp_off, pc_off):
    """Per-bucket cost n_t (W_PP L_pp + W_PC L_pc), int64."""
    count = np.asarray(count, np.int64)
    lpp = np.diff(np.asarray(pp_off, np.int64)) if pp_off is not None else 0
    lpc = np.diff(np.asarray(pc_off, np.int64)) if pc_off is not None else 0
    return count * (W_PP * lpp + W_PC * lpc)


def shard_bounds(cost, world: int) -> np.ndarray:
    """Contiguous (tree-order) bucket ranges of near-equal cost: bounds[r] .. bounds[r+1] for rank r.

    Cut r is placed at the first bucket whose inclusive prefix cost reaches r/world of the total, so the
    result is deterministic, monotone, covers [0, n) exactly and is the same on every rank."""
    cost = np.asarray(cost, np.int64)
    n = cost.shape[0]
    if world < 1:
        raise ValueError("world must be >= 1")
    bounds = np.zeros(world + 1, np.int64)
    bounds[world] = n
    if n == 0 or world == 1:
        return bounds
    pre = np.cumsum(cost)
    total = int(pre[-1])
    if total == 0:  # no work anywhere: split by count
        return (np.arange(world + 1, dtype=np.int64) * n) // world
    for r in range(1, world):
        target = -(-total * r // world)  # ceil
        bounds[r] = min(n, int(np.searchsorted(pre, target, side="left")) + 1)
    bounds[1:world] = np.maximum.accumulate(bounds[1:world])
    return bounds


def slice_problem(first, count, pp_off, pp_idx, pc_off, pc_idx, b0: int, b1: int):
    """Buckets [b0, b1) with their CSR lists rebased to start at 0 (views where possible)."""
    def cut(off, idx):
        if off is None:
            return None, None
        off = np.asarray(off)
        lo, hi = int(off[b0]), int(off[b1])
        return (off[b0:b1 + 1] - lo).astype(np.int64), idx[lo:hi]
    ppo, ppi = cut(pp_off, pp_idx)
    pco, pci = cut(pc_off, pc_idx)
    return first[b0:b1], count[b0:b1], ppo, ppi, pco, pci


def rank_rows(first, count, b0: int, b1: int) -> np.ndarray:
    """Output rows (particle indices) rank [b0, b1) writes."""
    f = np.asarray(first[b0:b1], np.int64)
    c = np.asarray(count[b0:b1], np.int64)
    if f.size == 0:
        return np.zeros(0, np.int64)
    return np.concatenate([np.arange(a, a + k) for a, k in zip(f, c)]) if f.size < 1 << 16 else \
        np.repeat(f - np.concatenate([[0], np.cumsum(c)[:-1]]), c) + np.arange(int(c.sum()))
