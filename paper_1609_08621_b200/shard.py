"""Multi-GPU sharding of the list-evaluation path.

Buckets are independent units of work: they read shared read-only arrays (particles, cells) and
write disjoint output rows (PAPER.md:L65 sinks are walked independently; L99 GPU work packages are
independent).  So N ranks shard the bucket range; no data-path collective is needed.  This module
holds the HOST logic only (numpy): where to cut, and how to cut the CSR lists.  ``rank_piece`` is
the ONE function that decides what a rank evaluates: ``bench.py --gpus N`` and the world_size-2
gloo test both call it, and each rank then hands its piece to ``Context.gravity_eval_range`` (full
bucket arrays + its bucket range, so P-P leaf references keep indexing the global buckets).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

# cost model: flops per (sink, list entry) as executed by the default kernel
W_PP = 19
W_PC = 167


def bucket_cost(count, pp_off, pc_off, pp_weights=None):
    """Per-bucket cost n_t (W_PP L_pp + W_PC L_pc), int64.  pp_weights: per-entry source count of a leaf-form
    P-P list (count of the referenced bucket); None = one particle per entry."""
    count = np.asarray(count, np.int64)
    if pp_off is None:
        lpp = 0
    elif pp_weights is None:
        lpp = np.diff(np.asarray(pp_off, np.int64))
    else:
        csum = np.concatenate([[0], np.cumsum(np.asarray(pp_weights, np.int64))])
        lpp = csum[np.asarray(pp_off, np.int64)[1:]] - csum[np.asarray(pp_off, np.int64)[:-1]]
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


def slice_lists(pp_off, pp_idx, pc_off, pc_idx, b0: int, b1: int):
    """CSR lists of buckets [b0, b1), offsets rebased to start at 0 (idx are views)."""
    def cut(off, idx):
        if off is None:
            return None, None
        off = np.asarray(off)
        lo, hi = int(off[b0]), int(off[b1])
        return (off[b0:b1 + 1] - lo).astype(np.int64), (None if idx is None else idx[lo:hi])   # idx None: offsets only
    ppo, ppi = cut(pp_off, pp_idx)
    pco, pci = cut(pc_off, pc_idx)
    return ppo, ppi, pco, pci


@dataclass
class Piece:
    """What one rank evaluates: buckets [b0, b1) of the global problem."""
    rank: int
    world: int
    b0: int
    b1: int
    first: np.ndarray          # [b1-b0] sinks of the range (views of the global arrays)
    count: np.ndarray
    pp_off: np.ndarray | None  # [b1-b0+1], rebased to 0
    pp_idx: np.ndarray | None
    pc_off: np.ndarray | None
    pc_idx: np.ndarray | None
    cost: int                  # modelled flops of the piece
    cost_total: int            # of the whole problem
    bounds: np.ndarray         # all ranks' cut points

    @property
    def n_buckets(self): return self.b1 - self.b0


def rank_piece(p, rank: int, world: int, pp_weights=None) -> Piece:
    """The piece of problem `p` (anything with first, count, pp_off, pp_idx, pc_off, pc_idx) that `rank` of
    `world` evaluates: cost-balanced contiguous bucket range + its lists.  Same result on every rank."""
    if not 0 <= rank < world:
        raise ValueError("rank outside [0, world)")
    cost = bucket_cost(p.count, p.pp_off, p.pc_off, pp_weights)
    bounds = shard_bounds(cost, world)
    b0, b1 = int(bounds[rank]), int(bounds[rank + 1])
    ppo, ppi, pco, pci = slice_lists(p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, b0, b1)
    return Piece(rank=rank, world=world, b0=b0, b1=b1, first=p.first[b0:b1], count=p.count[b0:b1], pp_off=ppo,
                 pp_idx=ppi, pc_off=pco, pc_idx=pci, cost=int(cost[b0:b1].sum()), cost_total=int(cost.sum()),
                 bounds=bounds)


def rank_rows(first, count, b0: int, b1: int) -> np.ndarray:
    """Output rows (particle indices) the range [b0, b1) writes."""
    f = np.asarray(first[b0:b1], np.int64)
    c = np.asarray(count[b0:b1], np.int64)
    if f.size == 0:
        return np.zeros(0, np.int64)
    return np.repeat(f - np.concatenate([[0], np.cumsum(c)[:-1]]), c) + np.arange(int(c.sum()))
