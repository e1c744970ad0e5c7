"""One problem on N ranks: rank 0 owns the host arrays.  What every
rank READS IN FULL -- particles, cells, the bucket arrays and the (small) list offsets -- is replicated by
``dist.broadcast`` (NCCL over NVLink on GPUs, gloo in the CPU test); the list ENTRIES, by far the largest arrays
(1.6 GB at N = 2^24), are not: every rank takes the bucket range ``shard.rank_piece`` gives it and receives only
the entries of that range from rank 0 (one ``send`` / ``recv`` per list and rank).  No collective is on the data
path afterwards: ranks write disjoint output rows.  ``bench.py --gpus N`` and ``tests/test_shard_gloo.py`` both
call ``distribute``.
"""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np

from . import shard

_REPLICATED = ("xyzm", "cells", "first", "count", "pp_off", "pc_off")
_SLICED = ("pp_idx", "pc_idx")


def distribute(p, dist, rank: int, world: int, device, torch, pp_weights=None):
    """p: the problem on rank 0 (numpy arrays xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps),
    ignored elsewhere.  Returns (g, piece): g holds the replicated arrays as tensors on `device` plus eps (and, on
    rank 0 only, the full pp_idx / pc_idx it owns anyway); piece is this rank's shard.Piece with pp_idx / pc_idx as
    tensors on `device` holding the entries of ITS bucket range only and the rebased offsets as tensors on `device`
    (piece.d_pp_off, piece.d_pc_off).  pp_weights(host, g) -> per-entry weights of a leaf-form P-P list, evaluated
    on rank 0's full list and broadcast (one int per entry would defeat the purpose: pass None for particle lists)."""
    meta = [None]
    if rank == 0:
        meta = [{k: (tuple(getattr(p, k).shape), str(getattr(p, k).dtype)) for k in _REPLICATED + _SLICED} | {"eps": float(p.eps)}]
    if world > 1:
        dist.broadcast_object_list(meta, src=0)
    meta = meta[0]
    g = SimpleNamespace(eps=meta["eps"])
    for k in _REPLICATED:
        shape, dtype = meta[k]
        if rank == 0:
            t = torch.from_numpy(np.ascontiguousarray(getattr(p, k))).to(device)
        else:
            t = torch.empty(shape, dtype=getattr(torch, dtype), device=device)
        if world > 1:
            dist.broadcast(t, src=0)
        setattr(g, k, t)
    for k in _SLICED:   # the owner keeps its lists on the device; nobody else ever holds them whole
        setattr(g, k, torch.from_numpy(np.ascontiguousarray(getattr(p, k))).to(device) if rank == 0 else None)
    # the cut is computed from the (small) count / offset arrays on the host, identically on every rank
    host = SimpleNamespace(first=g.first.cpu().numpy(), count=g.count.cpu().numpy(), pp_off=g.pp_off.cpu().numpy(),
                           pc_off=g.pc_off.cpu().numpy(), pp_idx=None, pc_idx=None)
    w = None
    if pp_weights is not None:
        host_w = SimpleNamespace(**vars(host)); host_w.pp_idx, host_w.pc_idx = g.pp_idx, g.pc_idx
        cost = [shard.bucket_cost(host.count, host.pp_off, host.pc_off, pp_weights(host_w, g)) if rank == 0 else None]
        if world > 1:
            dist.broadcast_object_list(cost, src=0)
        piece = _piece_from_cost(host, cost[0], rank, world)
    else:
        piece = shard.rank_piece(host, rank, world, w)
    # every rank's entries: rank 0 sends [off[b0_r], off[b1_r]) of each list to rank r, and keeps views of its own
    for k, off in (("pp_idx", host.pp_off), ("pc_idx", host.pc_off)):
        dtype = getattr(torch, meta[k][1])
        if rank == 0:
            full = getattr(g, k)
            for r in range(1, world):
                lo, hi = int(off[piece.bounds[r]]), int(off[piece.bounds[r + 1]])
                if hi > lo:
                    dist.send(full[lo:hi].contiguous(), dst=r)
            mine = full[int(off[piece.b0]):int(off[piece.b1])]
        else:
            n = int(off[piece.b1]) - int(off[piece.b0])
            mine = torch.empty(n, dtype=dtype, device=device)
            if n > 0:
                dist.recv(mine, src=0)
        setattr(piece, k, mine)
    piece.d_pp_off = torch.from_numpy(piece.pp_off).to(device)
    piece.d_pc_off = torch.from_numpy(piece.pc_off).to(device)
    return g, piece


def _piece_from_cost(host, cost, rank: int, world: int):
    """shard.rank_piece with a per-bucket cost computed elsewhere (rank 0, which alone holds the full lists)."""
    bounds = shard.shard_bounds(cost, world)
    b0, b1 = int(bounds[rank]), int(bounds[rank + 1])
    ppo, _, pco, _ = shard.slice_lists(host.pp_off, None, host.pc_off, None, b0, b1)
    return shard.Piece(rank=rank, world=world, b0=b0, b1=b1, first=host.first[b0:b1], count=host.count[b0:b1], pp_off=ppo,
                       pp_idx=None, pc_off=pco, pc_idx=None, cost=int(cost[b0:b1].sum()), cost_total=int(cost.sum()),
                       bounds=bounds)
