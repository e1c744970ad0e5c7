"""One problem on N ranks: rank 0 owns the host arrays, every
rank receives the read-only arrays by ``dist.broadcast`` (NCCL over NVLink on GPUs, gloo in the CPU test) and
takes the bucket range ``shard.rank_piece`` gives it.  No collective is on the data path afterwards: ranks
write disjoint output rows.  ``bench.py --gpus N`` and ``tests/test_shard_gloo.py`` both call ``distribute``.
"""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np

from . import shard

_ARRAYS = ("xyzm", "cells", "first", "count", "pp_off", "pp_idx", "pc_off", "pc_idx")


def distribute(p, dist, rank: int, world: int, device, torch, pp_weights=None):
    """p: the problem on rank 0 (numpy arrays xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps),
    ignored elsewhere.  Returns (g, piece): g holds the replicated arrays as tensors on `device` plus eps;
    piece is this rank's shard.Piece with pp_idx / pc_idx as views of the replicated tensors and the rebased
    offsets as tensors on `device` (piece.d_pp_off, piece.d_pc_off)."""
    meta = [None]
    if rank == 0:
        meta = [{k: (tuple(getattr(p, k).shape), str(getattr(p, k).dtype)) for k in _ARRAYS} | {"eps": float(p.eps)}]
    if world > 1:
        dist.broadcast_object_list(meta, src=0)
    meta = meta[0]
    g = SimpleNamespace(eps=meta["eps"])
    for k in _ARRAYS:
        shape, dtype = meta[k]
        if rank == 0:
            t = torch.from_numpy(np.ascontiguousarray(getattr(p, k))).to(device)
        else:
            t = torch.empty(shape, dtype=getattr(torch, dtype), device=device)
        if world > 1:
            dist.broadcast(t, src=0)
        setattr(g, k, t)
    # the cut is computed from the (small) count / offset arrays on the host, identically on every rank
    host = SimpleNamespace(first=g.first.cpu().numpy(), count=g.count.cpu().numpy(), pp_off=g.pp_off.cpu().numpy(),
                           pc_off=g.pc_off.cpu().numpy(), pp_idx=g.pp_idx, pc_idx=g.pc_idx)
    w = None
    if pp_weights is not None:
        w = pp_weights(host, g)
    piece = shard.rank_piece(host, rank, world, w)
    piece.d_pp_off = torch.from_numpy(piece.pp_off).to(device)
    piece.d_pc_off = torch.from_numpy(piece.pc_off).to(device)
    return g, piece
