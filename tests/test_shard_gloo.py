"""-m "not gpu": the multi-GPU path's host logic on CPU, world_size 2, gloo.

Rank 0 owns the problem; multigpu.distribute (the function bench.py --gpus N calls) broadcasts it and gives
each rank its shard.rank_piece; every rank evaluates ITS buckets (with the oracle standing in for the device
call -- this tests the sharding, not the kernels) and the ranks' disjoint output rows are summed with an
all-reduce; the result must equal the unsharded one bit for bit.
"""
import os
import socket

import numpy as np
import pytest


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, ret):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_1609_08621_b200 import inputs, multigpu, shard
        ref_p = inputs.config1(2048, seed=11)                     # what rank 0 owns (built everywhere only to compare)
        # the function bench.py --gpus N calls: rank 0's arrays are broadcast, every rank takes its piece
        g, piece = multigpu.distribute(ref_p if rank == 0 else None, dist, rank, world, "cpu", torch)
        for k in ("xyzm", "cells", "first", "count", "pp_off", "pc_off"):
            assert np.array_equal(getattr(g, k).numpy(), getattr(ref_p, k)), k   # the broadcast delivered rank 0's bits
        assert g.eps == ref_p.eps
        # list entries are NOT replicated: only the owner holds them whole, every rank holds its own range's
        assert (g.pp_idx is None and g.pc_idx is None) if rank else (g.pp_idx is not None and g.pc_idx is not None)
        for off, got, full in ((ref_p.pp_off, piece.pp_idx, ref_p.pp_idx), (ref_p.pc_off, piece.pc_idx, ref_p.pc_idx)):
            assert np.array_equal(got.numpy(), full[off[piece.b0]:off[piece.b1]])
        # every rank derives the same cut
        tb = torch.from_numpy(piece.bounds.copy())
        tmax = tb.clone(); tmin = tb.clone()
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX); dist.all_reduce(tmin, op=dist.ReduceOp.MIN)
        assert torch.equal(tmax, tmin)
        b0, b1 = piece.b0, piece.b1
        ppi, pci = piece.pp_idx.numpy(), piece.pc_idx.numpy()
        assert piece.pp_off[0] == 0 and piece.pc_off[0] == 0 and piece.pp_off[-1] == ppi.shape[0] and piece.pc_off[-1] == pci.shape[0]
        assert np.array_equal(piece.d_pp_off.numpy(), piece.pp_off) and np.array_equal(piece.d_pc_off.numpy(), piece.pc_off)
        # the oracle stands in for the device call (this tests the sharding, not the kernels)
        part = oracle.gravity_eval(g.xyzm.numpy(), g.cells.numpy(), piece.first, piece.count, piece.pp_off, ppi, piece.pc_off,
                                   pci, g.eps)
        rows = shard.rank_rows(g.first.numpy(), g.count.numpy(), b0, b1)
        mask = np.zeros(ref_p.n, bool); mask[rows] = True
        assert np.all(np.isnan(part[~mask])) and np.all(np.isfinite(part[mask]))   # writes only its own rows
        part = np.where(mask[:, None], part, 0.0)
        owned = torch.from_numpy(mask.astype(np.int64))
        dist.all_reduce(owned)
        assert int(owned.min()) == 1 and int(owned.max()) == 1  # disjoint and complete
        tot = torch.from_numpy(part.copy())
        dist.all_reduce(tot)
        p = ref_p
        full = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
        assert np.array_equal(tot.numpy(), full)               # same per-bucket arithmetic, bit for bit
        share = piece.cost / piece.cost_total
        assert abs(share - 1.0 / world) < 0.02, share
        # leaf-form P-P lists: references stay GLOBAL bucket indices in a piece; the cost model weighs them
        lo, li = inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)
        import copy
        q = copy.copy(p); q.pp_off, q.pp_idx = lo, li
        lp = shard.rank_piece(q, rank, world, pp_weights=p.count[li])
        assert np.array_equal(lp.bounds, piece.bounds)          # same cut as with particle lists
        eo, ei = inputs.expand_leaves(p.first, p.count, lp.pp_off, lp.pp_idx)
        assert np.array_equal(eo, piece.pp_off) and np.array_equal(ei, ppi)
        ret[rank] = (b0, b1, share)
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_and_reassemble():
    import torch.multiprocessing as mp
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    ret = ctx.Manager().dict()
    procs = [ctx.Process(target=_worker, args=(r, world, port, ret)) for r in range(world)]
    for q in procs:
        q.start()
    for q in procs:
        q.join(180)
        assert q.exitcode == 0
    assert ret[0][0] == 0 and ret[0][1] == ret[1][0]


@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_shard_bounds_properties(world):
    from paper_1609_08621_b200 import shard
    rng = np.random.default_rng(world)
    cost = rng.integers(0, 1000, 500).astype(np.int64)
    b = shard.shard_bounds(cost, world)
    assert b[0] == 0 and b[-1] == 500 and np.all(np.diff(b) >= 0)
    loads = np.array([cost[b[r]:b[r + 1]].sum() for r in range(world)])
    assert loads.sum() == cost.sum()
    assert loads.max() <= cost.sum() / world + cost.max()
    # degenerate inputs
    assert list(shard.shard_bounds(np.zeros(0, np.int64), 4)) == [0, 0, 0, 0, 0]
    z = shard.shard_bounds(np.zeros(10, np.int64), 2)
    assert z[0] == 0 and z[-1] == 10
    one = shard.shard_bounds(np.array([5], np.int64), 3)
    assert one[0] == 0 and one[-1] == 1 and np.all(np.diff(one) >= 0)
