"""-m "not gpu": the multi-GPU path's host logic on CPU, world_size 2, gloo.

Each rank cuts the bucket range with shard.shard_bounds, slices the CSR lists, evaluates ITS buckets
(with the oracle standing in for the device call -- this tests the sharding, not the kernels) and the
ranks' disjoint output rows are summed with an all-reduce; the result must equal the unsharded one.
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
        from paper_1609_08621_b200 import inputs, shard
        p = inputs.config1(2048, seed=11)
        cost = shard.bucket_cost(p.count, p.pp_off, p.pc_off)
        bounds = shard.shard_bounds(cost, world)
        # every rank must derive the same cut
        tb = torch.from_numpy(bounds.copy())
        tmax = tb.clone(); tmin = tb.clone()
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX); dist.all_reduce(tmin, op=dist.ReduceOp.MIN)
        assert torch.equal(tmax, tmin)
        b0, b1 = int(bounds[rank]), int(bounds[rank + 1])
        first, count, ppo, ppi, pco, pci = shard.slice_problem(p.first, p.count, p.pp_off, p.pp_idx, p.pc_off,
                                                               p.pc_idx, b0, b1)
        assert ppo[0] == 0 and pco[0] == 0 and ppo[-1] == ppi.shape[0] and pco[-1] == pci.shape[0]
        part = oracle.gravity_eval(p.xyzm, p.cells, first, count, ppo, ppi, pco, pci, p.eps)
        rows = shard.rank_rows(p.first, p.count, b0, b1)
        mask = np.zeros(p.n, bool); mask[rows] = True
        assert np.all(np.isnan(part[~mask])) and np.all(np.isfinite(part[mask]))   # writes only its own rows
        part = np.where(mask[:, None], part, 0.0)
        owned = torch.from_numpy(mask.astype(np.int64))
        dist.all_reduce(owned)
        assert int(owned.min()) == 1 and int(owned.max()) == 1  # disjoint and complete
        tot = torch.from_numpy(part.copy())
        dist.all_reduce(tot)
        full = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps)
        assert np.array_equal(tot.numpy(), full)               # same per-bucket arithmetic, bit for bit
        share = float(cost[b0:b1].sum()) / float(cost.sum())
        assert abs(share - 1.0 / world) < 0.02, share
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
