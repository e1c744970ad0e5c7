"""-m "not gpu": host-side harness logic that both the oracle and the CUDA path are fed from."""
import numpy as np
import pytest

from paper_1609_08621_b200 import inputs


def test_pp_leaves_round_trip_and_compression(cfg1):
    p = cfg1
    off, idx = inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)
    assert off[0] == 0 and off[-1] == idx.shape[0] and np.all(np.diff(off) >= 1)      # own bucket is always listed
    assert idx.min() >= 0 and idx.max() < p.n_buckets
    eo, ei = inputs.expand_leaves(p.first, p.count, off, idx)
    assert np.array_equal(eo, p.pp_off) and np.array_equal(ei, p.pp_idx)
    assert int(p.count[idx].sum()) == p.pp_idx.shape[0]
    # every bucket's own reference is in its own list (self pairs are skipped by index in the kernels)
    for b in (0, 7, p.n_buckets - 1):
        assert b in idx[off[b]:off[b + 1]]


def test_pp_leaves_rejects_partial_buckets(cfg1):
    p = cfg1
    broken = p.pp_idx.copy()
    broken[1] = broken[0]                     # no longer a run of one whole bucket
    with pytest.raises(ValueError):
        inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, broken)


def test_expand_leaves_handles_empty_lists():
    first = np.array([0, 3, 5], np.int32); count = np.array([3, 2, 4], np.int32)
    off = np.array([0, 2, 2, 3], np.int64); idx = np.array([2, 0, 1], np.int32)
    eo, ei = inputs.expand_leaves(first, count, off, idx)
    assert list(eo) == [0, 7, 7, 9]
    assert list(ei) == [5, 6, 7, 8, 0, 1, 2, 3, 4]


def test_configs_are_seeded_and_tree_ordered():
    a = inputs.config3(16); b = inputs.config3(16)
    assert np.array_equal(a.xyzm, b.xyzm) and np.array_equal(a.pp_idx, b.pp_idx) and np.array_equal(a.pc_idx, b.pc_idx)
    # buckets tile the particle array in order (what pkdg_gravity_eval_host's per-chunk copy-back relies on)
    assert a.first[0] == 0 and np.array_equal(a.first[1:], (a.first + a.count)[:-1]) and a.first[-1] + a.count[-1] == a.n
    assert a.count.max() <= 16 and a.count.min() >= 1
