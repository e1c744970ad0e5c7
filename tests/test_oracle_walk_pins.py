"""-m "not gpu": pins of the oracle's tree walk (oracle.walk_lists, readings A6 / A22).

The walk is pinned to things that are not itself:
  1. hand-built three-cell trees with the expected lists written down by hand, one case on each side of every
     threshold: centre distance vs b_max,B + RO_k; box gap vs 2 eps; count = 1; k = B; and for the four-list rule
     1.5 RO_B + RO_k (C-C), 1.5 RO_B (C-P);
  2. a numpy evaluation of the written inequality for EVERY (sink, cell) pair of an N ~ 500 tree (no walk, no
     recursion, parents derived here from the pre-order arrays): every listed cell satisfies it, no proper ancestor of
     a listed cell or of a listed leaf does (so the list is the coarsest admissible cover the paper's top-down walk
     stops at), every P-P leaf fails it, and the lists cover every particle exactly once;
  3. the same for group sinks (L69, g = 64) and for the four lists.
Then the fast input generator (paper_1609_08621_b200/inputs/treegen.c, the skip-list loop) is compared with the oracle
walk -- the generator is checked by the oracle, not the other way round.
"""
import numpy as np
import pytest

import oracle
from paper_1609_08621_b200 import inputs


# ------------------------------------------------------------------------------------------------
# 1. hand-built trees: root (cell 0) with two leaves (cells 1, 2); sink B = cell 1
# ------------------------------------------------------------------------------------------------
def _three_cells(dist, bmax_B=0.1, bmax_k=0.07, count_k=3, box_half_B=0.05, box_half_k=0.05):
    """Leaf B at the origin with 2 particles, leaf k at (dist, 0, 0) with count_k particles.  COM, b_max and boxes
    are set BY HAND (the walk reads them from the arrays, it does not recompute them)."""
    nB = 2
    first = np.array([0, 0, nB], np.int32)
    count = np.array([nB + count_k, nB, count_k], np.int32)
    end = np.array([3, 2, 3], np.int32)
    isleaf = np.array([0, 1, 1], np.int32)
    cells = np.zeros((3, 36), np.float32)
    cells[0, :3] = (dist / 2, 0, 0); cells[0, 35] = 10.0          # the root is never acceptable (b_max huge)
    cells[1, :3] = (0, 0, 0); cells[1, 35] = bmax_B
    cells[2, :3] = (dist, 0, 0); cells[2, 35] = bmax_k
    bblo = np.array([[-1, -1, -1], [-box_half_B] * 3, [dist - box_half_k, -box_half_k, -box_half_k]], np.float32)
    bbhi = np.array([[dist + 1, 1, 1], [box_half_B] * 3, [dist + box_half_k, box_half_k, box_half_k]], np.float32)
    xyzm = np.zeros((nB + count_k, 4), np.float32)
    xyzm[nB:, 0] = dist
    tree = dict(first=first, count=count, end=end, isleaf=isleaf, bblo=bblo, bbhi=bbhi)
    return tree, cells, xyzm


def _lists(tree, cells, theta, eps, **kw):
    return [idx.tolist() for _, idx in oracle.walk_lists(tree, cells, np.array([1], np.int32), theta, eps, **kw)]


def test_two_list_rule_on_either_side_of_every_threshold():
    theta = 0.7                      # RO_k = 0.07 / 0.7 = 0.1, threshold distance = b_max,B + RO_k = 0.2
    own = [0, 1]                     # B's own particles are always P-P entries (skipped by index at evaluation)
    far, near = _three_cells(0.2002), _three_cells(0.1998)
    assert _lists(far[0], far[1], theta, 0.0) == [own, [2]]                 # beyond: cell 2 is a P-C source
    assert _lists(near[0], near[1], theta, 0.0) == [own + [2, 3, 4], []]    # inside: its particles, one by one
    # the threshold moves with theta as RO = b_max / theta says: theta = 0.35 -> RO_k = 0.2, threshold 0.3
    mid = _three_cells(0.25)
    assert _lists(mid[0], mid[1], 0.7, 0.0) == [own, [2]] and _lists(mid[0], mid[1], 0.35, 0.0) == [own + [2, 3, 4], []]
    # and with b_max,B alone (not b_max,B / theta): b_max,B = 0.2 -> threshold 0.3 at theta = 0.7
    big = _three_cells(0.25, bmax_B=0.2)
    assert _lists(big[0], big[1], 0.7, 0.0) == [own + [2, 3, 4], []]
    # box gap: boxes [-.05, .05] and [.45, .55] are 0.4 apart; 2 eps = 0.4 (eps 0.2) passes (>=), eps 0.2001 fails
    t = _three_cells(0.5)
    assert _lists(t[0], t[1], theta, 0.2 * (1 - 1e-6)) == [own, [2]]
    assert _lists(t[0], t[1], theta, 0.2001) == [own + [2, 3, 4], []]
    # a cell of ONE particle is never a multipole source, however far
    one = _three_cells(5.0, count_k=1)
    assert _lists(one[0], one[1], theta, 0.0) == [own + [2], []]
    # leaf references: a rejected leaf is ONE entry, its rank; B itself too
    rank = np.array([-1, 0, 1], np.int32)
    assert _lists(near[0], near[1], theta, 0.0, leaf_rank=rank) == [[0, 1], []]
    assert _lists(far[0], far[1], theta, 0.0, leaf_rank=rank) == [[0], [2]]


def test_four_list_rule_on_either_side_of_every_threshold():
    theta = 0.7                      # RO_B = 0.07 / 0.7 = 0.1, RO_k = 0.1: C-C beyond 1.5 RO_B + RO_k = 0.25,
    own = [0, 1]                     # P-C beyond b_max,B + RO_k = 0.17, C-P beyond 1.5 RO_B = 0.15
    kw = dict(four=True)
    def run(dist, **g):
        tree, cells, xyzm = _three_cells(dist, bmax_B=0.07, **g)
        return _lists(tree, cells, theta, 0.0, xyzm=xyzm, **kw)          # [P-P, P-C, C-P, C-C]
    assert run(0.2502) == [own, [], [], [2]]
    assert run(0.2498) == [own, [2], [], []]
    assert run(0.1702) == [own, [2], [], []]
    assert run(0.1698) == [own, [], [2, 3, 4], []]                       # leaf opened: particles beyond 1.5 RO_B are C-P
    assert run(0.1502) == [own, [], [2, 3, 4], []]
    assert run(0.1498) == [own + [2, 3, 4], [], [], []]
    assert run(5.0, count_k=1) == [own, [], [2], []]                     # a single far particle: C-P, never a cell
    # gap rule for a particle: the point must be 2 eps from B's box ([-.05, .05]): at x = 0.16 the gap is 0.11
    tree, cells, xyzm = _three_cells(0.16, bmax_B=0.07)
    assert _lists(tree, cells, theta, 0.05, xyzm=xyzm, **kw) == [own, [], [2, 3, 4], []]
    assert _lists(tree, cells, theta, 0.06, xyzm=xyzm, **kw) == [own + [2, 3, 4], [], [], []]


# ------------------------------------------------------------------------------------------------
# 2. the inequality for every (sink, cell) pair, in numpy, on a real tree
# ------------------------------------------------------------------------------------------------
def _accept_matrices(p, sinks, theta, eps, xyzm=None):
    """A_pc[s, k], A_cc[s, k]: the written rules evaluated for every pair (fp64 on the fp32 inputs)."""
    t = p.tree
    com = p.cells[:, :3].astype(np.float64); bmax = p.cells[:, 35].astype(np.float64)
    lo = t["bblo"].astype(np.float64); hi = t["bbhi"].astype(np.float64)
    d = np.sqrt(((com[sinks][:, None, :] - com[None, :, :]) ** 2).sum(-1))
    g = np.maximum(0.0, np.maximum(lo[None, :, :] - hi[sinks][:, None, :], lo[sinks][:, None, :] - hi[None, :, :]))
    gap_ok = (g ** 2).sum(-1) >= (2 * eps) ** 2
    base = gap_ok & (t["count"][None, :] >= 2) & (np.arange(com.shape[0])[None, :] != np.asarray(sinks)[:, None])
    RO = bmax / theta
    A_pc = base & (d > bmax[sinks][:, None] + RO[None, :])
    A_cc = base & (d > 1.5 * RO[sinks][:, None] + RO[None, :])
    return A_pc, A_cc


def _parents(end):
    """parent[k] from the pre-order / subtree-end arrays: the nearest earlier cell whose subtree contains k."""
    parent = np.full(end.shape[0], -1, np.int64)
    stack = []
    for k in range(end.shape[0]):
        while stack and end[stack[-1]] <= k:
            stack.pop()
        if stack:
            parent[k] = stack[-1]
        stack.append(k)
    return parent


def _ancestors(parent, k):
    out = []
    k = parent[k]
    while k >= 0:
        out.append(k); k = parent[k]
    return out


def _small_problem(mode, seed):
    xyzm = inputs.particles_plummer_mix(512, seed, n_spheres=3, a=0.05) if mode == "binary" else inputs.particles_uniform(512, seed)
    return inputs.build_tree(xyzm, mode, 16)


@pytest.mark.parametrize("mode,theta,eps,groups", [("octree", 0.7, 1e-3, False), ("binary", 0.55, 4e-3, False),
                                                   ("binary", 0.7, 1e-3, True), ("octree", 0.4, 0.0, False)])
def test_two_list_walk_is_the_coarsest_admissible_cover(mode, theta, eps, groups):
    p = _small_problem(mode, 7)
    t = p.tree
    sinks = inputs.build_groups(p)[0] if groups else t["leaf_cell"].astype(np.int32)
    (pp_off, pp_idx), (pc_off, pc_idx) = oracle.walk_lists(t, p.cells, sinks, theta, eps)
    A, _ = _accept_matrices(p, sinks, theta, eps)
    parent = _parents(t["end"])
    leaf_of = np.full(p.n, -1, np.int64)
    for k in np.flatnonzero(t["isleaf"] != 0):
        leaf_of[t["first"][k]: t["first"][k] + t["count"][k]] = k
    assert A.any() and (~A).any()
    n_pc = 0
    for s in range(len(sinks)):
        cells = pc_idx[pc_off[s]:pc_off[s + 1]]
        parts = pp_idx[pp_off[s]:pp_off[s + 1]]
        n_pc += len(cells)
        assert A[s, cells].all()                                              # (i) every listed cell satisfies the rule
        for k in cells:
            assert not A[s, _ancestors(parent, k)].any()                      # (ii) none of its ancestors does
        leaves = np.unique(leaf_of[parts])
        for k in leaves:
            assert not A[s, k] and not A[s, _ancestors(parent, k)].any()      # (iii) P-P leaves fail it, all the way up
            assert np.isin(np.arange(t["first"][k], t["first"][k] + t["count"][k]), parts).all()   # a leaf joins whole
        covered = np.zeros(p.n, np.int64)                                     # (iv) every particle exactly once
        np.add.at(covered, parts, 1)
        for k in cells:
            covered[t["first"][k]: t["first"][k] + t["count"][k]] += 1
        assert (covered == 1).all()
    assert n_pc > 0


@pytest.mark.parametrize("mode,theta,eps", [("octree", 0.7, 1e-3), ("binary", 0.55, 2e-3)])
def test_four_list_walk_is_the_coarsest_admissible_cover(mode, theta, eps):
    p = _small_problem(mode, 11)
    t = p.tree
    sinks = t["leaf_cell"].astype(np.int32)
    (pp_off, pp_idx), (pc_off, pc_idx), (cp_off, cp_idx), (cc_off, cc_idx) = oracle.walk_lists(
        t, p.cells, sinks, theta, eps, four=True, xyzm=p.xyzm)
    A_pc, A_cc = _accept_matrices(p, sinks, theta, eps)
    parent = _parents(t["end"])
    com = p.cells[:, :3].astype(np.float64); RO = p.cells[:, 35].astype(np.float64) / theta
    x = p.xyzm[:, :3].astype(np.float64)
    lo = t["bblo"].astype(np.float64); hi = t["bbhi"].astype(np.float64)
    assert len(cc_idx) > 0 and len(cp_idx) > 0 and len(pc_idx) > 0
    for s, B in enumerate(sinks):
        cc = cc_idx[cc_off[s]:cc_off[s + 1]]; pc = pc_idx[pc_off[s]:pc_off[s + 1]]
        cp = cp_idx[cp_off[s]:cp_off[s + 1]]; pp = pp_idx[pp_off[s]:pp_off[s + 1]]
        assert A_cc[s, cc].all()                                              # C-C entries pass the 1.5 RO_B + RO_k rule
        assert A_pc[s, pc].all() and not A_cc[s, pc].any()                    # P-C entries pass A6 but not the C-C rule
        for k in np.concatenate([cc, pc]):
            anc = _ancestors(parent, k)
            assert not A_pc[s, anc].any() and not A_cc[s, anc].any()
        # particles: C-P iff outside B, beyond 1.5 RO_B from COM_B and 2 eps from B's box
        dj = np.sqrt(((x - com[B]) ** 2).sum(-1))
        gj = np.maximum(0.0, np.maximum(x - hi[B], lo[B] - x))
        inB = (np.arange(p.n) >= t["first"][B]) & (np.arange(p.n) < t["first"][B] + t["count"][B])
        rule = ~inB & (dj > 1.5 * RO[B]) & ((gj ** 2).sum(-1) >= (2 * eps) ** 2)
        assert rule[cp].all() and not rule[pp].any()
        covered = np.zeros(p.n, np.int64)
        np.add.at(covered, pp, 1); np.add.at(covered, cp, 1)
        for k in np.concatenate([cc, pc]):
            covered[t["first"][k]: t["first"][k] + t["count"][k]] += 1
        assert (covered == 1).all()


def test_walk_order_is_node_left_right():
    """cells are visited node-left-right, so list entries come in ascending pre-order index."""
    p = inputs.config1(n=2048, seed=3)
    for off, idx in oracle.walk_lists(p.tree, p.cells, p.tree["leaf_cell"], 0.7, p.eps):
        for s in range(len(off) - 1):
            assert (np.diff(idx[off[s]:off[s + 1]]) > 0).all()


def test_malformed_trees_are_refused():
    p = inputs.config1(n=512, seed=3)
    with pytest.raises(ValueError):
        oracle.walk_lists(p.tree, p.cells, np.array([p.cells.shape[0]], np.int32), 0.7, p.eps)
    bad = dict(p.tree); bad["end"] = p.tree["end"].copy(); bad["end"][4] = 4
    with pytest.raises(ValueError):
        oracle.walk_lists(bad, p.cells, p.tree["leaf_cell"], 0.7, p.eps)


# ------------------------------------------------------------------------------------------------
# 3. the input generator's fast walks against the oracle walk (the generator is what is being checked)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("make,theta", [(lambda: inputs.config1(), 0.7), (lambda: inputs.config2(n=1 << 13, seed=5), 0.55),
                                        (lambda: inputs.config3(16), 0.7)])
def test_generator_lists_equal_the_oracle_walk(make, theta):
    p = make()
    if theta != p.theta:
        p = inputs.with_lists(p, theta, p.eps)
    t = p.tree
    (pp_off, pp_idx), (pc_off, pc_idx) = oracle.walk_lists(t, p.cells, t["leaf_cell"], theta, p.eps)
    for a, b in zip((pp_off, pp_idx, pc_off, pc_idx), (p.pp_off, p.pp_idx, p.pc_off, p.pc_idx)):
        assert np.array_equal(a, b)
    # group-shared lists (L69: the walk stops at cells of up to g = 64 particles)
    gc, gf, gn = inputs.build_groups(p)
    want = inputs.build_group_lists(p, gc, theta, p.eps)
    got = oracle.walk_lists(t, p.cells, gc, theta, p.eps)
    assert all(np.array_equal(a, b) for a, b in zip((got[0][0], got[0][1], got[1][0], got[1][1]), want))
    # leaf-form P-P entries
    rank = (np.cumsum(t["isleaf"] != 0) - 1).astype(np.int32)
    lo, li = inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)
    got = oracle.walk_lists(t, p.cells, t["leaf_cell"], theta, p.eps, leaf_rank=rank)
    assert np.array_equal(got[0][0], lo) and np.array_equal(got[0][1], li) and np.array_equal(got[1][1], p.pc_idx)
    # four lists (reading A22)
    f = inputs.build_fmm_lists(p, theta, p.eps)
    got = oracle.walk_lists(t, p.cells, t["leaf_cell"], theta, f["eps"], four=True, xyzm=p.xyzm)
    for q, name in enumerate(("pp", "pc", "cp", "cc")):
        assert np.array_equal(got[q][0], f[name][0]) and np.array_equal(got[q][1], f[name][1]), name
