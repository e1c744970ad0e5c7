"""fp64 CPU oracle for the PKDGRAV3 gravity list-evaluation path -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The arithmetic lives in
``pkdg_oracle.c`` (plain C, fp64); this file only builds it with gcc and
marshals numpy arrays through ctypes.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_float, c_int, c_int32, c_int64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pkdg_oracle.c")
_LIB = os.path.join(_HERE, "libpkdg_oracle.so")
TDIM = 13  # ORC_TDIM in pkdg_oracle.c


def build(force: bool = False) -> str:
    """Compile pkdg_oracle.c -> libpkdg_oracle.so (gcc -O2 -fopenmp)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.orc_num_threads.restype = c_int
        L.orc_spline.argtypes = [c_double, POINTER(c_double), POINTER(c_double)]
        L.orc_pp_pair.argtypes = [c_void_p, c_void_p, c_double, c_double, c_void_p, c_void_p]
        L.orc_taylor_coeffs.argtypes = [c_void_p, c_int, c_void_p]
        L.orc_pc_pair.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p]
        L.orc_gravity_eval.restype = c_int
        L.orc_gravity_eval.argtypes = [c_int64, c_void_p, c_int64, c_void_p, c_int32, c_int64,
                                       c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                       c_double, c_void_p, c_int64, c_void_p]
        L.orc_contribution_norms.restype = c_int
        L.orc_contribution_norms.argtypes = L.orc_gravity_eval.argtypes
        L.orc_contribution_norms2.restype = c_int
        L.orc_contribution_norms2.argtypes = L.orc_gravity_eval.argtypes
        L.orc_cc_accumulate.argtypes = [c_void_p, c_void_p, c_void_p]
        L.orc_cp_accumulate.argtypes = [c_void_p, c_void_p, c_double, c_void_p]
        L.orc_local_eval.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
        L.orc_fmm_eval.restype = c_int
        L.orc_fmm_eval.argtypes = [c_int64, c_void_p, c_int64, c_void_p, c_int32, c_int64, c_void_p, c_void_p, c_void_p,
                                   c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
        L.orc_direct_sum.argtypes = [c_int64, c_void_p, c_double, c_void_p, c_int64, c_void_p]
        L.orc_pack_tiles.restype = c_int64
        L.orc_pack_tiles.argtypes = [c_int64, c_void_p, c_void_p, c_void_p, c_void_p]
        L.orc_interactions.restype = c_int64
        L.orc_interactions.argtypes = [c_int64, c_void_p, c_void_p]
        L.orc_chunk_bounds.restype = c_int64
        L.orc_chunk_bounds.argtypes = [c_int64, c_void_p, c_void_p, c_int64, c_void_p]
        L.orc_walk_lists.restype = c_int
        L.orc_walk_lists.argtypes = [c_int64] + [c_void_p] * 10 + [c_int64, c_double, c_double, c_int, c_void_p, c_void_p]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(c_void_p)


def _c(a, dtype):
    if a is None:
        return None
    return np.ascontiguousarray(a, dtype=dtype)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def spline(u: float):
    """(g(u), w(u)) of the cubic-spline softened pair interaction, u = r/h."""
    g, w = c_double(), c_double()
    lib().orc_spline(float(u), ctypes.byref(g), ctypes.byref(w))
    return g.value, w.value


def pp_pair(xt, xs, ms: float, eps: float):
    """Acceleration[3] and potential on a target at xt from one source (xs, ms)."""
    xt = _c(xt, np.float64); xs = _c(xs, np.float64)
    acc = np.zeros(3); pot = np.zeros(1)
    lib().orc_pp_pair(_p(xt), _p(xs), float(ms), float(eps), _p(acc), _p(pot))
    return acc, float(pot[0])


def taylor_coeffs(r, order: int) -> np.ndarray:
    """Table t[a,b,c] = d^k(1/|r|)/(a!b!c!) for |k| <= order (order <= 12)."""
    assert 0 <= order <= TDIM - 1
    r = _c(r, np.float64)
    t = np.zeros((TDIM, TDIM, TDIM))
    lib().orc_taylor_coeffs(_p(r), int(order), _p(t))
    return t


def pc_pair(xt, rec):
    """Acceleration[3] and potential on a target at xt from one canonical 36-float cell record."""
    xt = _c(xt, np.float64); rec = _c(rec, np.float32)
    assert rec.size >= 36
    acc = np.zeros(3); pot = np.zeros(1)
    lib().orc_pc_pair(_p(xt), _p(rec), _p(acc), _p(pot))
    return acc, float(pot[0])


def gravity_eval(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps, sel=None):
    """The whole path in fp64.  Returns out[n_particles,4] (ax,ay,az,phi); rows of particles that
    belong to no evaluated bucket are NaN."""
    xyzm = _c(xyzm, np.float32)
    n = xyzm.shape[0]
    if cells is None:
        cells = np.zeros((0, 36), np.float32)
    cells = _c(cells, np.float32)
    stride = cells.shape[1] if cells.ndim == 2 else 36
    first = _c(first, np.int32); count = _c(count, np.int32)
    pp_off = _c(pp_off, np.int64); pp_idx = _c(pp_idx, np.int32)
    pc_off = _c(pc_off, np.int64); pc_idx = _c(pc_idx, np.int32)
    sel_a = _c(sel, np.int64)
    out = np.full((n, 4), np.nan)
    err = lib().orc_gravity_eval(n, _p(xyzm), cells.shape[0], _p(cells), stride, first.shape[0],
                                 _p(first), _p(count), _p(pp_off), _p(pp_idx), _p(pc_off),
                                 _p(pc_idx), float(eps), _p(sel_a),
                                 0 if sel_a is None else sel_a.shape[0], _p(out))
    if err:
        raise ValueError("oracle: index out of range in buckets or lists")
    return out


def contribution_norms(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps, sel=None, squared=False):
    """S_i = sum over list entries of |a_ij| for the targets of the evaluated buckets (NaN elsewhere).
    kappa_i = S_i / |a_i| is the condition number of the sum a_i.  squared=True: the sum
    of |a_ij|^2 instead (kappa2_i = sqrt(S2_i) / |a_i|, what independent rounding errors grow with)."""
    xyzm = _c(xyzm, np.float32)
    n = xyzm.shape[0]
    if cells is None:
        cells = np.zeros((0, 36), np.float32)
    cells = _c(cells, np.float32)
    stride = cells.shape[1] if cells.ndim == 2 else 36
    first = _c(first, np.int32); count = _c(count, np.int32)
    pp_off = _c(pp_off, np.int64); pp_idx = _c(pp_idx, np.int32)
    pc_off = _c(pc_off, np.int64); pc_idx = _c(pc_idx, np.int32)
    sel_a = _c(sel, np.int64)
    out = np.full(n, np.nan)
    fn = lib().orc_contribution_norms2 if squared else lib().orc_contribution_norms
    err = fn(n, _p(xyzm), cells.shape[0], _p(cells), stride, first.shape[0],
                                       _p(first), _p(count), _p(pp_off), _p(pp_idx), _p(pc_off),
                                       _p(pc_idx), float(eps), _p(sel_a),
                                       0 if sel_a is None else sel_a.shape[0], _p(out))
    if err:
        raise ValueError("oracle: bucket index out of range")
    return out


NLOC = 56  # local-expansion coefficients, |n| <= 5


def local_index():
    """Multi-indices (a, b, c) of the 56 local coefficients in storage order."""
    return [(a, b, n - a - b) for n in range(6) for a in range(n, -1, -1) for b in range(n - a, -1, -1)]


def cc_accumulate(zB, rec, L=None):
    """L (56 fp64, created if None) += local expansion about zB of one source cell (canonical 36-float record)."""
    zB = _c(zB, np.float64); rec = _c(rec, np.float32)
    L = np.zeros(NLOC) if L is None else L
    lib().orc_cc_accumulate(_p(zB), _p(rec), _p(L))
    return L


def cp_accumulate(zB, xs, ms, L=None):
    """L += local expansion about zB of one source particle."""
    zB = _c(zB, np.float64); xs = _c(xs, np.float64)
    L = np.zeros(NLOC) if L is None else L
    lib().orc_cp_accumulate(_p(zB), _p(xs), float(ms), _p(L))
    return L


def local_eval(zB, L, xt):
    """(acc[3], pot) of the local expansion L about zB at xt."""
    zB = _c(zB, np.float64); L = _c(L, np.float64); xt = _c(xt, np.float64)
    acc = np.zeros(3); pot = np.zeros(1)
    lib().orc_local_eval(_p(zB), _p(L), _p(xt), _p(acc), _p(pot))
    return acc, float(pot[0])


def fmm_eval(xyzm, cells, first, count, zB, cc_off, cc_idx, cp_off, cp_idx, out=None, want_L=False):
    """The C-C / C-P part of the path: per bucket, local expansion about zB[b] from its C-C and C-P lists,
    evaluated at the bucket's particles and ADDED to out[n,4] (zeros if None).  Returns out (and L[n_b,56])."""
    xyzm = _c(xyzm, np.float32); n = xyzm.shape[0]
    cells = _c(np.zeros((0, 36), np.float32) if cells is None else cells, np.float32)
    first = _c(first, np.int32); count = _c(count, np.int32); zB = _c(zB, np.float32)
    cc_off = _c(cc_off, np.int64); cc_idx = _c(cc_idx, np.int32); cp_off = _c(cp_off, np.int64); cp_idx = _c(cp_idx, np.int32)
    out = np.zeros((n, 4)) if out is None else out
    assert out.dtype == np.float64 and out.flags["C_CONTIGUOUS"]
    Lout = np.zeros((first.shape[0], NLOC)) if want_L else None
    err = lib().orc_fmm_eval(n, _p(xyzm), cells.shape[0], _p(cells), cells.shape[1] if cells.ndim == 2 else 36,
                             first.shape[0], _p(first), _p(count), _p(zB), _p(cc_off), _p(cc_idx), _p(cp_off), _p(cp_idx),
                             _p(out), _p(Lout))
    if err:
        raise ValueError("oracle: index out of range in buckets or lists")
    return (out, Lout) if want_L else out


def direct_sum(xyzm, eps, targets=None):
    """Softened direct summation over all other particles, for the listed targets (default all)."""
    xyzm = _c(xyzm, np.float32)
    n = xyzm.shape[0]
    t = _c(targets, np.int64)
    nt = n if t is None else t.shape[0]
    out = np.zeros((nt, 4))
    lib().orc_direct_sum(n, _p(xyzm), float(eps), _p(t), nt, _p(out))
    return out


def pack_tiles(off, idx):
    """Packer spec: (tile_off[n_buckets+1] int64, tiles[n_tiles,32] int32 padded with -1)."""
    off = _c(off, np.int64); idx = _c(idx, np.int32)
    nb = off.shape[0] - 1
    tile_off = np.zeros(nb + 1, np.int64)
    nt = lib().orc_pack_tiles(nb, _p(off), _p(idx), _p(tile_off), None)
    tiles = np.empty((nt, 32), np.int32)
    lib().orc_pack_tiles(nb, _p(off), _p(idx), _p(tile_off), _p(tiles))
    return tile_off, tiles


def interactions(count, off) -> int:
    count = _c(count, np.int32); off = _c(off, np.int64)
    return int(lib().orc_interactions(count.shape[0], _p(count), _p(off)))


def chunk_bounds(pp_off, pc_off, max_entries: int) -> np.ndarray:
    pp_off = _c(pp_off, np.int64); pc_off = _c(pc_off, np.int64)
    nb = pp_off.shape[0] - 1
    bounds = np.zeros(nb + 2, np.int64)
    nc = lib().orc_chunk_bounds(nb, _p(pp_off), _p(pc_off), int(max_entries), _p(bounds))
    return bounds[: nc + 1].copy()


def walk_lists(tree, cells, sink_cell, theta, eps, four=False, xyzm=None, leaf_rank=None):
    """The tree walk written out (readings A6, A22): lists of every sink cell.

    tree: dict of first, count, end, isleaf (int32 [n_cells], depth-first pre-order, subtree of k = [k, end[k]))
    and bblo, bbhi (float32 [n_cells, 3]); cells: canonical records (COM, b_max).  sink_cell: the sink cells
    (buckets, or group cells).  Returns [(off, idx)] for P-P, P-C (and C-P, C-C with four=True; xyzm needed).
    leaf_rank: a rejected leaf's P-P entry is leaf_rank[k] (one bucket reference) instead of its particles."""
    i32 = lambda a: _c(a, np.int32)
    first, count, end, isleaf = i32(tree["first"]), i32(tree["count"]), i32(tree["end"]), i32(tree["isleaf"])
    bblo, bbhi = _c(tree["bblo"], np.float32), _c(tree["bbhi"], np.float32)
    cells = _c(cells, np.float32)
    assert cells.ndim == 2 and cells.shape[1] == 36 and cells.shape[0] == first.shape[0]
    sink_cell = i32(sink_cell); ns = sink_cell.shape[0]
    xyzm = _c(xyzm, np.float32); leaf_rank = None if leaf_rank is None else i32(leaf_rank)
    assert not four or xyzm is not None
    nl = 4 if four else 2
    off = [np.zeros(ns + 1, np.int64) for _ in range(nl)]
    OffArr = c_void_p * 4
    offp = OffArr(*([o.ctypes.data for o in off] + [None] * (4 - nl)))
    args = (first.shape[0], _p(first), _p(count), _p(end), _p(isleaf), _p(cells), _p(bblo), _p(bbhi), _p(xyzm),
            _p(leaf_rank), _p(sink_cell), ns, float(theta), float(eps), 1 if four else 0)
    if lib().orc_walk_lists(*args, offp, None) != 0:
        raise ValueError("malformed tree: a sink cell or an end[] out of range")
    idx = [np.empty(int(o[-1]), np.int32) for o in off]
    idxp = OffArr(*([i.ctypes.data for i in idx] + [None] * (4 - nl)))
    lib().orc_walk_lists(*args, offp, idxp)
    return list(zip(off, idx))
