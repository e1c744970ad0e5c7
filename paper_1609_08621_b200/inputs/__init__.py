"""Seeded synthetic inputs for the gravity list-evaluation path (harness, never timed).

This module serves BOTH the fp64 oracle and the CUDA library (through the tests and
``bench.py``); it holds none of the method's evaluation arithmetic.  It produces, for
BASELINE.json's five configs, what the hot path consumes: tree-ordered particles
``xyzm``, canonical 36-float cell records, buckets ``{first,count}`` and per-bucket CSR
P-P / P-C lists.  The recipes are stated in DESIGN.md ("Input recipe"); they stand in for
the paper's LambdaCDM snapshots, which are not available offline.

The tree / moment / list code is plain C (``treegen.c``, OpenMP) built in-tree with gcc.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import c_double, c_int, c_int64, c_void_p
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "treegen.c")
_LIB = os.path.join(_HERE, "libpkdg_treegen.so")
REC = 36


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.tg_tree_build.restype = c_void_p
        L.tg_tree_build.argtypes = [c_int64, c_void_p, c_int, c_int]
        L.tg_tree_ncells.restype = c_int64
        L.tg_tree_ncells.argtypes = [c_void_p]
        L.tg_tree_nleaves.restype = c_int64
        L.tg_tree_nleaves.argtypes = [c_void_p]
        L.tg_tree_free.argtypes = [c_void_p]
        L.tg_tree_export.argtypes = [c_void_p] * 10
        L.tg_lists_build.restype = c_void_p
        L.tg_lists_build.argtypes = [c_int64] + [c_void_p] * 8 + [c_int64, c_int64, c_double, c_double]
        L.tg_lists_totals.argtypes = [c_void_p, c_void_p, c_void_p]
        L.tg_lists_export_free.argtypes = [c_void_p] * 5
        L.tg_cloud_records.argtypes = [c_int64, c_int64, c_void_p, c_void_p]
        L.tg_pp_to_leaves.restype = c_int64
        L.tg_pp_to_leaves.argtypes = [c_int64, c_int64, c_void_p, c_void_p, c_int64, c_void_p, c_void_p, c_void_p,
                                      c_void_p]
        L.tg_fmm_build.restype = c_void_p
        L.tg_fmm_build.argtypes = [c_int64] + [c_void_p] * 9 + [c_int64, c_int64, c_double, c_double]
        L.tg_fmm_totals.argtypes = [c_void_p, c_void_p]
        L.tg_fmm_export_free.argtypes = [c_void_p, c_void_p, c_void_p]
        L.tg_num_threads.restype = c_int
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(c_void_p)


# ----------------------------------------------------------------------------- particles
def particles_uniform(n: int, seed: int) -> np.ndarray:
    """Config 1: n equal-mass particles uniform in the unit cube."""
    rng = np.random.Generator(np.random.PCG64(seed))
    out = np.empty((n, 4), np.float32)
    out[:, :3] = rng.random((n, 3), dtype=np.float64).astype(np.float32)
    out[:, 3] = np.float32(1.0 / n)
    return out


def particles_plummer_mix(n: int, seed: int, n_spheres: int = 32, a: float = 0.01,
                          frac: float = 0.7, rmax_a: float = 10.0) -> np.ndarray:
    """Config 2: `frac` of the particles in n_spheres Plummer spheres (scale radius a, equal
    membership, centres uniform in the unit cube, radii rejected beyond rmax_a*a), the rest uniform."""
    rng = np.random.Generator(np.random.PCG64(seed))
    per = int(frac * n) // n_spheres
    centres = rng.random((n_spheres, 3))
    pos = np.empty((n, 3), np.float64)
    k = 0
    for s in range(n_spheres):
        got = 0
        while got < per:
            m = int((per - got) * 1.1) + 16
            u = rng.random(m)
            u = np.clip(u, 1e-12, 1 - 1e-12)
            r = a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
            r = r[r <= rmax_a * a][: per - got]
            mu = rng.uniform(-1.0, 1.0, r.size)
            ph = rng.uniform(0.0, 2 * np.pi, r.size)
            st = np.sqrt(1 - mu * mu)
            pos[k:k + r.size, 0] = centres[s, 0] + r * st * np.cos(ph)
            pos[k:k + r.size, 1] = centres[s, 1] + r * st * np.sin(ph)
            pos[k:k + r.size, 2] = centres[s, 2] + r * mu
            k += r.size
            got += r.size
    pos[k:] = rng.random((n - k, 3))
    out = np.empty((n, 4), np.float32)
    out[:, :3] = pos.astype(np.float32)
    out[:, 3] = np.float32(1.0 / n)
    return out


def _zeldovich_field(ng: int, index: float, seed: int):
    """Three displacement components on an ng^3 periodic mesh, psi = grad inverse-laplacian delta,
    delta Gaussian with P(k) ~ k^index.  Returned in arbitrary units (caller normalises)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    white = rng.standard_normal((ng, ng, ng), dtype=np.float32)
    dk = np.fft.rfftn(white)
    del white
    kx = np.fft.fftfreq(ng, 1.0 / ng).astype(np.float32)
    kz = np.fft.rfftfreq(ng, 1.0 / ng).astype(np.float32)
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    amp = k2 ** (0.25 * index - 1.0)  # sqrt(P) / k^2 = k^(index/2 - 2)
    amp[0, 0, 0] = 0.0
    dk *= amp
    del amp, k2
    psi = []
    for ax in range(3):
        kk = (kx[:, None, None], kx[None, :, None], kz[None, None, :])[ax]
        psi.append(np.fft.irfftn(1j * kk * dk, s=(ng, ng, ng), axes=(0, 1, 2)).astype(np.float32))
    return psi


def particles_zeldovich(ng: int, seed: int, index: float = -2.0, rms_cells: float = 0.3,
                        n_keep: int | None = None, mesh: int | None = None) -> np.ndarray:
    """Configs 3 and 5: an ng^3 lattice (cell centres of the unit box) displaced by a Zel'dovich
    field, rms |psi| = rms_cells lattice cells, wrapped into [0,1).  If `mesh` is given the field
    lives on a mesh^3 grid and is sampled at the nearest mesh point of each site; n_keep keeps the
    first n_keep sites in lexicographic order."""
    m = mesh or ng
    psi = _zeldovich_field(m, index, seed)
    rms = np.sqrt(sum(float(np.mean(p.astype(np.float64) ** 2)) for p in psi))
    scale = rms_cells / rms / ng
    n_all = ng ** 3
    n = n_all if n_keep is None else n_keep
    out = np.empty((n, 4), np.float32)
    idx = np.arange(n, dtype=np.int64)
    ijk = (idx // (ng * ng), (idx // ng) % ng, idx % ng)
    if m == ng:
        flat = idx
    else:
        mi = [np.minimum((c.astype(np.float64) + 0.5) * (m / ng), m - 1).astype(np.int64) for c in ijk]
        flat = (mi[0] * m + mi[1]) * m + mi[2]
    for ax in range(3):
        x = (ijk[ax].astype(np.float64) + 0.5) / ng + psi[ax].reshape(-1)[flat].astype(np.float64) * scale
        x -= np.floor(x)
        xf = x.astype(np.float32)
        xf[xf >= 1.0] = np.float32(0.0)
        out[:, ax] = xf
    out[:, 3] = np.float32(1.0 / n)
    return out


# ----------------------------------------------------------------------------- tree + lists
def _part1by2(x: np.ndarray) -> np.ndarray:
    x = x.astype(np.uint64) & np.uint64(0x1FFFFF)
    x = (x | (x << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
    x = (x | (x << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
    x = (x | (x << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
    x = (x | (x << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
    x = (x | (x << np.uint64(2))) & np.uint64(0x1249249249249249)
    return x


def morton_keys(xyz: np.ndarray, lo: np.ndarray, size: float) -> np.ndarray:
    q = np.floor((xyz.astype(np.float64) - lo) * (2.0 ** 21 / size))
    q = np.clip(q, 0, 2 ** 21 - 1).astype(np.uint64)
    return (_part1by2(q[:, 0]) << np.uint64(2)) | (_part1by2(q[:, 1]) << np.uint64(1)) | _part1by2(q[:, 2])


@dataclass
class Problem:
    """Everything one call of the hot path consumes (host numpy arrays)."""
    name: str
    xyzm: np.ndarray            # [n,4] f32 tree order
    cells: np.ndarray           # [n_cells,36] f32 canonical records
    first: np.ndarray           # [n_b] i32
    count: np.ndarray           # [n_b] i32
    pp_off: np.ndarray | None   # [n_b+1] i64
    pp_idx: np.ndarray | None   # i32
    pc_off: np.ndarray | None
    pc_idx: np.ndarray | None
    eps: float
    theta: float = 0.0
    perm: np.ndarray | None = None      # tree order -> generation order
    tree: dict = field(default_factory=dict)  # cell arrays used by the list builder

    @property
    def n(self): return int(self.xyzm.shape[0])
    @property
    def n_buckets(self): return int(self.first.shape[0])
    @property
    def I_pp(self): return 0 if self.pp_off is None else int(np.dot(self.count.astype(np.int64), np.diff(self.pp_off)))
    @property
    def I_pc(self): return 0 if self.pc_off is None else int(np.dot(self.count.astype(np.int64), np.diff(self.pc_off)))


def build_tree(xyzm_in: np.ndarray, mode: str = "binary", cap: int = 16, name: str = "") -> Problem:
    """Sort particles into tree order and build cells/buckets.  mode: 'octree' or 'binary'."""
    L = _L()
    n = xyzm_in.shape[0]
    xyz = xyzm_in[:, :3]
    lo = xyz.min(axis=0).astype(np.float64)
    hi = xyz.max(axis=0).astype(np.float64)
    if np.all(lo >= 0.0) and np.all(hi <= 1.0):
        lo = np.zeros(3); size = 1.0           # unit cube
    else:
        size = float((hi - lo).max()) * (1 + 1e-6) + 1e-30
        lo = 0.5 * (lo + hi) - 0.5 * size      # bounding cube
    keys = morton_keys(xyz, lo, size)
    perm = np.argsort(keys, kind="stable")
    keys = np.ascontiguousarray(keys[perm])
    xyzm = np.ascontiguousarray(xyzm_in[perm], dtype=np.float32)
    t = L.tg_tree_build(n, _p(keys), 0 if mode == "octree" else 1, cap)
    try:
        nc = L.tg_tree_ncells(t); nl = L.tg_tree_nleaves(t)
        first = np.empty(nc, np.int32); count = np.empty(nc, np.int32); end = np.empty(nc, np.int32)
        isleaf = np.empty(nc, np.int32); rec = np.empty((nc, REC), np.float32)
        bblo = np.empty((nc, 3), np.float32); bbhi = np.empty((nc, 3), np.float32)
        leaf_cell = np.empty(nl, np.int32)
        L.tg_tree_export(t, _p(xyzm), _p(first), _p(count), _p(end), _p(isleaf), _p(rec), _p(bblo),
                         _p(bbhi), _p(leaf_cell))
    finally:
        L.tg_tree_free(t)
    tree = dict(first=first, count=count, end=end, isleaf=isleaf, bblo=bblo, bbhi=bbhi,
                leaf_cell=leaf_cell, mode=mode, cap=cap)
    return Problem(name=name, xyzm=xyzm, cells=rec, first=np.ascontiguousarray(first[leaf_cell]),
                   count=np.ascontiguousarray(count[leaf_cell]), pp_off=None, pp_idx=None, pc_off=None,
                   pc_idx=None, eps=0.0, perm=perm, tree=tree)


def build_lists(p: Problem, theta: float, eps: float, b0: int = 0, b1: int | None = None):
    """CSR P-P / P-C lists for buckets [b0,b1) (offsets relative to b0)."""
    L = _L()
    t = p.tree
    b1 = p.n_buckets if b1 is None else b1
    h = L.tg_lists_build(t["first"].shape[0], _p(t["first"]), _p(t["count"]), _p(t["end"]), _p(t["isleaf"]),
                         _p(p.cells), _p(t["bblo"]), _p(t["bbhi"]), _p(t["leaf_cell"]), b0, b1,
                         float(theta), float(eps))
    npp = c_int64(); npc = c_int64()
    L.tg_lists_totals(h, ctypes.byref(npp), ctypes.byref(npc))
    pp_off = np.empty(b1 - b0 + 1, np.int64); pc_off = np.empty(b1 - b0 + 1, np.int64)
    pp_idx = np.empty(npp.value, np.int32); pc_idx = np.empty(npc.value, np.int32)
    L.tg_lists_export_free(h, _p(pp_off), _p(pp_idx), _p(pc_off), _p(pc_idx))
    return pp_off, pp_idx, pc_off, pc_idx


def build_groups(p: Problem, gmax: int = 64):
    """Groups of sibling buckets (the walk stops at cells of fewer than g = 64 particles and resolves
    the checklist into lists there): the maximal tree cells with at most gmax particles, in tree order.  Returns
    (group_cell int32[n_g], first_bucket int32[n_g], n_buckets int32[n_g]); the groups tile the bucket range."""
    t = p.tree
    count, end, isleaf = t["count"], t["end"].astype(np.int64), t["isleaf"]
    small = (count <= gmax) | (isleaf != 0)                  # a leaf is always a group of its own at least
    e = np.where(small, end, 0)
    covered_to = np.concatenate([[0], np.maximum.accumulate(e)[:-1]])   # end of the last small cell before k
    top = small & (covered_to <= np.arange(count.shape[0]))
    group_cell = np.flatnonzero(top).astype(np.int32)
    leaves_before = np.concatenate([[0], np.cumsum(isleaf != 0)])
    first_bucket = leaves_before[group_cell].astype(np.int32)
    n_buckets = (leaves_before[end[group_cell]] - leaves_before[group_cell]).astype(np.int32)
    return group_cell, first_bucket, n_buckets


def build_group_lists(p: Problem, group_cell: np.ndarray, theta: float, eps: float, g0: int = 0, g1: int | None = None):
    """CSR P-P / P-C lists per GROUP (reading A6 with the group cell as the sink: its centre of mass, b_max and
    bounding box): what every bucket of the group evaluates.  Offsets relative to g0."""
    L = _L()
    t = p.tree
    g1 = group_cell.shape[0] if g1 is None else g1
    gc = np.ascontiguousarray(group_cell, np.int32)
    h = L.tg_lists_build(t["first"].shape[0], _p(t["first"]), _p(t["count"]), _p(t["end"]), _p(t["isleaf"]),
                         _p(p.cells), _p(t["bblo"]), _p(t["bbhi"]), _p(gc), g0, g1, float(theta), float(eps))
    npp = c_int64(); npc = c_int64()
    L.tg_lists_totals(h, ctypes.byref(npp), ctypes.byref(npc))
    pp_off = np.empty(g1 - g0 + 1, np.int64); pc_off = np.empty(g1 - g0 + 1, np.int64)
    pp_idx = np.empty(npp.value, np.int32); pc_idx = np.empty(npc.value, np.int32)
    L.tg_lists_export_free(h, _p(pp_off), _p(pp_idx), _p(pc_off), _p(pc_idx))
    return pp_off, pp_idx, pc_off, pc_idx


def expand_groups(first_bucket: np.ndarray, n_buckets: np.ndarray, g_off: np.ndarray, g_idx: np.ndarray, sel=None):
    """Per-bucket CSR lists the group lists stand for (pure indexing): every bucket of a group gets the group's
    list.  sel: bucket indices to expand (default all, in order).  Returns (off int64[len+1], idx int32)."""
    nb = int(first_bucket[-1] + n_buckets[-1]) if first_bucket.shape[0] else 0
    group_of = np.repeat(np.arange(first_bucket.shape[0]), n_buckets)
    assert group_of.shape[0] == nb
    g = group_of if sel is None else group_of[np.asarray(sel, np.int64)]
    lens = (g_off[1:] - g_off[:-1])[g]
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    start = np.repeat(g_off[:-1][g] - off[:-1], lens)
    idx = g_idx[start + np.arange(int(lens.sum()), dtype=np.int64)]
    return off, np.ascontiguousarray(idx, np.int32)


def f32(x: float) -> float:
    """x rounded to fp32: the C ABI takes the softening as a float, so the harness hands the SAME value to the
    oracle, to the list builder and to the library."""
    return float(np.float32(x))


def build_fmm_lists(p: Problem, theta: float, eps: float, b0: int = 0, b1: int | None = None):
    """FMM-style lists per bucket: a dict of four CSR lists
    'pp', 'pc' (particle-particle / particle-cell, evaluated per sink), 'cp', 'cc' (cell-particle / cell-cell:
    they feed the bucket's local expansion), each (off int64[n+1], idx int32), plus 'centre' float32[n,3], the
    bucket centres of mass the local expansions are taken about."""
    L = _L()
    t = p.tree
    b1 = p.n_buckets if b1 is None else b1
    eps = f32(eps)
    h = L.tg_fmm_build(t["first"].shape[0], _p(t["first"]), _p(t["count"]), _p(t["end"]), _p(t["isleaf"]), _p(p.cells),
                       _p(t["bblo"]), _p(t["bbhi"]), _p(t["leaf_cell"]), _p(p.xyzm), b0, b1, float(theta), float(eps))
    tot = np.zeros(4, np.int64)
    L.tg_fmm_totals(h, _p(tot))
    offs = [np.empty(b1 - b0 + 1, np.int64) for _ in range(4)]
    idxs = [np.empty(int(tot[q]), np.int32) for q in range(4)]
    op = (c_void_p * 4)(*[a.ctypes.data for a in offs]); ip = (c_void_p * 4)(*[a.ctypes.data for a in idxs])
    L.tg_fmm_export_free(h, op, ip)
    out = {k: (offs[q], idxs[q]) for q, k in enumerate(("pp", "pc", "cp", "cc"))}
    out["centre"] = np.ascontiguousarray(p.cells[t["leaf_cell"][b0:b1], :3])
    out["theta"] = theta; out["eps"] = eps
    return out


def with_lists(p: Problem, theta: float, eps: float) -> Problem:
    eps = f32(eps)
    p.pp_off, p.pp_idx, p.pc_off, p.pc_idx = build_lists(p, theta, eps)
    p.theta = theta; p.eps = eps
    return p


def pp_leaves(n_particles: int, gfirst: np.ndarray, gcount: np.ndarray, pp_off: np.ndarray, pp_idx: np.ndarray):
    """P-P lists in leaf form (PKDG_PP_LEAVES): every run of a whole bucket's particles becomes one
    reference to that bucket (index into the GLOBAL bucket arrays gfirst / gcount).  Returns
    (leaf_off int64[n_b+1], leaf_idx int32)."""
    L = _L()
    gfirst = np.ascontiguousarray(gfirst, np.int32); gcount = np.ascontiguousarray(gcount, np.int32)
    pp_off = np.ascontiguousarray(pp_off, np.int64); pp_idx = np.ascontiguousarray(pp_idx, np.int32)
    nb = pp_off.shape[0] - 1
    off = np.empty(nb + 1, np.int64)
    n = L.tg_pp_to_leaves(n_particles, gfirst.shape[0], _p(gfirst), _p(gcount), nb, _p(pp_off), _p(pp_idx), _p(off), None)
    if n < 0:
        raise ValueError("a P-P list is not a sequence of whole buckets")
    idx = np.empty(n, np.int32)
    L.tg_pp_to_leaves(n_particles, gfirst.shape[0], _p(gfirst), _p(gcount), nb, _p(pp_off), _p(pp_idx), _p(off), _p(idx))
    return off, idx


def expand_leaves(gfirst: np.ndarray, gcount: np.ndarray, leaf_off: np.ndarray, leaf_idx: np.ndarray):
    """Inverse of pp_leaves (numpy): the particle-index lists the leaf references stand for."""
    c = gcount[leaf_idx].astype(np.int64)
    per_bucket = np.add.reduceat(np.concatenate([c, [0]]), np.minimum(leaf_off[:-1], c.shape[0]))[: leaf_off.shape[0] - 1]
    per_bucket[np.diff(leaf_off) == 0] = 0
    off = np.concatenate([[0], np.cumsum(per_bucket)]).astype(np.int64)
    start = np.repeat(gfirst[leaf_idx].astype(np.int64) - np.concatenate([[0], np.cumsum(c)[:-1]]), c)
    idx = (start + np.arange(int(c.sum()), dtype=np.int64)).astype(np.int32)
    return off, idx


def cloud_records(pts: np.ndarray, k: int) -> np.ndarray:
    """Canonical records of consecutive k-point clouds of pts[n*k,4]."""
    pts = np.ascontiguousarray(pts, np.float32)
    nc = pts.shape[0] // k
    rec = np.empty((nc, REC), np.float32)
    _L().tg_cloud_records(nc, k, _p(pts), _p(rec))
    return rec


# ----------------------------------------------------------------------------- the five configs
def config1(n: int = 4096, seed: int = 1, theta: float = 0.7) -> Problem:
    """Uniform cube, octree cap 16, eps = 0.02 n^-1/3 (BASELINE.json configs[0])."""
    p = build_tree(particles_uniform(n, seed), "octree", 16, name=f"cfg1_uniform_n{n}")
    return with_lists(p, theta, 0.02 * n ** (-1.0 / 3.0))


def config2(n: int = 1 << 20, seed: int = 2, theta: float = 0.7, tree: str = "binary") -> Problem:
    """Plummer mix (configs[1]); eps = 1/(50 n^1/3)."""
    p = build_tree(particles_plummer_mix(n, seed), tree, 16, name=f"cfg2_plummer_n{n}")
    return with_lists(p, theta, 1.0 / (50.0 * n ** (1.0 / 3.0)))


def config3(ng: int = 256, seed: int = 3, theta: float = 0.7, tree: str = "binary") -> Problem:
    """Zel'dovich-displaced ng^3 lattice, P(k)~k^-2, rms 0.3 cells (configs[2], the headline at ng=256)."""
    p = build_tree(particles_zeldovich(ng, seed, -2.0, 0.3), tree, 16, name=f"cfg3_zeldovich_{ng}^3")
    return with_lists(p, theta, 1.0 / (50.0 * ng))


def config5_particles(n: int = 1 << 26, seed: int = 5, mesh: int = 512) -> tuple[np.ndarray, float]:
    """configs[4]: first n sites of the smallest lattice with >= n sites; P(k)~k^-2.5, rms 0.5 cells."""
    ng = int(np.ceil(n ** (1.0 / 3.0) - 1e-9))
    while ng ** 3 < n:
        ng += 1
    m = mesh if mesh < ng or (ng & (ng - 1)) else None
    xyzm = particles_zeldovich(ng, seed, -2.5, 0.5, n_keep=n, mesh=m)
    return xyzm, f32(1.0 / (50.0 * n ** (1.0 / 3.0)))


def config4(n_buckets: int, l_pp: int, l_pc: int, seed: int = 4, reuse: int = 16, r_b: float = 0.005,
            cloud: int = 64) -> Problem:
    """Kernel shape sweep (configs[3]): buckets of 16 targets in a ball of radius r_b; `reuse`
    co-centred buckets share one source pool: l_pp particles uniform by volume in the shell
    2..10 r_b and l_pc cells whose centres lie in the same shell and whose moments come from
    `cloud` equal-mass points in a ball of radius 0.5 r_b.  eps = 0.02 r_b."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000 * l_pp + l_pc))
    ncl = (n_buckets + reuse - 1) // reuse
    centres = rng.random((ncl, 3))

    def ball(m, rmin, rmax):
        u = rng.random(m)
        r = (rmin ** 3 + u * (rmax ** 3 - rmin ** 3)) ** (1.0 / 3.0)
        mu = rng.uniform(-1, 1, m); ph = rng.uniform(0, 2 * np.pi, m); st = np.sqrt(1 - mu * mu)
        return np.stack([r * st * np.cos(ph), r * st * np.sin(ph), r * mu], axis=1)

    nt = n_buckets * 16
    tgt = np.repeat(centres, reuse * 16, axis=0)[:nt] + ball(nt, 0.0, r_b)
    src = np.repeat(centres, l_pp, axis=0) + ball(ncl * l_pp, 2 * r_b, 10 * r_b)
    n = nt + ncl * l_pp
    xyzm = np.empty((n, 4), np.float32)
    xyzm[:nt, :3] = tgt; xyzm[nt:, :3] = src
    xyzm[:, 3] = np.float32(1.0 / max(n, 1))
    first = (np.arange(n_buckets, dtype=np.int64) * 16).astype(np.int32)
    count = np.full(n_buckets, 16, np.int32)
    cl = np.arange(n_buckets, dtype=np.int64) // reuse
    pp_off = np.arange(n_buckets + 1, dtype=np.int64) * l_pp
    pp_idx = (nt + cl[:, None] * l_pp + np.arange(l_pp, dtype=np.int64)[None, :]).astype(np.int32).reshape(-1)
    ncell = ncl * l_pc
    if ncell:
        com = np.repeat(centres, l_pc, axis=0) + ball(ncell, 2 * r_b, 10 * r_b)
        pts = np.empty((ncell * cloud, 4), np.float32)
        pts[:, :3] = np.repeat(com, cloud, axis=0) + ball(ncell * cloud, 0.0, 0.5 * r_b)
        pts[:, 3] = np.float32(1.0 / max(n, 1))
        cells = cloud_records(pts, cloud)
    else:
        cells = np.zeros((0, REC), np.float32)
    pc_off = np.arange(n_buckets + 1, dtype=np.int64) * l_pc
    pc_idx = (cl[:, None] * l_pc + np.arange(l_pc, dtype=np.int64)[None, :]).astype(np.int32).reshape(-1)
    return Problem(name=f"cfg4_sweep_b{n_buckets}_pp{l_pp}_pc{l_pc}", xyzm=xyzm, cells=cells, first=first,
                   count=count, pp_off=pp_off, pp_idx=pp_idx, pc_off=pc_off, pc_idx=pc_idx,
                   eps=f32(0.02 * r_b))
