"""Thin ctypes binding over the C ABI of include/pkdg.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libpkdg.so; there is no Python or CPU
fallback: importing this module raises if the library has not been built
(``python -m paper_1609_08621_b200.build``) and every call raises ``PkdgError`` on a non-zero
status.  Device buffers are torch CUDA tensors (torch is used for memory and streams only),
host buffers are numpy arrays or pinned CPU tensors.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_float, c_int, c_int32, c_int64, c_uint32, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpkdg.so")

ACCUMULATE = 0x1
SKIP_PP = 0x2
SKIP_PC = 0x4
PP_LEAVES = 0x8
NO_FIXUP = 0x10
FIXUP_ALL = 0x20
VALIDATE = 0x40
OPT_KAPPA2 = 1
CELL_FLOATS = 36
CELLQ_FLOATS = 32

STATIC_MAX_BUCKETS = 32768
STATIC_MAX_CELLS = 32768
STATIC_MAX_PARTICLES = 524288

EXPORTS = ["pkdg_create", "pkdg_destroy", "pkdg_gravity_eval", "pkdg_gravity_eval_static", "pkdg_gravity_eval_range", "pkdg_gravity_eval_streamed",
           "pkdg_gravity_eval_host", "pkdg_gravity_eval_host_range", "pkdg_gravity_eval_groups",
           "pkdg_gravity_eval_host_groups", "pkdg_gravity_eval_fmm", "pkdg_build_lists_count", "pkdg_build_lists_fill",
           "pkdg_gravity_eval_tree_host", "pkdg_pack_export", "pkdg_chunk_bounds", "pkdg_prepare_cells_export",
           "pkdg_get_stats", "pkdg_set_option", "pkdg_profile_enable", "pkdg_profile_read", "pkdg_launch_count",
           "pkdg_status_string", "pkdg_last_error", "pkdg_version", "pkdg_fma_peak_probe"]


class PkdgError(RuntimeError):
    pass


class _Particles(Structure):
    _fields_ = [("xyzm", c_void_p), ("n", c_int64)]


class _Cells(Structure):
    _fields_ = [("rec", c_void_p), ("n", c_int64), ("stride_floats", c_int32)]


class _Buckets(Structure):
    _fields_ = [("first", c_void_p), ("count", c_void_p), ("n", c_int64)]


class _Groups(Structure):
    _fields_ = [("first_bucket", c_void_p), ("n_buckets", c_void_p), ("n", c_int64)]


class _Tree(Structure):
    _fields_ = [("first", c_void_p), ("count", c_void_p), ("end", c_void_p), ("isleaf", c_void_p), ("bblo", c_void_p),
                ("bbhi", c_void_p), ("leaf_rank", c_void_p), ("n_cells", c_int64)]


class _List(Structure):
    _fields_ = [("offsets", c_void_p), ("idx", c_void_p)]


class Stats(Structure):
    _fields_ = [("n_buckets", c_int64), ("interactions_pp", c_int64), ("interactions_pc", c_int64),
                ("tiles_pp", c_int64), ("tiles_pc", c_int64), ("bad_entries", c_int64), ("chunks", c_int64),
                ("fixup_sinks", c_int64), ("invalid_values", c_int64), ("invalid_pairs", c_int64),
                ("interactions_cc", c_int64), ("interactions_cp", c_int64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


def _load():
    if not os.path.exists(LIB_PATH):
        raise PkdgError(f"{LIB_PATH} is missing: build it with `python -m paper_1609_08621_b200.build` "
                        "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    L.pkdg_create.argtypes = [POINTER(c_void_p), c_int]
    L.pkdg_destroy.argtypes = [c_void_p]
    L.pkdg_gravity_eval.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                    POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p, c_void_p]
    L.pkdg_gravity_eval_static.argtypes = [c_int, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                           POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p, c_void_p]
    L.pkdg_gravity_eval_range.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets), c_int64,
                                          c_int64, POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p,
                                          c_void_p]
    L.pkdg_gravity_eval_streamed.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                             POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p,
                                             c_int32, c_int64, c_void_p]
    L.pkdg_gravity_eval_host.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                         POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p, c_int32,
                                         c_int64]
    L.pkdg_gravity_eval_host_range.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                               c_int64, c_int64, POINTER(_List), POINTER(_List), c_float, c_uint32,
                                               c_void_p, c_int32, c_int64]
    L.pkdg_gravity_eval_groups.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                           POINTER(_Groups), POINTER(_List), POINTER(_List), c_float, c_uint32, c_void_p,
                                           c_void_p]
    L.pkdg_gravity_eval_host_groups.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets),
                                                POINTER(_Groups), POINTER(_List), POINTER(_List), c_float, c_uint32,
                                                c_void_p, c_int32, c_int64]
    L.pkdg_gravity_eval_fmm.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Buckets), c_void_p,
                                        POINTER(_List), POINTER(_List), POINTER(_List), POINTER(_List), c_float, c_uint32,
                                        c_void_p, c_void_p]
    L.pkdg_build_lists_count.argtypes = [c_void_p, POINTER(_Tree), POINTER(_Cells), c_void_p, c_int64, c_double, c_double,
                                         c_uint32, c_void_p, c_void_p, c_void_p, c_void_p]
    L.pkdg_build_lists_fill.argtypes = [c_void_p, POINTER(_Tree), POINTER(_Cells), c_void_p, c_int64, c_double, c_double,
                                        c_uint32, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]
    L.pkdg_gravity_eval_tree_host.argtypes = [c_void_p, POINTER(_Particles), POINTER(_Cells), POINTER(_Tree),
                                              POINTER(_Buckets), c_void_p, c_double, c_float, c_uint32, c_void_p, c_int32]
    L.pkdg_pack_export.argtypes = [c_void_p, c_int64, POINTER(_List), c_void_p, c_void_p, c_int64, c_void_p]
    L.pkdg_chunk_bounds.argtypes = [c_int64, c_void_p, c_void_p, c_int64, c_void_p, POINTER(c_int64)]
    L.pkdg_prepare_cells_export.argtypes = [c_void_p, POINTER(_Cells), c_void_p, c_void_p]
    L.pkdg_get_stats.argtypes = [c_void_p, POINTER(Stats)]
    L.pkdg_profile_enable.argtypes = [c_void_p, c_int32]
    L.pkdg_profile_read.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_double), POINTER(c_double)]
    L.pkdg_launch_count.argtypes = [c_void_p]
    L.pkdg_launch_count.restype = c_int64
    L.pkdg_status_string.argtypes = [c_int32]
    L.pkdg_status_string.restype = c_char_p
    L.pkdg_last_error.argtypes = [c_void_p]
    L.pkdg_last_error.restype = c_char_p
    L.pkdg_version.argtypes = [POINTER(c_int32), POINTER(c_int32)]
    L.pkdg_fma_peak_probe.argtypes = [c_void_p, c_int64, POINTER(c_float), POINTER(c_double)]
    L.pkdg_set_option.argtypes = [c_void_p, c_int32, c_double]
    for name in EXPORTS:
        if name not in ("pkdg_launch_count", "pkdg_status_string", "pkdg_last_error", "pkdg_version"):
            getattr(L, name).restype = c_int32
    return L


_lib = _load()


def lib():
    return _lib


def version():
    a, b = c_int32(), c_int32()
    _lib.pkdg_version(byref(a), byref(b))
    return a.value, b.value


def status_string(s: int) -> str:
    return _lib.pkdg_status_string(int(s)).decode()


def _ptr(a):
    """Address of a torch tensor (any device) or a numpy array; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise PkdgError("numpy buffers must be C-contiguous")
        return a.ctypes.data
    if not a.is_contiguous():
        raise PkdgError("tensors must be contiguous")
    return a.data_ptr()


def _dt(a, want, name):
    if a is None:
        return
    got = str(a.dtype).replace("torch.", "")
    if got != want:
        raise PkdgError(f"{name}: dtype {got}, expected {want}")


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def chunk_bounds(pp_off, pc_off, max_entries: int) -> np.ndarray:
    """Chunk boundaries of the streamed variants from HOST offsets (pkdg_chunk_bounds)."""
    ref = pp_off if pp_off is not None else pc_off
    nb = int(ref.shape[0]) - 1
    bounds = np.zeros(nb + 2, np.int64)
    n = c_int64()
    s = _lib.pkdg_chunk_bounds(nb, _ptr(pp_off), _ptr(pc_off), int(max_entries), bounds.ctypes.data, byref(n))
    if s != 0:
        raise PkdgError(status_string(s))
    return bounds[: n.value + 1].copy()


def gravity_eval_static(device, xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps, out, flags=0,
                        stream=None):
    """pkdg_gravity_eval_static: pkdg_gravity_eval without a context and without any device allocation, for
    hosts that own all device memory themselves or must not call the CUDA allocator where they call us.  The
    workspace is a fixed array inside the library (about 6 MB per GPU, shared by every call on that GPU), so
    the problem is limited to STATIC_MAX_BUCKETS / STATIC_MAX_CELLS / STATIC_MAX_PARTICLES and calls whose GPU
    work could overlap must be ordered by the caller.  Asynchronous on `stream`; raises PkdgError (with the
    limit in the text) for anything larger.  Marshalling only, like every function here."""
    P, C, B, pp, pc = Context._structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx)
    _dt(out, "float32", "out")
    s = _lib.pkdg_gravity_eval_static(int(device), byref(P), byref(C) if C else None, byref(B),
                                      byref(pp) if pp else None, byref(pc) if pc else None, float(eps), int(flags),
                                      _ptr(out), _stream_ptr(stream))
    if s != 0:
        raise PkdgError(f"{status_string(s)}: {_lib.pkdg_last_error(None).decode()}")
    return out


class Context:
    """A pkdg_ctx: owns internal workspace only (pkdg_create / pkdg_destroy)."""

    def __init__(self, device: int = 0):
        self._h = c_void_p()
        s = _lib.pkdg_create(byref(self._h), int(device))
        if s != 0:
            self._h = c_void_p()
            raise PkdgError(f"pkdg_create: {status_string(s)}: {_lib.pkdg_last_error(None).decode()}")
        self.device = device

    def close(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.pkdg_destroy(self._h)
            self._h = c_void_p()

    __del__ = close

    def _check(self, s, what):
        if s != 0:
            raise PkdgError(f"{what}: {status_string(s)}: {_lib.pkdg_last_error(self._h).decode()}")

    @staticmethod
    def _structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx):
        _dt(xyzm, "float32", "xyzm"); _dt(cells, "float32", "cells"); _dt(first, "int32", "first")
        _dt(count, "int32", "count"); _dt(pp_off, "int64", "pp_off"); _dt(pp_idx, "int32", "pp_idx")
        _dt(pc_off, "int64", "pc_off"); _dt(pc_idx, "int32", "pc_idx")
        P = _Particles(_ptr(xyzm), int(xyzm.shape[0]))
        C = None
        if cells is not None:
            C = _Cells(_ptr(cells), int(cells.shape[0]), int(cells.shape[1]) if cells.ndim == 2 else CELL_FLOATS)
        B = _Buckets(_ptr(first), _ptr(count), int(first.shape[0]))
        pp = _List(_ptr(pp_off), _ptr(pp_idx)) if pp_off is not None else None
        pc = _List(_ptr(pc_off), _ptr(pc_idx)) if pc_off is not None else None
        return P, C, B, pp, pc

    def gravity_eval(self, xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx, eps, out, flags=0,
                     stream=None):
        """pkdg_gravity_eval: everything resident on the device; asynchronous on `stream`."""
        P, C, B, pp, pc = self._structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx)
        _dt(out, "float32", "out")
        s = _lib.pkdg_gravity_eval(self._h, byref(P), byref(C) if C else None, byref(B), byref(pp) if pp else None,
                                   byref(pc) if pc else None, float(eps), int(flags), _ptr(out), _stream_ptr(stream))
        self._check(s, "pkdg_gravity_eval")
        return out

    def gravity_eval_range(self, xyzm, cells, first, count, b0, b1, pp_off, pp_idx, pc_off, pc_idx, eps, out, flags=0,
                           stream=None):
        """pkdg_gravity_eval_range: buckets [b0, b1) of the full (first, count) arrays; the lists are those of the
        range only (b1 - b0 + 1 offsets).  Asynchronous on `stream`."""
        P, C, B, pp, pc = self._structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx)
        _dt(out, "float32", "out")
        s = _lib.pkdg_gravity_eval_range(self._h, byref(P), byref(C) if C else None, byref(B), int(b0), int(b1),
                                         byref(pp) if pp else None, byref(pc) if pc else None, float(eps), int(flags),
                                         _ptr(out), _stream_ptr(stream))
        self._check(s, "pkdg_gravity_eval_range")
        return out

    def gravity_eval_streamed(self, xyzm, cells, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h, eps, out,
                              n_streams=3, max_entries_per_chunk=1 << 24, flags=0, stream=None):
        """pkdg_gravity_eval_streamed: device particles/cells/out, HOST buckets and lists."""
        P, C, B, pp, pc = self._structs(xyzm, cells, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h)
        s = _lib.pkdg_gravity_eval_streamed(self._h, byref(P), byref(C) if C else None, byref(B),
                                            byref(pp) if pp else None, byref(pc) if pc else None, float(eps),
                                            int(flags), _ptr(out), int(n_streams), int(max_entries_per_chunk),
                                            _stream_ptr(stream))
        self._check(s, "pkdg_gravity_eval_streamed")
        return out

    def gravity_eval_host(self, xyzm_h, cells_h, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h, eps,
                          out_h, n_streams=3, max_entries_per_chunk=1 << 24, flags=0):
        """pkdg_gravity_eval_host: every buffer on the host; synchronous."""
        P, C, B, pp, pc = self._structs(xyzm_h, cells_h, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h)
        s = _lib.pkdg_gravity_eval_host(self._h, byref(P), byref(C) if C else None, byref(B),
                                        byref(pp) if pp else None, byref(pc) if pc else None, float(eps), int(flags),
                                        _ptr(out_h), int(n_streams), int(max_entries_per_chunk))
        self._check(s, "pkdg_gravity_eval_host")
        return out_h

    def gravity_eval_host_range(self, xyzm_h, cells_h, first_h, count_h, b0, b1, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h,
                                eps, out_h, n_streams=3, max_entries_per_chunk=1 << 24, flags=0):
        """pkdg_gravity_eval_host_range: buckets [b0, b1) of the full host bucket arrays, lists of the range only."""
        P, C, B, pp, pc = self._structs(xyzm_h, cells_h, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h)
        s = _lib.pkdg_gravity_eval_host_range(self._h, byref(P), byref(C) if C else None, byref(B), int(b0), int(b1),
                                              byref(pp) if pp else None, byref(pc) if pc else None, float(eps),
                                              int(flags), _ptr(out_h), int(n_streams), int(max_entries_per_chunk))
        self._check(s, "pkdg_gravity_eval_host_range")
        return out_h

    def gravity_eval_groups(self, xyzm, cells, first, count, g_first, g_n, pp_off, pp_idx, pc_off, pc_idx, eps, out,
                            flags=0, stream=None):
        """pkdg_gravity_eval_groups: one P-P and one P-C list per GROUP of consecutive buckets (offsets have
        n_groups + 1 entries); everything resident; asynchronous on `stream`."""
        P, C, B, pp, pc = self._structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx)
        _dt(g_first, "int32", "g_first"); _dt(g_n, "int32", "g_n"); _dt(out, "float32", "out")
        G = _Groups(_ptr(g_first), _ptr(g_n), int(g_first.shape[0]))
        s = _lib.pkdg_gravity_eval_groups(self._h, byref(P), byref(C) if C else None, byref(B), byref(G),
                                          byref(pp) if pp else None, byref(pc) if pc else None, float(eps), int(flags),
                                          _ptr(out), _stream_ptr(stream))
        self._check(s, "pkdg_gravity_eval_groups")
        return out

    def gravity_eval_host_groups(self, xyzm_h, cells_h, first_h, count_h, g_first_h, g_n_h, pp_off_h, pp_idx_h, pc_off_h,
                                 pc_idx_h, eps, out_h, n_streams=3, max_entries_per_chunk=1 << 24, flags=0):
        """pkdg_gravity_eval_host_groups: every buffer on the host, group-shared lists; synchronous."""
        P, C, B, pp, pc = self._structs(xyzm_h, cells_h, first_h, count_h, pp_off_h, pp_idx_h, pc_off_h, pc_idx_h)
        _dt(g_first_h, "int32", "g_first"); _dt(g_n_h, "int32", "g_n")
        G = _Groups(_ptr(g_first_h), _ptr(g_n_h), int(g_first_h.shape[0]))
        s = _lib.pkdg_gravity_eval_host_groups(self._h, byref(P), byref(C) if C else None, byref(B), byref(G),
                                               byref(pp) if pp else None, byref(pc) if pc else None, float(eps),
                                               int(flags), _ptr(out_h), int(n_streams), int(max_entries_per_chunk))
        self._check(s, "pkdg_gravity_eval_host_groups")
        return out_h

    def gravity_eval_fmm(self, xyzm, cells, first, count, centres, pp_off, pp_idx, pc_off, pc_idx, cp_off, cp_idx,
                         cc_off, cc_idx, eps, out, flags=0, stream=None):
        """pkdg_gravity_eval_fmm: four lists per bucket (P-P, P-C per sink; C-P, C-C through the bucket's local
        expansion about centres[b]); everything resident; asynchronous on `stream`."""
        P, C, B, pp, pc = self._structs(xyzm, cells, first, count, pp_off, pp_idx, pc_off, pc_idx)
        _dt(centres, "float32", "centres"); _dt(cp_off, "int64", "cp_off"); _dt(cp_idx, "int32", "cp_idx")
        _dt(cc_off, "int64", "cc_off"); _dt(cc_idx, "int32", "cc_idx"); _dt(out, "float32", "out")
        cp = _List(_ptr(cp_off), _ptr(cp_idx)) if cp_off is not None else None
        cc = _List(_ptr(cc_off), _ptr(cc_idx)) if cc_off is not None else None
        s = _lib.pkdg_gravity_eval_fmm(self._h, byref(P), byref(C) if C else None, byref(B), _ptr(centres),
                                       byref(pp) if pp else None, byref(pc) if pc else None, byref(cp) if cp else None,
                                       byref(cc) if cc else None, float(eps), int(flags), _ptr(out), _stream_ptr(stream))
        self._check(s, "pkdg_gravity_eval_fmm")
        return out

    @staticmethod
    def _tree(tree, cells):
        """tree: dict of device tensors first, count, end, isleaf (int32), bblo, bbhi (float32 [n,3]) and
        optionally leaf_rank (int32)."""
        for k in ("first", "count", "end", "isleaf"):
            _dt(tree[k], "int32", k)
        _dt(tree["bblo"], "float32", "bblo"); _dt(tree["bbhi"], "float32", "bbhi"); _dt(cells, "float32", "cells")
        T = _Tree(_ptr(tree["first"]), _ptr(tree["count"]), _ptr(tree["end"]), _ptr(tree["isleaf"]), _ptr(tree["bblo"]),
                  _ptr(tree["bbhi"]), _ptr(tree.get("leaf_rank")), int(tree["first"].shape[0]))
        C = _Cells(_ptr(cells), int(cells.shape[0]), int(cells.shape[1]))
        return T, C

    def build_lists_count(self, tree, cells, sink_cell, theta, eps, pp_off, pc_off, flags=0, stream=None, sync=True):
        """pkdg_build_lists_count: CSR offsets (device int64 [n_sinks + 1] each); returns (n_pp, n_pc) if sync."""
        T, C = self._tree(tree, cells)
        _dt(sink_cell, "int32", "sink_cell"); _dt(pp_off, "int64", "pp_off"); _dt(pc_off, "int64", "pc_off")
        tot = (c_int64 * 2)()
        s = _lib.pkdg_build_lists_count(self._h, byref(T), byref(C), _ptr(sink_cell), int(sink_cell.shape[0]),
                                        float(theta), float(eps), int(flags), _ptr(pp_off), _ptr(pc_off),
                                        ctypes.cast(tot, c_void_p) if sync else None, _stream_ptr(stream))
        self._check(s, "pkdg_build_lists_count")
        return (int(tot[0]), int(tot[1])) if sync else None

    def build_lists_fill(self, tree, cells, sink_cell, theta, eps, pp_off, pc_off, pp_idx, pc_idx, flags=0, stream=None):
        """pkdg_build_lists_fill: the entries, in walk order, at the offsets build_lists_count wrote."""
        T, C = self._tree(tree, cells)
        _dt(pp_idx, "int32", "pp_idx"); _dt(pc_idx, "int32", "pc_idx")
        s = _lib.pkdg_build_lists_fill(self._h, byref(T), byref(C), _ptr(sink_cell), int(sink_cell.shape[0]),
                                       float(theta), float(eps), int(flags), _ptr(pp_off), _ptr(pc_off), _ptr(pp_idx),
                                       _ptr(pc_idx), _stream_ptr(stream))
        self._check(s, "pkdg_build_lists_fill")

    def gravity_eval_tree_host(self, xyzm_h, cells_h, tree_h, first_h, count_h, bucket_cell_h, theta, eps, out_h, flags=0,
                               n_ranges=4):
        """pkdg_gravity_eval_tree_host: every buffer on the host (numpy or CPU tensors, pinned for full speed); the
        lists are built on the device.  tree_h: dict of first, count, end, isleaf (int32), bblo, bbhi (float32 [n,3])."""
        T, C = self._tree(tree_h, cells_h)
        _dt(xyzm_h, "float32", "xyzm"); _dt(first_h, "int32", "first"); _dt(count_h, "int32", "count")
        _dt(bucket_cell_h, "int32", "bucket_cell"); _dt(out_h, "float32", "out")
        P = _Particles(_ptr(xyzm_h), int(xyzm_h.shape[0]))
        B = _Buckets(_ptr(first_h), _ptr(count_h), int(first_h.shape[0]))
        s = _lib.pkdg_gravity_eval_tree_host(self._h, byref(P), byref(C), byref(T), byref(B), _ptr(bucket_cell_h),
                                             float(theta), float(eps), int(flags), _ptr(out_h), int(n_ranges))
        self._check(s, "pkdg_gravity_eval_tree_host")
        return out_h

    def pack_export(self, n_buckets, off, idx, tile_offsets, tiles, stream=None):
        """pkdg_pack_export: tile_offsets[n_buckets+1] int64 and tiles[cap,32] int32 (device)."""
        L = _List(_ptr(off), _ptr(idx))
        cap = 0 if tiles is None else int(tiles.shape[0])
        s = _lib.pkdg_pack_export(self._h, int(n_buckets), byref(L), _ptr(tile_offsets), _ptr(tiles), cap,
                                  _stream_ptr(stream))
        self._check(s, "pkdg_pack_export")

    def prepare_cells_export(self, cells, out, stream=None):
        C = _Cells(_ptr(cells), int(cells.shape[0]), int(cells.shape[1]))
        s = _lib.pkdg_prepare_cells_export(self._h, byref(C), _ptr(out), _stream_ptr(stream))
        self._check(s, "pkdg_prepare_cells_export")
        return out

    def get_stats(self, check: bool = True) -> dict:
        st = Stats()
        s = _lib.pkdg_get_stats(self._h, byref(st))
        if check:
            self._check(s, "pkdg_get_stats")
        return st.as_dict()

    def profile_enable(self, on: bool = True):
        self._check(_lib.pkdg_profile_enable(self._h, 1 if on else 0), "pkdg_profile_enable")

    def profile_read(self):
        """(n_calls, eval_kernel_ms_total, fixup_kernel_ms_total) since the last read (synchronises)."""
        n, ms, fx = c_int64(), c_double(), c_double()
        self._check(_lib.pkdg_profile_read(self._h, byref(n), byref(ms), byref(fx)), "pkdg_profile_read")
        return n.value, ms.value, fx.value

    def launch_count(self) -> int:
        return int(_lib.pkdg_launch_count(self._h))

    def set_option(self, option: int, value: float):
        self._check(_lib.pkdg_set_option(self._h, int(option), float(value)), "pkdg_set_option")

    def fma_peak_probe(self, iters: int = 1 << 14):
        ms, fl = c_float(), c_double()
        self._check(_lib.pkdg_fma_peak_probe(self._h, int(iters), byref(ms), byref(fl)), "pkdg_fma_peak_probe")
        return ms.value, fl.value
