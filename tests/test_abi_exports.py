"""-m "not gpu": the C-ABI library loads without a GPU and exports every symbol include/pkdg.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_1609_08621_b200 import build
    lib = ctypes.CDLL(build.build())
    hdr = open(os.path.join(ROOT, "include", "pkdg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pkdg_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), name
    from paper_1609_08621_b200 import binding
    assert set(binding.EXPORTS) == declared
    assert binding.version() == (0, 1)


def test_host_only_entry_points_work_without_gpu():
    import numpy as np
    import oracle
    from paper_1609_08621_b200 import binding
    rng = np.random.default_rng(0)
    pp = np.concatenate([[0], np.cumsum(rng.integers(0, 400, 300))]).astype(np.int64)
    pc = np.concatenate([[0], np.cumsum(rng.integers(0, 200, 300))]).astype(np.int64)
    for cap in (1, 50, 1000, 10 ** 9):
        assert np.array_equal(binding.chunk_bounds(pp, pc, cap), oracle.chunk_bounds(pp, pc, cap))
    assert binding.status_string(0) == "PKDG_OK" and "EINVAL" in binding.status_string(-1)
