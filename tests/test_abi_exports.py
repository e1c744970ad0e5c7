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
    assert binding.version() == (0, 2)


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


def test_binding_fails_loudly_without_the_library(monkeypatch, tmp_path):
    """No CPU fallback: without libpkdg.so the binding refuses to load instead of degrading."""
    import pytest
    from paper_1609_08621_b200 import binding
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "libpkdg.so"))
    with pytest.raises(binding.PkdgError, match="no CPU fallback"):
        binding._load()


def test_product_package_does_not_import_the_oracle():
    """The product path (package + bench.py's own arm) never reaches into oracle/."""
    import ast
    pkg = os.path.join(ROOT, "paper_1609_08621_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if not f.endswith(".py"):
                continue
            tree = ast.parse(open(os.path.join(dirpath, f)).read())
            for node in ast.walk(tree):
                names = []
                if isinstance(node, ast.Import):
                    names = [a.name for a in node.names]
                elif isinstance(node, ast.ImportFrom):
                    names = [node.module or ""]
                assert not any(n == "oracle" or n.startswith("oracle.") for n in names), (f, names)
    for src in ("csrc/pkdg.cu", "csrc/pkdg_kernels.cuh"):
        text = open(os.path.join(pkg, src)).read()
        assert "oracle" not in text.lower().replace("the oracle", "")  # comments may mention it; no include
        assert "#include \"../../oracle" not in text and "pkdg_oracle" not in text


def test_generated_fmm_header_is_current():
    """pkdg_fmm_gen.cuh is what gen_fmm.py writes (the header is committed; the generator is its source)."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_1609_08621_b200", "csrc")
    spec = importlib.util.spec_from_file_location("gen_fmm", os.path.join(here, "gen_fmm.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    text = gen.emit()[0]
    with open(os.path.join(here, "pkdg_fmm_gen.cuh")) as f:
        assert f.read() == text


def test_create_failure_is_reported_through_the_abi():
    """Without a CUDA device pkdg_create fails and pkdg_last_error(NULL) says why (nothing is printed to stderr)."""
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1609_08621_b200 import binding
    with pytest.raises(binding.PkdgError) as e:
        binding.Context(0)
    assert "PKDG_ECUDA" in str(e.value) and "pkdg_create:" in str(e.value) and len(str(e.value)) > 40
