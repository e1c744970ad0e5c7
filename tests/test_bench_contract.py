"""-m "not gpu": bench.py's contract that can be checked without a GPU -- the reference arm prints the
required JSON line (the oracle on host cores), and the product arm refuses to run without a CUDA device
instead of falling back to anything."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env_extra=None, timeout=300):
    env = dict(os.environ)
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True,
                          timeout=timeout, env=env, cwd=ROOT)


def test_reference_arm_prints_the_contract_line():
    r = _run(["--impl", "reference", "--ng", "16", "--steps", "2", "--warmup", "1"], {"OMP_NUM_THREADS": "2"})
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert k in d, k
    assert d["impl"] == "reference" and d["dtype"] == "f64" and d["vs_baseline"] is None and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert "workload" in d["config"] and d["config"]["parallelism"] == "1 GPU"   # the same key set as the product arm's config


def test_reference_arm_other_ranks_exit_quietly():
    r = _run(["--impl", "reference", "--ng", "16", "--steps", "1", "--warmup", "0", "--gpus", "2"],
             {"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"})
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_product_arm_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        import pytest
        pytest.skip("a CUDA device is present")
    r = _run(["--ng", "16", "--steps", "1", "--warmup", "0"])
    assert r.returncode != 0
    assert "no CUDA device" in (r.stderr + r.stdout)


import pytest


@pytest.mark.gpu
def test_product_arm_line_on_gpu():
    """The product arm at a small lattice (same code path as the headline run): one JSON line with the
    keys the measurement contract asks for, a roofline fraction in (0, 1.05) and a counted launch number."""
    r = _run(["--ng", "64", "--steps", "3", "--warmup", "3", "--cpu-seconds", "1", "--configs-cpu-seconds", "1"], timeout=900)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["dtype"] == "f32" and d["data"] == "synthetic" and d["scaling"] == "strong" and d["vs_baseline"] is None
    assert d["gpu_launches"] == 4 and d["warmup"] >= 3   # cell prep, packer, evaluation, fp64 fix-up
    rf = d["roofline"]
    assert rf["bound"] == "alu" and rf["unit"] == "TFLOP/s" and 0.0 < rf["frac"] < 1.05
    assert abs(rf["frac"] - rf["achieved"] / rf["peak"]) < 1e-12
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] == 16 * d["config"]["n_particles"]
    assert d["e2e"]["value"] < d["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["pp_leaves"]["e2e"]["h2d_bytes_per_step"] < d["e2e"]["h2d_bytes_per_step"]
    assert d["config"]["parallelism"] == "1 GPU" and "sm_mhz" in d["clocks_extra_keys"]
    # the other configs, measured in the same run: each with its own clock record, a roofline fraction and parity
    assert len(d["configs"]) == 4
    for c in d["configs"]:
        assert "sm_mhz" in c["clocks"] and 0.0 < c["frac_fp32_fma_peak"] < 1.05 and c["kernel_ms_median"] > 0
        assert c["max_rel_err_acc"] <= 2e-5 and c["max_rel_err_pot"] <= 2e-5, c
