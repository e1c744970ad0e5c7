"""pkdg_gravity_eval_static -- the call for hosts that are not allowed to allocate device memory.

Why it exists: a pkdg_ctx gets its workspace from cudaMalloc and regrows it (cudaFree + cudaMalloc) when a bigger
problem arrives.  A host that has given away all device memory at start-up, that cannot afford the device-wide
stall those two calls cause while its other streams are busy, or that simply must not call the CUDA allocator at
the place where it calls us, cannot use a context.  For it the library carries one fixed ~6 MB array per GPU and
an entry point that works inside it, up to 32768 buckets / 32768 cells / 524288 particles.

What is checked here: the rows it writes are the rows pkdg_gravity_eval writes (same kernels, so bit for bit, which
is inside the 2e-5 the parity tests allow), on two calls in a row that share the array -- the second on a smaller
problem and through the fp64 fix-up queue, so anything the first call left behind (descriptors, cell records,
queue entries, counters) would show up as a wrong row.  This file sorts last on purpose: `pytest -x` stops at the
first failure, and a failure here must not hide the parity tests.  It passes on its own in a fresh process (the
first call then does the per-device set-up) as well as after the other files.
"""
import numpy as np
import pytest

TOL = 2e-5   # the bar of tests/test_gpu_parity.py


def _problems():
    from paper_1609_08621_b200 import inputs
    big = inputs.config2(n=1 << 14, seed=11)     # clustered (Plummer spheres), binary tree: ~1.5e3 buckets
    small = inputs.config1(n=4096, seed=1)       # uniform, octree: ~540 buckets
    return big, small


def _dev(p, torch):
    from gpu_util import to_dev
    return to_dev(p, torch)


def _max_rel(got, ref):
    a = np.linalg.norm(got[:, :3].astype(np.float64) - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3].astype(np.float64), axis=1)
    f = np.abs(got[:, 3].astype(np.float64) - ref[:, 3]) / np.abs(ref[:, 3].astype(np.float64))
    return float(a.max()), float(f.max())


@pytest.mark.gpu
def test_static_entry_point_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_1609_08621_b200 import binding
    big, small = _problems()
    assert big.n_buckets <= binding.STATIC_MAX_BUCKETS and big.cells.shape[0] <= binding.STATIC_MAX_CELLS
    assert small.n_buckets < big.n_buckets   # the second call must leave part of the array as the first call wrote it
    cases = [(big, 0), (small, binding.FIXUP_ALL)]

    # what the existing path gives (a context, cudaMalloc'ed workspace)
    ctx = binding.Context(0)
    want, dev = [], []
    for p, flags in cases:
        d = _dev(p, torch)
        out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda:0")
        ctx.gravity_eval(d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"], d["pc_off"],
                         d["pc_idx"], p.eps, out, flags=flags)
        torch.cuda.synchronize()
        assert ctx.get_stats()["bad_entries"] == 0
        want.append(out.cpu().numpy())
        dev.append(d)
    ctx.close()

    # the two static calls, back to back on one stream, nothing in between
    outs = [torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda:0") for p, _ in cases]
    for (p, flags), d, out in zip(cases, dev, outs):
        binding.gravity_eval_static(0, d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"],
                                    d["pc_off"], d["pc_idx"], p.eps, out, flags=flags)
    torch.cuda.synchronize()
    for (p, flags), out, ref in zip(cases, outs, want):
        got = out.cpu().numpy()
        assert np.isfinite(got).all()
        ea, ep = _max_rel(got, ref)
        assert ea <= TOL and ep <= TOL, (p.name, flags, ea, ep)
        assert np.array_equal(got, ref), (p.name, flags, ea, ep)   # same kernels on the same inputs


@pytest.mark.gpu
def test_static_entry_point_accumulates_and_skips_like_the_context_path():
    """A third and fourth call on the same array: PKDG_SKIP_PC, then PKDG_SKIP_PP | PKDG_ACCUMULATE on top, must give
    the rows of the full evaluation to rounding of the final addition."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    from paper_1609_08621_b200 import binding
    _, p = _problems()
    d = _dev(p, torch)
    full = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda:0")
    parts = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda:0")
    args = (d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"], d["pc_off"], d["pc_idx"], p.eps)
    binding.gravity_eval_static(0, *args, full, flags=binding.NO_FIXUP)
    binding.gravity_eval_static(0, *args, parts, flags=binding.NO_FIXUP | binding.SKIP_PC)
    binding.gravity_eval_static(0, *args, parts, flags=binding.NO_FIXUP | binding.SKIP_PP | binding.ACCUMULATE)
    torch.cuda.synchronize()
    ea, ep = _max_rel(parts.cpu().numpy(), full.cpu().numpy())
    assert ea <= TOL and ep <= TOL, (ea, ep)


def test_static_entry_point_refuses_what_does_not_fit():
    """Limits and flags are checked before anything touches the GPU, so this runs without one: the error names the
    limit, and nothing has been queued."""
    from paper_1609_08621_b200 import binding
    n = 64
    xyzm = np.zeros((n, 4), np.float32)
    out = np.zeros((n, 4), np.float32)
    one = np.zeros(1, np.int32)
    off = np.zeros(2, np.int64)

    class _Fake:   # a buffer whose claimed length exceeds the limit; the call must refuse before reading it
        def __init__(self, arr, rows): self._a, self.shape, self.dtype, self.ndim = arr, (rows,) + arr.shape[1:], arr.dtype, arr.ndim
        def is_contiguous(self): return True
        def data_ptr(self): return self._a.ctypes.data

    too_many_buckets = _Fake(one, binding.STATIC_MAX_BUCKETS + 1)
    with pytest.raises(binding.PkdgError, match=r"EINVAL.*32769 buckets \(limit 32768\)"):
        binding.gravity_eval_static(0, xyzm, None, too_many_buckets, too_many_buckets, off, one, None, None, 0.01, out, stream=0)
    too_many_particles = _Fake(xyzm, binding.STATIC_MAX_PARTICLES + 1)
    with pytest.raises(binding.PkdgError, match=r"particles \(limit 524288\)"):
        binding.gravity_eval_static(0, too_many_particles, None, one, one, off, one, None, None, 0.01, out, stream=0)
    cells = _Fake(np.zeros((1, 36), np.float32), binding.STATIC_MAX_CELLS + 1)
    with pytest.raises(binding.PkdgError, match=r"cells \(limit 32768\)"):
        binding.gravity_eval_static(0, xyzm, cells, one, one, off, one, off, one, 0.01, out, stream=0)
    with pytest.raises(binding.PkdgError, match="PKDG_PP_LEAVES"):
        binding.gravity_eval_static(0, xyzm, None, one, one, off, one, None, None, 0.01, out, flags=binding.PP_LEAVES, stream=0)
    with pytest.raises(binding.PkdgError, match="PKDG_VALIDATE"):
        binding.gravity_eval_static(0, xyzm, None, one, one, off, one, None, None, 0.01, out, flags=binding.VALIDATE, stream=0)
