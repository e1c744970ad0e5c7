"""-m gpu parity tests of the FMM form of the path: C-C and C-P lists accumulated into
the 5th-order local expansion of every bucket and evaluated at its particles (pkdg_gravity_eval_fmm) against the
fp64 oracle (oracle.fmm_eval, pinned in tests/test_oracle_fmm_pins.py) on the same seeded inputs.  Bars as for the
rest of the path: list handling bit-exact, per-particle |a_gpu - a_or| / |a_or| <= 2e-5 and the same for the
potential, on the TOTAL of the four lists."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    return torch


@pytest.fixture(scope="module")
def ctx(torch):
    from paper_1609_08621_b200 import binding
    c = binding.Context(0)
    yield c
    c.close()


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _run(ctx, torch, p, F, near=True, far=True, flags=0, fill=float("nan")):
    t = lambda a: _dev(torch, a)
    out = torch.full((p.n, 4), fill, dtype=torch.float32, device="cuda:0")
    pp = F["pp"] if near else (None, None); pc = F["pc"] if near else (None, None)
    cp = F["cp"] if far else (None, None); cc = F["cc"] if far else (None, None)
    ctx.gravity_eval_fmm(t(p.xyzm), t(p.cells), t(p.first), t(p.count), t(F["centre"]), t(pp[0]), t(pp[1]), t(pc[0]),
                         t(pc[1]), t(cp[0]), t(cp[1]), t(cc[0]), t(cc[1]), F["eps"], out, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _oracle(p, F, near=True, far=True):
    import oracle
    out = np.zeros((p.n, 4))
    if near:
        out = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, F["pp"][0], F["pp"][1], F["pc"][0], F["pc"][1], F["eps"])
    if far:
        out = oracle.fmm_eval(p.xyzm, p.cells, p.first, p.count, F["centre"], F["cc"][0], F["cc"][1], F["cp"][0], F["cp"][1],
                              out=out)
    return out


def _assert_parity(out, ref_total, ref_part=None, label=""):
    """Errors of `out` against ref_part (default ref_total), relative to the TOTAL acceleration / potential."""
    ref_part = ref_total if ref_part is None else ref_part
    an = np.linalg.norm(ref_total[:, :3], axis=1)
    ea = np.linalg.norm(out[:, :3].astype(np.float64) - ref_part[:, :3], axis=1) / an
    ep = np.abs(out[:, 3].astype(np.float64) - ref_part[:, 3]) / np.abs(ref_total[:, 3])
    print(f"\n[{label}] acc max {ea.max():.2e} rms {np.sqrt(np.mean(ea ** 2)):.2e} | pot max {ep.max():.2e}")
    assert np.isfinite(out).all()
    assert ea.max() <= TOL and ep.max() <= TOL, (label, float(ea.max()), float(ep.max()))
    return ea, ep


@pytest.mark.parametrize("theta", [0.7, 0.5])
def test_config1_four_lists_every_particle(ctx, torch, theta):
    """configs[0] (N = 4096, octree) with the four-list walk: total, local-expansion part alone and near part alone."""
    from paper_1609_08621_b200 import inputs
    p = inputs.config1(4096, seed=1, theta=theta)
    F = inputs.build_fmm_lists(p, theta, p.eps)
    ref = _oracle(p, F)
    ref_far = _oracle(p, F, near=False)
    out = _run(ctx, torch, p, F)
    st = ctx.get_stats()
    _assert_parity(out, ref, label=f"cfg1 theta={theta} four lists")
    cnt = p.count.astype(np.int64)
    assert st["interactions_cc"] == len(F["cc"][1]) and st["interactions_cp"] == len(F["cp"][1])      # bit-exact integers
    assert st["interactions_pp"] == int(np.dot(cnt, np.diff(F["pp"][0])))
    assert st["interactions_pc"] == int(np.dot(cnt, np.diff(F["pc"][0])))
    assert st["bad_entries"] == 0 and st["n_buckets"] == p.n_buckets
    far = _run(ctx, torch, p, F, near=False)
    _assert_parity(far, ref, ref_far, label=f"cfg1 theta={theta} local expansion only")
    # the local-expansion part on its own terms as well (it is a smooth field: no cancellation to speak of)
    e_own = np.linalg.norm(far[:, :3] - ref_far[:, :3], axis=1) / np.linalg.norm(ref_far[:, :3], axis=1)
    assert e_own.max() <= TOL, e_own.max()
    near = _run(ctx, torch, p, F, far=False)
    _assert_parity(near, ref, ref - ref_far, label=f"cfg1 theta={theta} P-P + P-C only")
    # the sum of the two separate calls is the combined call up to fp32 rounding of the final addition
    assert np.allclose(near[:, :3] + far[:, :3], out[:, :3], rtol=0, atol=2e-6 * np.abs(out[:, :3]).max())


def test_clustered_binary_tree(ctx, torch):
    """configs[1] recipe at N = 2^16 (Plummer spheres + background, binary tree): sinks in dense cores, sources from
    1e-3 to 1 away -- the dynamic range the scaled form has to cover."""
    from paper_1609_08621_b200 import inputs
    p = inputs.config2(1 << 16, seed=2)
    F = inputs.build_fmm_lists(p, 0.7, p.eps)
    assert len(F["cc"][1]) > 0 and len(F["cp"][1]) > 0
    out = _run(ctx, torch, p, F)
    st = ctx.get_stats()
    assert st["interactions_cc"] == len(F["cc"][1]) and st["interactions_cp"] == len(F["cp"][1]) and st["bad_entries"] == 0
    _assert_parity(out, _oracle(p, F), label="plummer 2^16 four lists")


def _edge_fmm():
    """Hand-made buckets: counts 0, 1, 16, 17, 40 (> one warp of sinks), a bucket whose single particle sits AT its
    centre, empty C-C / C-P lists, lists longer than a few warps, padding entries, a monopole-only cell."""
    from paper_1609_08621_b200 import inputs
    rng = np.random.default_rng(11)
    counts = [0, 1, 16, 17, 40, 1, 5, 9]
    n_t = sum(counts)
    n_src = 600
    xyzm = np.empty((n_t + n_src, 4), np.float32)
    xyzm[:n_t, :3] = 0.5 + 0.004 * rng.standard_normal((n_t, 3))
    xyzm[n_t:, :3] = 0.5 + rng.choice([-1, 1], (n_src, 3)) * rng.uniform(0.08, 0.45, (n_src, 3))
    xyzm[:, 3] = rng.uniform(0.5, 1.5, n_t + n_src) / (n_t + n_src)
    first = np.concatenate([[0], np.cumsum(counts)[:-1]]).astype(np.int32)
    count = np.array(counts, np.int32)
    centre = np.zeros((len(counts), 3), np.float32)
    for b in range(len(counts)):
        if counts[b]:
            centre[b] = xyzm[first[b]:first[b] + counts[b], :3].astype(np.float64).mean(axis=0)
    centre[0] = 0.5
    centre[5] = xyzm[first[5], :3]                                       # the lone particle sits at the centre: s = 0
    ncell = 200
    com = 0.5 + rng.choice([-1, 1], (ncell, 3)) * rng.uniform(0.1, 0.45, (ncell, 3))
    pts = np.empty((ncell * 20, 4), np.float32)
    pts[:, :3] = np.repeat(com, 20, axis=0) + 0.015 * rng.standard_normal((ncell * 20, 3))
    pts[:, 3] = rng.uniform(0.5, 1.5, ncell * 20) / (ncell * 20)
    cells = inputs.cloud_records(pts, 20)
    cells[9, 4:35] = 0.0                                                # pure monopole cell
    cc_lens = [3, 200, 0, 33, 64, 7, 200, 1]
    cp_lens = [2, 0, 600, 31, 97, 5, 1, 0]
    cc = [rng.choice(ncell, L, replace=False).astype(np.int32) for L in cc_lens]
    cp = [(n_t + rng.choice(n_src, L, replace=False)).astype(np.int32) for L in cp_lens]
    cc[3][4] = -1; cp[4][10] = -1                                       # padding inside a list is ignored
    F = {"cc": (np.concatenate([[0], np.cumsum(cc_lens)]).astype(np.int64), np.concatenate(cc).astype(np.int32)),
         "cp": (np.concatenate([[0], np.cumsum(cp_lens)]).astype(np.int64), np.concatenate(cp).astype(np.int32)),
         "pp": (None, None), "pc": (None, None), "centre": centre, "eps": float(np.float32(0.001))}
    p = inputs.Problem(name="edge_fmm", xyzm=xyzm, cells=cells, first=first, count=count, pp_off=None, pp_idx=None,
                       pc_off=None, pc_idx=None, eps=F["eps"])
    return p, F


def test_edge_cases_and_accumulate(ctx, torch):
    from paper_1609_08621_b200 import binding
    p, F = _edge_fmm()
    ref = _oracle(p, F, near=False)
    out = _run(ctx, torch, p, F, near=False)
    st = ctx.get_stats()
    n_t = int(p.count.sum())
    _assert_parity(out[:n_t], ref[:n_t], label="edge buckets, local expansion only")
    assert np.isnan(out[n_t:]).all()                                    # particles in no bucket: untouched
    assert st["interactions_cc"] == len(F["cc"][1]) and st["interactions_cp"] == len(F["cp"][1]) and st["bad_entries"] == 0
    acc = _run(ctx, torch, p, F, near=False, flags=binding.ACCUMULATE, fill=1.0)
    assert np.allclose(acc[:n_t], out[:n_t] + 1.0, rtol=1e-6, atol=1e-6) and np.all(acc[n_t:] == 1.0)


def test_out_of_range_entries_are_counted_not_followed(ctx, torch):
    p, F = _edge_fmm()
    cc_idx = F["cc"][1].copy(); cp_idx = F["cp"][1].copy()
    cc_idx[5] = p.cells.shape[0] + 3; cc_idx[40] = 2 ** 31 - 1; cp_idx[7] = p.n + 100
    G = dict(F); G["cc"] = (F["cc"][0], cc_idx); G["cp"] = (F["cp"][0], cp_idx)
    out = _run(ctx, torch, p, G, near=False)
    st = ctx.get_stats(check=False)
    assert st["bad_entries"] == 3
    ok = dict(F); cc2 = cc_idx.copy(); cp2 = cp_idx.copy()
    cc2[[5, 40]] = -1; cp2[7] = -1                                       # the same lists with those entries as padding
    ok["cc"] = (F["cc"][0], cc2); ok["cp"] = (F["cp"][0], cp2)
    ref = _oracle(p, ok, near=False)
    n_t = int(p.count.sum())
    _assert_parity(out[:n_t], ref[:n_t], label="bad entries skipped")


def test_invalid_arguments_fail_loudly(ctx, torch):
    from paper_1609_08621_b200 import binding
    p, F = _edge_fmm()
    t = lambda a: _dev(torch, a)
    out = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda:0")
    with pytest.raises(binding.PkdgError):     # C-C list without cells
        ctx.gravity_eval_fmm(t(p.xyzm), None, t(p.first), t(p.count), t(F["centre"]), None, None, None, None, None, None,
                             t(F["cc"][0]), t(F["cc"][1]), F["eps"], out)
    with pytest.raises(binding.PkdgError):     # lists without centres
        ctx.gravity_eval_fmm(t(p.xyzm), t(p.cells), t(p.first), t(p.count), None, None, None, None, None, t(F["cp"][0]),
                             t(F["cp"][1]), None, None, F["eps"], out)
    with pytest.raises(binding.PkdgError):     # leaf-form P-P lists are not supported here
        ctx.gravity_eval_fmm(t(p.xyzm), t(p.cells), t(p.first), t(p.count), t(F["centre"]), None, None, None, None,
                             t(F["cp"][0]), t(F["cp"][1]), None, None, F["eps"], out, flags=binding.PP_LEAVES)


def test_conditioning_test_sees_the_total(ctx, torch):
    """With PKDG_FIXUP_ALL every sink's near part is re-evaluated in fp64 and added to the local-expansion part the
    first kernel wrote: the combined call must still be the oracle's total."""
    from paper_1609_08621_b200 import binding, inputs
    p = inputs.config1(4096, seed=3, theta=0.6)
    F = inputs.build_fmm_lists(p, 0.6, p.eps)
    ref = _oracle(p, F)
    for flags in (binding.FIXUP_ALL, binding.NO_FIXUP):
        out = _run(ctx, torch, p, F, flags=flags)
        _assert_parity(out, ref, label=f"cfg1 theta=0.6 flags={flags:#x}")
    assert ctx.get_stats()["fixup_sinks"] == 0
