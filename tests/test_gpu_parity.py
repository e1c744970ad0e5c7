"""-m gpu parity tests: the CUDA path, called through the C ABI, against the fp64 oracle on the
same seeded inputs.  Bars (BASELINE.json north_star): integer work bit-exact; per-particle
|a_gpu - a_or|/|a_or| <= 2e-5 and |phi_gpu - phi_or|/|phi_or| <= 2e-5."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-5
MODES = [0, 0x10, 0x20]   # default (fp32 + conditioning-triggered fp64 fix-up), PKDG_NO_FIXUP, PKDG_FIXUP_ALL


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


def _oracle(p, sel=None):
    import oracle
    return oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, sel=sel)


@pytest.mark.parametrize("flags", MODES)
def test_config1_full_parity(ctx, torch, cfg1, flags):
    """configs[0]: N = 4096 uniform, octree, theta = 0.7 -- every particle against the oracle."""
    from gpu_util import rel_errors, run_resident
    ref = _oracle(cfg1)
    out = run_resident(ctx, cfg1, torch, flags=flags)
    ea, ep = rel_errors(out, ref)
    assert np.isfinite(out).all()
    assert ea.max() <= TOL and ep.max() <= TOL, (ea.max(), ep.max())
    st = ctx.get_stats()
    import oracle
    assert st["interactions_pp"] == oracle.interactions(cfg1.count, cfg1.pp_off) == cfg1.I_pp
    assert st["interactions_pc"] == oracle.interactions(cfg1.count, cfg1.pc_off) == cfg1.I_pc
    assert st["bad_entries"] == 0 and st["n_buckets"] == cfg1.n_buckets


def test_pp_only_and_pc_only_sum_to_full(ctx, torch, cfg1):
    from paper_1609_08621_b200 import binding
    from gpu_util import rel_errors, run_resident
    import oracle
    p = cfg1
    ref_pp = oracle.gravity_eval(p.xyzm, None, p.first, p.count, p.pp_off, p.pp_idx, None, None, p.eps)
    ref_pc = oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, None, None, p.pc_off, p.pc_idx, p.eps)
    out_pp = run_resident(ctx, p, torch, flags=binding.SKIP_PC)
    out_pc = run_resident(ctx, p, torch, flags=binding.SKIP_PP)
    for out, ref in ((out_pp, ref_pp), (out_pc, ref_pc)):
        ea, ep = rel_errors(out, ref)
        assert ea.max() <= TOL and ep.max() <= TOL


def test_accumulate_flag_adds(ctx, torch, cfg1):
    from paper_1609_08621_b200 import binding
    from gpu_util import run_resident
    base = run_resident(ctx, cfg1, torch)
    acc = run_resident(ctx, cfg1, torch, flags=binding.ACCUMULATE, fill=1.0)
    assert np.allclose(acc, base + 1.0, rtol=1e-6, atol=1e-6)


def test_pack_export_bit_exact(ctx, torch, cfg1):
    """a1: tiles and tile offsets equal the oracle's packer spec bit for bit (list order kept)."""
    import oracle
    for off, idx in ((cfg1.pp_off, cfg1.pp_idx), (cfg1.pc_off, cfg1.pc_idx)):
        tile_off, tiles = oracle.pack_tiles(off, idx)
        d_off = torch.from_numpy(off).cuda(); d_idx = torch.from_numpy(idx).cuda()
        g_off = torch.zeros(off.shape[0], dtype=torch.int64, device="cuda")
        g_tiles = torch.full((tiles.shape[0] + 3, 32), -7, dtype=torch.int32, device="cuda")
        ctx.pack_export(off.shape[0] - 1, d_off, d_idx, g_off, g_tiles)
        torch.cuda.synchronize()
        assert np.array_equal(g_off.cpu().numpy(), tile_off)
        assert np.array_equal(g_tiles.cpu().numpy()[: tiles.shape[0]], tiles)
        assert np.all(g_tiles.cpu().numpy()[tiles.shape[0]:] == -7)


def test_pack_export_ragged_empty_and_paper_example(ctx, torch):
    import oracle
    lens = [0, 1, 31, 32, 33, 655, 0, 64, 0]
    off = np.concatenate([[5], 5 + np.cumsum(lens)]).astype(np.int64)      # offsets[0] != 0
    idx = (np.arange(off[-1], dtype=np.int64) * 7 % 1000).astype(np.int32)
    tile_off, tiles = oracle.pack_tiles(off, idx)
    g_off = torch.zeros(off.shape[0], dtype=torch.int64, device="cuda")
    g_tiles = torch.zeros((tiles.shape[0], 32), dtype=torch.int32, device="cuda")
    ctx.pack_export(len(lens), torch.from_numpy(off).cuda(), torch.from_numpy(idx).cuda(), g_off, g_tiles)
    torch.cuda.synchronize()
    assert np.array_equal(g_off.cpu().numpy(), tile_off) and np.array_equal(g_tiles.cpu().numpy(), tiles)
    assert tile_off[6] - tile_off[5] == 21                                 # 655 -> 20 full tiles + 15
    # capacity too small: offsets still complete
    g_off.zero_()
    ctx.pack_export(len(lens), torch.from_numpy(off).cuda(), torch.from_numpy(idx).cuda(), g_off, g_tiles[:3].contiguous())
    torch.cuda.synchronize()
    assert np.array_equal(g_off.cpu().numpy(), tile_off)


def _edge_problem():
    """Ragged and degenerate buckets: empty bucket, empty lists, counts 1, 17 and 27 (> 16), padding
    entries, a coincident pair, softened neighbours, list lengths around the tile size."""
    from paper_1609_08621_b200 import inputs
    rng = np.random.default_rng(42)
    counts = [0, 1, 16, 17, 27, 3, 8, 5]
    n_t = sum(counts)
    n_src = 700
    xyzm = np.empty((n_t + n_src, 4), np.float32)
    xyzm[:n_t, :3] = 0.5 + 0.01 * rng.standard_normal((n_t, 3))
    xyzm[n_t:, :3] = rng.random((n_src, 3))
    xyzm[:, 3] = rng.uniform(0.5, 1.5, n_t + n_src) / (n_t + n_src)
    xyzm[3, :3] = xyzm[2, :3]                                           # coincident distinct particles
    first = np.concatenate([[0], np.cumsum(counts)[:-1]]).astype(np.int32)
    count = np.array(counts, np.int32)
    pp_lens = [40, 0, 33, 64, 700 + n_t, 31, 1, 0]
    pp = []
    for b, L in enumerate(pp_lens):
        own = np.arange(first[b], first[b] + count[b])
        if L >= n_src + n_t:
            l = np.arange(n_t + n_src)
        else:
            l = np.concatenate([own, n_t + rng.choice(n_src, max(L - own.size, 0), replace=False)])[:L]
        l = l.astype(np.int32)
        if b == 2:
            l[5] = -1                                                   # padding inside a list is ignored
        pp.append(l)
    pp_off = np.concatenate([[0], np.cumsum([len(l) for l in pp])]).astype(np.int64)
    pp_idx = np.concatenate(pp).astype(np.int32)
    # cells: clouds well away from the targets
    ncell = 150
    com = 0.5 + rng.choice([-1, 1], (ncell, 3)) * rng.uniform(0.15, 0.45, (ncell, 3))
    pts = np.empty((ncell * 20, 4), np.float32)
    pts[:, :3] = np.repeat(com, 20, axis=0) + 0.02 * rng.standard_normal((ncell * 20, 3))
    pts[:, 3] = rng.uniform(0.5, 1.5, ncell * 20) / (ncell * 20)
    cells = inputs.cloud_records(pts, 20)
    cells[7, 35] = 0.0                                                  # b_max <= 0: scale from 2nd moments
    cells[9, 4:35] = 0.0                                                # pure monopole cell
    pc_lens = [0, 150, 32, 31, 65, 1, 150, 0]
    pc = [rng.choice(ncell, L, replace=False).astype(np.int32) for L in pc_lens]
    pc_off = np.concatenate([[0], np.cumsum(pc_lens)]).astype(np.int64)
    pc_idx = np.concatenate(pc).astype(np.int32)
    return inputs.Problem(name="edge", xyzm=xyzm, cells=cells, first=first, count=count, pp_off=pp_off,
                          pp_idx=pp_idx, pc_off=pc_off, pc_idx=pc_idx, eps=float(np.float32(0.004)))


@pytest.mark.parametrize("flags", MODES)
def test_edge_cases(ctx, torch, flags):
    from gpu_util import rel_errors, run_resident
    p = _edge_problem()
    ref = _oracle(p)
    out = run_resident(ctx, p, torch, flags=flags)
    rows = np.arange(int(p.first[7]))                                   # bucket 7 has no lists at all
    ea, ep = rel_errors(out, ref, rows)
    assert ea.max() <= TOL and ep.max() <= TOL, (ea.max(), ep.max())
    lone = out[p.first[7]: p.first[7] + p.count[7]]
    assert np.all(lone == 0.0) and np.all(ref[p.first[7]: p.first[7] + p.count[7]] == 0.0)   # overwritten with 0
    assert np.isnan(out[int(p.count.sum()):]).all()                     # particles in no bucket: untouched
    assert ctx.get_stats()["bad_entries"] == 0


def _layout_problem(seed=7):
    """Every bucket occupancy 0 .. 35 (all lane layouts of the bucket kernel: 1 x 32, 2 x 16, 3 x 10, 4 x 8, 5 x 6,
    6 x 5, 8 x 4, and passes beyond 16 sinks) against list lengths on both sides of the 30- and 32-slot tile
    boundaries.  The buckets' own particles are on their P-P lists (self pairs), some pairs are softened."""
    from paper_1609_08621_b200 import inputs
    rng = np.random.default_rng(seed)
    lens = [0, 1, 4, 5, 29, 30, 31, 32, 33, 59, 60, 61, 63, 64, 65, 90, 96, 127, 150, 301]
    counts = [c for c in range(36) for _ in range(3)]
    nb = len(counts)
    n_t = sum(counts)
    n_src = 1200
    xyzm = np.empty((n_t + n_src, 4), np.float32)
    centre = 0.5 + 0.2 * rng.standard_normal((nb, 3))
    first = np.concatenate([[0], np.cumsum(counts)[:-1]]).astype(np.int32)
    count = np.array(counts, np.int32)
    for b in range(nb):
        xyzm[first[b]: first[b] + count[b], :3] = centre[b] + 0.004 * rng.standard_normal((count[b], 3))
    xyzm[n_t:, :3] = 0.5 + 0.25 * rng.standard_normal((n_src, 3))
    xyzm[:, 3] = rng.uniform(0.5, 1.5, n_t + n_src) / (n_t + n_src)
    pp, pc = [], []
    ncell = 400
    com = 0.5 + rng.choice([-1, 1], (ncell, 3)) * rng.uniform(1.2, 2.0, (ncell, 3))
    pts = np.empty((ncell * 12, 4), np.float32)
    pts[:, :3] = np.repeat(com, 12, axis=0) + 0.03 * rng.standard_normal((ncell * 12, 3))
    pts[:, 3] = rng.uniform(0.5, 1.5, ncell * 12) / (ncell * 12)
    cells = inputs.cloud_records(pts, 12)
    for b in range(nb):
        own = np.arange(first[b], first[b] + count[b])
        L = lens[(b * 7 + 3) % len(lens)]
        l = np.concatenate([own, n_t + rng.choice(n_src, L, replace=False)]).astype(np.int32)
        rng.shuffle(l)                                                  # own particles anywhere in the list
        pp.append(l)
        pc.append(rng.choice(ncell, lens[(b * 11 + 5) % len(lens)], replace=False).astype(np.int32))
    pp_off = np.concatenate([[0], np.cumsum([len(l) for l in pp])]).astype(np.int64)
    pc_off = np.concatenate([[0], np.cumsum([len(l) for l in pc])]).astype(np.int64)
    return inputs.Problem(name="layouts", xyzm=xyzm, cells=cells, first=first, count=count, pp_off=pp_off,
                          pp_idx=np.concatenate(pp).astype(np.int32), pc_off=pc_off,
                          pc_idx=np.concatenate(pc).astype(np.int32), eps=float(np.float32(0.003)))


@pytest.mark.parametrize("flags", MODES)
def test_every_bucket_occupancy_and_lane_layout(ctx, torch, flags):
    from gpu_util import rel_errors, run_resident
    p = _layout_problem()
    ref = _oracle(p)
    out = run_resident(ctx, p, torch, flags=flags)
    st = ctx.get_stats()
    assert st["interactions_pp"] == p.I_pp and st["interactions_pc"] == p.I_pc and st["bad_entries"] == 0
    n_t = int(p.count.sum())
    ea, ep = rel_errors(out, ref, np.arange(n_t))
    worst = int(np.argmax(ea))
    assert ea.max() <= TOL and ep.max() <= TOL, (ea.max(), ep.max(), int(np.searchsorted(p.first, worst, "right") - 1))
    assert np.isnan(out[n_t:]).all()                                    # sources are in no bucket: untouched


def test_softened_plummer_cores(ctx, torch):
    """configs[1] recipe at N = 2^15: dense Plummer cores put many pairs inside the spline."""
    from paper_1609_08621_b200 import inputs
    from gpu_util import rel_errors, run_resident
    p = inputs.config2(n=1 << 15)
    ref = _oracle(p)
    out = run_resident(ctx, p, torch)
    ea, ep = rel_errors(out, ref)
    assert ea.max() <= TOL and ep.max() <= TOL, (ea.max(), ep.max())


def test_out_of_range_indices_are_reported_not_followed(ctx, torch, cfg1):
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import run_resident
    import copy
    p = copy.copy(cfg1)
    p.pp_idx = cfg1.pp_idx.copy(); p.pc_idx = cfg1.pc_idx.copy()
    p.pp_idx[10] = cfg1.n + 5
    p.pc_idx[3] = cfg1.cells.shape[0]
    run_resident(ctx, p, torch)
    with pytest.raises(binding.PkdgError):
        ctx.get_stats()
    assert ctx.get_stats(check=False)["bad_entries"] >= 2


def test_invalid_arguments_fail_loudly(ctx, torch, cfg1):
    from paper_1609_08621_b200 import binding
    from gpu_util import to_dev
    d = to_dev(cfg1, torch)
    out = torch.zeros((cfg1.n, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(binding.PkdgError):
        ctx.gravity_eval(d["xyzm"], d["cells"][:, :20].contiguous(), d["first"], d["count"], d["pp_off"], d["pp_idx"],
                         d["pc_off"], d["pc_idx"], cfg1.eps, out)
    with pytest.raises(binding.PkdgError):
        ctx.set_option(binding.OPT_KAPPA2, -1.0)
    with pytest.raises(binding.PkdgError):
        ctx.set_option(77, 1.0)


def test_streamed_and_host_variants_match_resident(ctx, torch, cfg1):
    """a6: chunked evaluation from host lists gives the same bits as the resident call."""
    from paper_1609_08621_b200 import binding
    from gpu_util import run_resident, to_dev
    import oracle
    p = cfg1
    base = run_resident(ctx, p, torch)
    d = to_dev(p, torch)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h = dict(first=pin(p.first), count=pin(p.count), pp_off=pin(p.pp_off), pp_idx=pin(p.pp_idx),
             pc_off=pin(p.pc_off), pc_idx=pin(p.pc_idx))
    for n_streams, max_entries in ((1, 1 << 30), (3, 5000), (2, 300), (4, 1)):
        out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda")
        ctx.gravity_eval_streamed(d["xyzm"], d["cells"], h["first"], h["count"], h["pp_off"], h["pp_idx"],
                                  h["pc_off"], h["pc_idx"], p.eps, out, n_streams=n_streams,
                                  max_entries_per_chunk=max_entries)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), base)
        st = ctx.get_stats()
        b_or = oracle.chunk_bounds(p.pp_off, p.pc_off, max_entries)
        b_lib = binding.chunk_bounds(p.pp_off, p.pc_off, max_entries)
        assert np.array_equal(b_or, b_lib) and st["chunks"] == len(b_or) - 1
        assert st["interactions_pp"] == p.I_pp and st["interactions_pc"] == p.I_pc
    out_h = np.full((p.n, 4), np.nan, np.float32)
    ctx.gravity_eval_host(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, out_h,
                          n_streams=3, max_entries_per_chunk=20000)
    assert np.array_equal(out_h, base)


def test_prepared_cells_reproduce_oracle_pc_over_distances(ctx, torch):
    """P-C alone, one cell, targets from 1.5 to 40 cell radii in many directions."""
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import rel_errors, run_resident
    rng = np.random.default_rng(3)
    pts = np.empty((48, 4), np.float32)
    pts[:, :3] = 0.3 + 0.01 * rng.standard_normal((48, 3)); pts[:, 3] = rng.uniform(0.5, 1.5, 48) / 48
    cells = inputs.cloud_records(pts, 48)
    b = float(cells[0, 35])
    nt = 16 * 40
    v = rng.standard_normal((nt, 3)); v /= np.linalg.norm(v, axis=1)[:, None]
    dist = b * np.exp(rng.uniform(np.log(1.5), np.log(40), nt))
    xyzm = np.zeros((nt, 4), np.float32)
    xyzm[:, :3] = cells[0, :3] + dist[:, None] * v
    xyzm[:, 3] = 1.0 / nt
    first = np.arange(0, nt, 16, dtype=np.int32); count = np.full(40, 16, np.int32)
    pc_off = np.arange(41, dtype=np.int64); pc_idx = np.zeros(40, np.int32)
    p = inputs.Problem(name="pc1", xyzm=xyzm, cells=cells, first=first, count=count, pp_off=None, pp_idx=None,
                       pc_off=pc_off, pc_idx=pc_idx, eps=0.0)
    ref = _oracle(p)
    out = run_resident(ctx, p, torch)
    ea, ep = rel_errors(out, ref)
    assert ea.max() <= 5e-6 and ep.max() <= 2e-6, (ea.max(), ep.max())


def test_config4_sweep_small(ctx, torch):
    """configs[3] recipe at 256 buckets: a few (L_pp, L_pc) shapes incl. non-multiples of 32."""
    from paper_1609_08621_b200 import inputs
    from gpu_util import rel_errors, run_resident
    for lpp, lpc in ((32, 32), (128, 0), (0, 128), (100, 70), (512, 512)):
        p = inputs.config4(256, lpp, lpc)
        ref = _oracle(p)
        out = run_resident(ctx, p, torch)
        ea, ep = rel_errors(out, ref, np.arange(256 * 16))
        assert ea.max() <= TOL and ep.max() <= TOL, (lpp, lpc, ea.max(), ep.max())


def _leaf_problem(p):
    """The same problem with its P-P lists in leaf form (references to whole buckets)."""
    import copy
    from paper_1609_08621_b200 import inputs
    q = copy.copy(p)
    q.pp_off, q.pp_idx = inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)
    eo, ei = inputs.expand_leaves(p.first, p.count, q.pp_off, q.pp_idx)
    assert np.array_equal(eo, p.pp_off) and np.array_equal(ei, p.pp_idx)      # the references stand for the same lists
    return q


@pytest.mark.parametrize("flags", MODES)
def test_pp_leaves_resident(ctx, torch, cfg1, flags):
    """PKDG_PP_LEAVES: leaf references give the oracle's result of the expanded lists, and the same
    interaction count; tiles_pp counts two references per tile."""
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import rel_errors, run_resident
    for p in (cfg1, inputs.config2(n=1 << 15), inputs.config3(32)):
        q = _leaf_problem(p)
        ref = _oracle(p)
        out = run_resident(ctx, q, torch, flags=flags | binding.PP_LEAVES)
        st = ctx.get_stats()
        ea, ep = rel_errors(out, ref)
        assert ea.max() <= TOL and ep.max() <= TOL, (p.name, ea.max(), ep.max())
        assert st["interactions_pp"] == p.I_pp and st["interactions_pc"] == p.I_pc and st["bad_entries"] == 0
        assert st["tiles_pp"] == int(((np.diff(q.pp_off) + 1) // 2).sum())
        base = run_resident(ctx, p, torch, flags=flags)                       # particle lists: same sums, other order
        eb, epb = rel_errors(out, base.astype(np.float64))
        assert eb.max() <= 1e-5 and epb.max() <= 2e-6


def test_pp_leaves_streamed_host_and_bad_references(ctx, torch, cfg1):
    from paper_1609_08621_b200 import binding
    from gpu_util import run_resident, to_dev
    p = cfg1
    q = _leaf_problem(p)
    base = run_resident(ctx, q, torch, flags=binding.PP_LEAVES)
    d = to_dev(q, torch)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    h = dict(first=pin(q.first), count=pin(q.count), pp_off=pin(q.pp_off), pp_idx=pin(q.pp_idx),
             pc_off=pin(q.pc_off), pc_idx=pin(q.pc_idx))
    for n_streams, max_entries in ((1, 1 << 30), (3, 700), (2, 40)):
        out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda")
        ctx.gravity_eval_streamed(d["xyzm"], d["cells"], h["first"], h["count"], h["pp_off"], h["pp_idx"],
                                  h["pc_off"], h["pc_idx"], p.eps, out, n_streams=n_streams,
                                  max_entries_per_chunk=max_entries, flags=binding.PP_LEAVES)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), base)
        st = ctx.get_stats()
        assert st["interactions_pp"] == p.I_pp and st["interactions_pc"] == p.I_pc and st["chunks"] >= 1
    out_h = np.full((p.n, 4), np.nan, np.float32)
    ctx.gravity_eval_host(q.xyzm, q.cells, q.first, q.count, q.pp_off, q.pp_idx, q.pc_off, q.pc_idx, p.eps, out_h,
                          n_streams=3, max_entries_per_chunk=5000, flags=binding.PP_LEAVES)
    assert np.array_equal(out_h, base)
    # a reference out of range is reported, not followed (fp32 path and fp64 fix-up kernel alike)
    bad = _leaf_problem(p)
    bad.pp_idx = bad.pp_idx.copy(); bad.pp_idx[3] = p.n_buckets + 5
    for fl in (0, binding.FIXUP_ALL):
        out = run_resident(ctx, bad, torch, flags=binding.PP_LEAVES | fl)
        assert np.isfinite(out).all()
        assert ctx.get_stats(check=False)["bad_entries"] > 0


def test_fixup_kernel_is_fp64_accurate(ctx, torch, cfg1):
    """PKDG_FIXUP_ALL: every sink through pkdg_fixup_kernel (fp64 terms and accumulators).  What is left is
    the fp32 rounding of the OUTPUT (2^-24 per component), independent of the conditioning of the sum."""
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import rel_errors, run_resident
    for p in (cfg1, inputs.config2(n=1 << 14), _edge_problem(), inputs.config4(512, 100, 70)):
        ref = _oracle(p)
        out = run_resident(ctx, p, torch, flags=binding.FIXUP_ALL)
        st = ctx.get_stats()
        rows = np.flatnonzero(np.isfinite(ref[:, 0]) & (np.linalg.norm(ref[:, :3], axis=1) > 0))
        ea, ep = rel_errors(out, ref, rows)
        assert ea.max() <= 1.5e-7 and ep.max() <= 1.0e-7, (p.name, ea.max(), ep.max())
        assert st["fixup_sinks"] == int(p.count.sum()), (p.name, st["fixup_sinks"])
        # PKDG_NO_FIXUP never queues anything; the default queues a small minority
        run_resident(ctx, p, torch, flags=binding.NO_FIXUP)
        assert ctx.get_stats()["fixup_sinks"] == 0
        run_resident(ctx, p, torch)
        assert ctx.get_stats()["fixup_sinks"] <= 0.3 * int(p.count.sum()) + 4, p.name


def test_fixup_threshold_option_and_accumulate(ctx, torch, cfg1):
    """PKDG_OPT_KAPPA2 moves the threshold (a tiny kappa2 queues everything); PKDG_ACCUMULATE adds in both kernels."""
    from paper_1609_08621_b200 import binding
    from gpu_util import run_resident
    p = cfg1
    base = run_resident(ctx, p, torch, flags=binding.FIXUP_ALL)
    ctx.set_option(binding.OPT_KAPPA2, 1e-3)
    try:
        out = run_resident(ctx, p, torch)
        assert ctx.get_stats()["fixup_sinks"] == p.n
        assert np.array_equal(out, base)
        acc = run_resident(ctx, p, torch, flags=binding.ACCUMULATE, fill=1.0)
        assert np.allclose(acc, base + 1.0, rtol=1e-6, atol=1e-6)
        ctx.set_option(binding.OPT_KAPPA2, 1.5)
        mixed = run_resident(ctx, p, torch)
        n_fix = ctx.get_stats()["fixup_sinks"]
        assert 0 < n_fix < p.n
        acc = run_resident(ctx, p, torch, flags=binding.ACCUMULATE, fill=1.0)
        assert np.allclose(acc, mixed + 1.0, rtol=1e-6, atol=1e-6)
    finally:
        ctx.set_option(binding.OPT_KAPPA2, 6.0)   # the library default (kDefaultKappa2)


def test_validate_flag_checks_the_value_range_contract(ctx, torch, cfg1):
    """PKDG_VALIDATE (include/pkdg.h "Value range"): clean input passes; a NaN mass, a coordinate beyond 1e12
    and an infinite moment are counted as invalid_values; a listed cell whose b_max sphere holds the sinks
    (here: the root cell) is counted pair by pair as invalid_pairs; pkdg_get_stats reports PKDG_EBADVALUE."""
    import copy
    from paper_1609_08621_b200 import binding
    from gpu_util import run_resident
    p = cfg1
    base = run_resident(ctx, p, torch)
    out = run_resident(ctx, p, torch, flags=binding.VALIDATE)
    st = ctx.get_stats()
    assert st["invalid_values"] == 0 and st["invalid_pairs"] == 0 and np.array_equal(out, base)
    q = copy.copy(p)
    q.xyzm = p.xyzm.copy(); q.cells = p.cells.copy(); q.pc_idx = p.pc_idx.copy()
    q.xyzm[5, 3] = np.nan; q.xyzm[9, 1] = 2.0e13; q.cells[3, 17] = np.inf
    b = 40
    q.pc_idx[p.pc_off[b]] = 0                       # the root cell: every sink of bucket b lies inside its b_max
    run_resident(ctx, q, torch, flags=binding.VALIDATE)
    with pytest.raises(binding.PkdgError, match="EBADVALUE"):
        ctx.get_stats()
    st = ctx.get_stats(check=False)
    assert st["invalid_values"] == 3 and st["invalid_pairs"] == int(p.count[b]) and st["bad_entries"] == 0
    # the streamed variants check too
    d_x = torch.from_numpy(q.xyzm).cuda(); d_c = torch.from_numpy(q.cells).cuda()
    out = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda")
    pin = lambda a: torch.from_numpy(a).pin_memory()
    ctx.gravity_eval_streamed(d_x, d_c, pin(q.first), pin(q.count), pin(q.pp_off), pin(q.pp_idx), pin(q.pc_off),
                              pin(q.pc_idx), p.eps, out, n_streams=2, max_entries_per_chunk=20000, flags=binding.VALIDATE)
    st = ctx.get_stats(check=False)
    assert st["invalid_values"] == 3 and st["invalid_pairs"] == int(p.count[b])


def test_eps_zero_is_newtonian(ctx, torch, cfg1):
    """eps = 0: pure Newtonian pairs in both kernels (no pair of config 1 is closer than 1e-12)."""
    import copy
    from paper_1609_08621_b200 import binding
    from gpu_util import rel_errors, run_resident
    p = copy.copy(cfg1); p.eps = 0.0
    ref = _oracle(p)
    for fl in (0, binding.FIXUP_ALL):
        out = run_resident(ctx, p, torch, flags=fl)
        ea, ep = rel_errors(out, ref)
        assert ea.max() <= TOL and ep.max() <= TOL, (fl, ea.max(), ep.max())


def test_range_call_and_host_range_keep_other_rows(ctx, torch, cfg1):
    """pkdg_gravity_eval_range / pkdg_gravity_eval_host_range: buckets [b0, b1) over the FULL bucket arrays, lists
    of the range only; rows outside the range keep their values; leaf references stay global."""
    from paper_1609_08621_b200 import binding, shard
    from gpu_util import run_resident, to_dev
    p = cfg1
    base = run_resident(ctx, p, torch)
    q = _leaf_problem(p)
    base_l = run_resident(ctx, q, torch, flags=binding.PP_LEAVES)
    d = to_dev(p, torch)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for prob, ref, fl in ((p, base, 0), (q, base_l, binding.PP_LEAVES)):
        out = torch.full((p.n, 4), -7.0, dtype=torch.float32, device="cuda")
        out_h = np.full((p.n, 4), -7.0, np.float32)
        seen = np.zeros(p.n, bool)
        for r in range(3):
            pc = shard.rank_piece(prob, r, 3, pp_weights=p.count[prob.pp_idx] if fl else None)
            ctx.gravity_eval_range(d["xyzm"], d["cells"], d["first"], d["count"], pc.b0, pc.b1, t(pc.pp_off), t(pc.pp_idx),
                                   t(pc.pc_off), t(pc.pc_idx), p.eps, out, flags=fl)
            torch.cuda.synchronize()
            assert ctx.get_stats()["n_buckets"] == pc.n_buckets
            ctx.gravity_eval_host_range(p.xyzm, p.cells, p.first, p.count, pc.b0, pc.b1, pc.pp_off,
                                        np.ascontiguousarray(pc.pp_idx), pc.pc_off, np.ascontiguousarray(pc.pc_idx), p.eps,
                                        out_h, n_streams=2, max_entries_per_chunk=30000, flags=fl)
            seen[shard.rank_rows(p.first, p.count, pc.b0, pc.b1)] = True
            got = out.cpu().numpy()
            for o in (got, out_h):
                assert np.array_equal(o[seen], ref[seen]) and np.all(o[~seen] == -7.0), r
        assert seen.all()


def _group_problem(p, gmax=64):
    """Group-shared lists of problem p (reading A6 with the group cell as the sink) + the per-bucket lists they
    stand for (pure indexing), which is what the oracle evaluates."""
    import copy
    from paper_1609_08621_b200 import inputs
    gc, gf, gn = inputs.build_groups(p, gmax)
    ppo, ppi, pco, pci = inputs.build_group_lists(p, gc, p.theta, p.eps)
    q = copy.copy(p)
    q.pp_off, q.pp_idx = inputs.expand_groups(gf, gn, ppo, ppi)
    q.pc_off, q.pc_idx = inputs.expand_groups(gf, gn, pco, pci)
    return (gf, gn, ppo, ppi, pco, pci), q


def test_group_shared_lists(ctx, torch, cfg1):
    """SURVEY.md sec 8(f) NEXT-1 / PAPER.md:L69: one P-P and one P-C list per group of <= 64 particles.  The
    library's result on group lists equals the oracle's on the expanded per-bucket lists; counters count
    sink x entry interactions of the expanded lists; the all-host call gives the same bits; leaf-form P-P
    entries work with groups; groups that do not tile the buckets are rejected / reported."""
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import rel_errors
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    for p in (cfg1, inputs.config2(n=1 << 15), inputs.config3(32)):
        (gf, gn, ppo, ppi, pco, pci), q = _group_problem(p)
        assert gn.sum() == p.n_buckets and (ppo.shape[0] - 1) * 2 < p.n_buckets
        ref = _oracle(q)
        d = dict(xyzm=t(p.xyzm), cells=t(p.cells), first=t(p.first), count=t(p.count))
        for fl in MODES:
            out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda")
            ctx.gravity_eval_groups(d["xyzm"], d["cells"], d["first"], d["count"], t(gf), t(gn), t(ppo), t(ppi), t(pco),
                                    t(pci), p.eps, out, flags=fl)
            torch.cuda.synchronize()
            st = ctx.get_stats()
            assert st["interactions_pp"] == q.I_pp and st["interactions_pc"] == q.I_pc and st["bad_entries"] == 0
            assert st["tiles_pp"] == int((((np.diff(ppo) + 31) // 32) * gn).sum())
            ea, ep = rel_errors(out.cpu().numpy(), ref)
            assert ea.max() <= TOL and ep.max() <= TOL, (p.name, fl, ea.max(), ep.max())
        base = out.cpu().numpy() if fl == MODES[-1] else None
        out0 = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda")
        ctx.gravity_eval_groups(d["xyzm"], d["cells"], d["first"], d["count"], t(gf), t(gn), t(ppo), t(ppi), t(pco), t(pci),
                                p.eps, out0)
        torch.cuda.synchronize()
        base = out0.cpu().numpy()
        # all-host call, chunks are ranges of groups
        out_h = np.full((p.n, 4), np.nan, np.float32)
        ctx.gravity_eval_host_groups(p.xyzm, p.cells, p.first, p.count, gf, gn, ppo, ppi, pco, pci, p.eps, out_h,
                                     n_streams=3, max_entries_per_chunk=20000)
        assert np.array_equal(out_h, base) and ctx.get_stats()["chunks"] > 1
        # leaf-form P-P entries (bucket references) with groups
        lo, li = inputs.pp_leaves(p.n, p.first, p.count, ppo, ppi)
        outl = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device="cuda")
        ctx.gravity_eval_groups(d["xyzm"], d["cells"], d["first"], d["count"], t(gf), t(gn), t(lo), t(li), t(pco), t(pci),
                                p.eps, outl, flags=binding.PP_LEAVES)
        torch.cuda.synchronize()
        st = ctx.get_stats()
        assert st["interactions_pp"] == q.I_pp and st["bad_entries"] == 0
        ea, ep = rel_errors(outl.cpu().numpy(), ref)
        assert ea.max() <= TOL and ep.max() <= TOL, (p.name, "leaves", ea.max(), ep.max())
        out_h = np.full((p.n, 4), np.nan, np.float32)
        ctx.gravity_eval_host_groups(p.xyzm, p.cells, p.first, p.count, gf, gn, lo, li, pco, pci, p.eps, out_h,
                                     n_streams=2, max_entries_per_chunk=5000, flags=binding.PP_LEAVES)
        assert np.array_equal(out_h, outl.cpu().numpy())
    # groups that do not tile the buckets
    p = cfg1
    (gf, gn, ppo, ppi, pco, pci), q = _group_problem(p)
    bad_gn = gn.copy(); bad_gn[3] += 1
    out = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda")
    ctx.gravity_eval_groups(t(p.xyzm), t(p.cells), t(p.first), t(p.count), t(gf), t(bad_gn), t(ppo), t(ppi), t(pco), t(pci),
                            p.eps, out)
    torch.cuda.synchronize()
    assert ctx.get_stats(check=False)["bad_entries"] > 0
    # group 3 now reaches into group 4's first bucket, so group 4 no longer starts where group 3 ends: it gets no
    # work at all (its other buckets keep the caller's zeros) instead of racing with group 3 on the shared bucket;
    # every group that tiles correctly evaluates as before
    good = torch.zeros((p.n, 4), dtype=torch.float32, device="cuda")
    ctx.gravity_eval_groups(t(p.xyzm), t(p.cells), t(p.first), t(p.count), t(gf), t(gn), t(ppo), t(ppi), t(pco), t(pci),
                            p.eps, good)
    torch.cuda.synchronize()
    got, good = out.cpu().numpy(), good.cpu().numpy()
    rows = lambda g0, g1: np.arange(p.first[gf[g0]], p.first[gf[g1 - 1] + gn[g1 - 1] - 1] + p.count[gf[g1 - 1] + gn[g1 - 1] - 1])
    assert np.array_equal(got[rows(0, 3)], good[rows(0, 3)]) and np.array_equal(got[rows(5, len(gf))], good[rows(5, len(gf))])
    if gn[4] > 1:
        skipped = np.arange(p.first[gf[4] + 1], p.first[gf[4] + gn[4] - 1] + p.count[gf[4] + gn[4] - 1])
        assert (got[skipped] == 0).all()
    with pytest.raises(binding.PkdgError):
        ctx.gravity_eval_host_groups(p.xyzm, p.cells, p.first, p.count, gf, bad_gn, ppo, ppi, pco, pci, p.eps,
                                     np.zeros((p.n, 4), np.float32))


def _device_lists(ctx, torch, p, sink_cell, theta, eps, flags=0):
    """pkdg_build_lists_count + _fill for the tree of problem p; returns host arrays."""
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    tr = p.tree
    leaf_rank = (np.cumsum(tr["isleaf"] != 0) - 1).astype(np.int32)
    tree = dict(first=t(tr["first"]), count=t(tr["count"]), end=t(tr["end"]), isleaf=t(tr["isleaf"]), bblo=t(tr["bblo"]),
                bbhi=t(tr["bbhi"]), leaf_rank=t(leaf_rank))
    cells = t(p.cells); sc = t(sink_cell.astype(np.int32))
    ns = sink_cell.shape[0]
    pp_off = torch.empty(ns + 1, dtype=torch.int64, device="cuda"); pc_off = torch.empty(ns + 1, dtype=torch.int64, device="cuda")
    npp, npc = ctx.build_lists_count(tree, cells, sc, theta, eps, pp_off, pc_off, flags=flags)
    pp_idx = torch.full((npp + 1,), -9, dtype=torch.int32, device="cuda"); pc_idx = torch.full((npc + 1,), -9, dtype=torch.int32, device="cuda")
    ctx.build_lists_fill(tree, cells, sc, theta, eps, pp_off, pc_off, pp_idx, pc_idx, flags=flags)
    torch.cuda.synchronize()
    assert int(pp_idx[-1]) == -9 and int(pc_idx[-1]) == -9          # nothing written past the totals
    return pp_off.cpu().numpy(), pp_idx[:-1].cpu().numpy(), pc_off.cpu().numpy(), pc_idx[:-1].cpu().numpy()


def test_device_list_construction_is_bit_exact(ctx, torch, cfg1):
    """the tree walk on the device (pkdg_build_lists_*) gives the SAME offsets and the
    SAME indices as the ORACLE's walk (oracle.walk_lists: the recursive statement of PAPER.md:L65-69 / readings A6,
    pinned in tests/test_oracle_walk_pins.py) -- integer work, bit-exact -- for per-bucket lists, group-shared lists
    and leaf-form P-P entries; theta = 0.7 and 0.55; octree and binary trees.  The input generator's lists (what the
    other parity tests evaluate) are compared with the same oracle walk here at these sizes too."""
    import oracle
    from paper_1609_08621_b200 import binding, inputs
    flat = lambda w: (w[0][0], w[0][1], w[1][0], w[1][1])
    for p, theta in ((cfg1, 0.7), (inputs.config2(n=1 << 15), 0.7), (inputs.config3(32), 0.55), (inputs.config3(64), 0.7)):
        if theta != p.theta:
            p = inputs.with_lists(p, theta, p.eps)
        want = flat(oracle.walk_lists(p.tree, p.cells, p.tree["leaf_cell"], theta, p.eps))
        got = _device_lists(ctx, torch, p, p.tree["leaf_cell"], theta, p.eps)
        for a, b, c, name in zip(got, want, (p.pp_off, p.pp_idx, p.pc_off, p.pc_idx), ("pp_off", "pp_idx", "pc_off", "pc_idx")):
            assert a.dtype == b.dtype and np.array_equal(a, b), (p.name, name)
            assert np.array_equal(c, b), (p.name, name, "generator")
        # group-shared lists
        gc, gf, gn = inputs.build_groups(p)
        want = flat(oracle.walk_lists(p.tree, p.cells, gc, theta, p.eps))
        got = _device_lists(ctx, torch, p, gc, theta, p.eps)
        for a, b in zip(got, want):
            assert np.array_equal(a, b), p.name
        # leaf-form entries: one bucket reference per leaf
        rank = (np.cumsum(p.tree["isleaf"] != 0) - 1).astype(np.int32)
        want = flat(oracle.walk_lists(p.tree, p.cells, p.tree["leaf_cell"], theta, p.eps, leaf_rank=rank))
        got = _device_lists(ctx, torch, p, p.tree["leaf_cell"], theta, p.eps, flags=binding.PP_LEAVES)
        for a, b in zip(got, want):
            assert np.array_equal(a, b), (p.name, "leaf references")
    # empty sink set and bad arguments
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    p = cfg1
    z = _device_lists(ctx, torch, p, np.zeros(0, np.int32), 0.7, p.eps)
    assert list(z[0]) == [0] and list(z[2]) == [0] and z[1].size == 0
    with pytest.raises(binding.PkdgError):
        _device_lists(ctx, torch, p, p.tree["leaf_cell"], -1.0, p.eps)


def test_two_contexts_on_two_devices_in_one_process(torch, cfg1):
    """Function attributes (the dynamic shared-memory opt-in of the evaluation kernels) are per device and are set
    per context; the static workspace of pkdg_gravity_eval_static exists once per device.  Two devices in one process
    must therefore both work and agree bit for bit.  Skipped where only one GPU is visible."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    from paper_1609_08621_b200 import binding
    from gpu_util import to_dev
    p = cfg1
    outs = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            d = to_dev(p, torch, f"cuda:{dev}")
            c = binding.Context(dev)
            out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device=f"cuda:{dev}")
            c.gravity_eval(d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"], d["pc_off"], d["pc_idx"],
                           p.eps, out)
            st_out = torch.full((p.n, 4), float("nan"), dtype=torch.float32, device=f"cuda:{dev}")
            binding.gravity_eval_static(dev, d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"],
                                        d["pc_off"], d["pc_idx"], p.eps, st_out)
            torch.cuda.synchronize(dev)
            assert c.get_stats()["bad_entries"] == 0
            outs.append((out.cpu().numpy(), st_out.cpu().numpy()))
            c.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][0], outs[0][1]) and np.array_equal(outs[1][0], outs[1][1])


def test_device_walk_survives_malformed_trees(ctx, torch, cfg1):
    """A subtree end that does not advance and a sink that is no cell of the tree neither hang the walk nor send it
    out of bounds: the walk finishes, the sink gets empty lists, and pkdg_get_stats counts both as bad entries."""
    import copy
    p = cfg1
    lc = p.tree["leaf_cell"].astype(np.int32)
    want = _device_lists(ctx, torch, p, lc, p.theta, p.eps)
    assert ctx.get_stats()["bad_entries"] == 0
    # sinks outside [0, n_cells)
    sc = lc.copy(); sc[5] = p.cells.shape[0]; sc[9] = -3
    got = _device_lists(ctx, torch, p, sc, p.theta, p.eps)
    assert ctx.get_stats(check=False)["bad_entries"] == 2
    lp, lq = np.diff(got[0]), np.diff(want[0])
    assert lp[5] == 0 and lp[9] == 0 and np.diff(got[2])[5] == 0 and np.diff(got[2])[9] == 0
    keep = np.ones(len(lc), bool); keep[[5, 9]] = False
    assert np.array_equal(lp[keep], lq[keep])
    # end[k] <= k (would never advance) and end[k] > n_cells (would leave the array)
    q = copy.copy(p); q.tree = dict(p.tree); e = p.tree["end"].copy()
    k_self = int(np.flatnonzero(p.tree["isleaf"] != 0)[3]); e[k_self] = k_self
    k_far = int(np.flatnonzero(p.tree["isleaf"] != 0)[-1]); e[k_far] = p.cells.shape[0] + 1000
    q.tree["end"] = e
    got = _device_lists(ctx, torch, q, lc, p.theta, p.eps)      # returns: no hang; leaves' ends clamp to k + 1 / n_cells
    assert ctx.get_stats(check=False)["bad_entries"] == 2
    for a, b in zip(got, want):                                  # for a leaf, k + 1 (or n_cells for the last one) is the true end
        assert np.array_equal(a, b)


def test_tree_host_call_builds_lists_and_evaluates(ctx, torch, cfg1):
    """pkdg_gravity_eval_tree_host: every buffer on the host, lists built on the device.  Same bits as the resident
    call on the host generator's leaf-form lists (the device walk is bit-identical and ranges do not change a
    bucket's sums), the oracle's result within the tolerance, counters of the whole call, 1 / 3 / 4 ranges; rows in
    no bucket keep the caller's values; bad arguments fail loudly."""
    from paper_1609_08621_b200 import binding, inputs
    from gpu_util import rel_errors, run_resident
    for p in (cfg1, inputs.config2(n=1 << 15), inputs.config3(32)):
        q = _leaf_problem(p)
        base = run_resident(ctx, q, torch, flags=binding.PP_LEAVES)
        ref = _oracle(p)
        tr = p.tree
        tree = {k: np.ascontiguousarray(tr[k]) for k in ("first", "count", "end", "isleaf", "bblo", "bbhi")}
        cell_of = np.ascontiguousarray(tr["leaf_cell"].astype(np.int32))
        for n_ranges in (1, 3, 4):
            out = np.full((p.n, 4), np.nan, np.float32)
            ctx.gravity_eval_tree_host(p.xyzm, p.cells, tree, p.first, p.count, cell_of, p.theta, p.eps, out, n_ranges=n_ranges)
            st = ctx.get_stats()
            assert np.array_equal(out, base), (p.name, n_ranges)
            assert st["interactions_pp"] == p.I_pp and st["interactions_pc"] == p.I_pc and st["bad_entries"] == 0
            assert st["chunks"] == n_ranges and st["n_buckets"] == p.n_buckets
        ea, ep = rel_errors(out, ref)
        assert ea.max() <= TOL and ep.max() <= TOL, (p.name, ea.max(), ep.max())
    # a subset of the leaves is refused (the walk names P-P source leaves by bucket index: every leaf must be a
    # bucket), and so is a bucket that is not the particle run of the leaf cell it names; nothing is written
    p = cfg1
    tr = p.tree
    tree = {k: np.ascontiguousarray(tr[k]) for k in ("first", "count", "end", "isleaf", "bblo", "bbhi")}
    out = np.full((p.n, 4), np.nan, np.float32)
    for b0, b1 in ((100, 300), (0, p.n_buckets - 1), (1, p.n_buckets)):
        with pytest.raises(binding.PkdgError, match="ALL leaves"):
            ctx.gravity_eval_tree_host(p.xyzm, p.cells, tree, np.ascontiguousarray(p.first[b0:b1]), np.ascontiguousarray(p.count[b0:b1]),
                                       np.ascontiguousarray(tr["leaf_cell"][b0:b1].astype(np.int32)), p.theta, p.eps, out, n_ranges=2)
    wrong = np.ascontiguousarray(tr["leaf_cell"].astype(np.int32)); wrong[7] = 0   # the root is not a leaf
    with pytest.raises(binding.PkdgError, match="leaf cell"):
        ctx.gravity_eval_tree_host(p.xyzm, p.cells, tree, p.first, p.count, wrong, p.theta, p.eps, out)
    assert np.isnan(out).all()
    with pytest.raises(binding.PkdgError):      # buckets out of order
        ctx.gravity_eval_tree_host(p.xyzm, p.cells, tree, np.ascontiguousarray(p.first[::-1]), np.ascontiguousarray(p.count[::-1]),
                                   np.ascontiguousarray(tr["leaf_cell"][::-1].astype(np.int32)), p.theta, p.eps, out)
    with pytest.raises(binding.PkdgError):
        ctx.gravity_eval_tree_host(p.xyzm, p.cells, tree, p.first, p.count, np.ascontiguousarray(tr["leaf_cell"].astype(np.int32)),
                                   p.theta, p.eps, out, n_ranges=0)
