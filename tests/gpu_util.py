"""Helpers shared by the -m gpu tests: run a Problem through the C ABI and compare with the oracle."""
import numpy as np


def to_dev(p, torch, dev="cuda:0"):
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    return dict(xyzm=t(p.xyzm), cells=t(p.cells) if p.cells is not None and p.cells.shape[0] else None,
                first=t(p.first), count=t(p.count), pp_off=t(p.pp_off), pp_idx=t(p.pp_idx),
                pc_off=t(p.pc_off) if p.cells is not None and p.cells.shape[0] else None,
                pc_idx=t(p.pc_idx) if p.cells is not None and p.cells.shape[0] else None)


def run_resident(ctx, p, torch, flags=0, fill=float("nan")):
    d = to_dev(p, torch)
    out = torch.full((p.n, 4), fill, dtype=torch.float32, device="cuda:0")
    ctx.gravity_eval(d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"], d["pc_off"],
                     d["pc_idx"], p.eps, out, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def rel_errors(gpu, ref, rows=None):
    """Per-particle |a_gpu - a_or| / |a_or| (vector norms) and |phi_gpu - phi_or| / |phi_or| (A17)."""
    if rows is not None:
        gpu = gpu[rows]; ref = ref[rows]
    ea = np.linalg.norm(gpu[:, :3].astype(np.float64) - ref[:, :3], axis=1) / np.linalg.norm(ref[:, :3], axis=1)
    ep = np.abs(gpu[:, 3].astype(np.float64) - ref[:, 3]) / np.abs(ref[:, 3])
    return ea, ep


def bucket_rows(p, sel):
    rows = np.concatenate([np.arange(p.first[b], p.first[b] + p.count[b]) for b in sel]) if len(sel) else np.zeros(0, np.int64)
    return rows.astype(np.int64)
