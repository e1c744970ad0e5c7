#!/usr/bin/env python
"""bench.py -- headline measurement of pkdg-b200 (contract: the task's "Measurement" section).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--ng 256]

One "step" = one pass of the whole hot path (cell prep + packer + fused P-P/P-C evaluation +
reduction/write-back: SURVEY.md sec 8(a)) over one synthetic problem.  Workload at every N:
BASELINE.json configs[2], the configuration the metric is quoted on (N = 2^24 particles, 256^3
lattice displaced by a Zel'dovich field, binary tree, bucket 16, theta = 0.7); it fits one GPU.
With --gpus N > 1 (torchrun) ONE problem is strong-scaled: rank 0's arrays are broadcast over NCCL, every rank
evaluates the cost-balanced bucket range paper_1609_08621_b200/shard.py gives it, no data-path collective
(DESIGN.md "Multi-GPU"); --scaling weak runs N independent replicas instead.

Prints ONE JSON line on rank 0.  `--impl reference` times the fp64 CPU oracle (oracle/) on the host
cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# Flops per interaction AS EXECUTED by the kernels (add/sub/mul = 1, FMA = 2, rsqrt = 1); derived
# line by line in DESIGN.md "Flop audit".  The paper's own convention (Table 3: 53 / 215, rsqrt = 7)
# is reported beside it as context only.
F_PP = 19
F_PC = 167
PAPER_F_PP, PAPER_F_PC = 53, 215
# C-C / C-P path (pkdg_fmm.cuh, formulas as executed): per C-C entry, per C-P entry, per sink evaluated, per bucket
F_CC, F_CP, F_LOC_SINK, F_LOC_BUCKET = 815, 372, 488, 1488
PAPER_F_CC, PAPER_F_CP = 479, 213       # PAPER.md Table 3 (L216-217), context only
SM_COUNT_NOMINAL, FP32_LANES_PER_SM = 148, 128


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples SM clock and clock-event reasons with NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, torch, dev):
        self.samples, self.reasons, self.max_mhz, self.power = [], set(), None, []
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode() if hasattr(uuid, "encode") else uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(dev)
            self.nv = pynvml
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # no NVML: report that instead of inventing numbers
            self.nv = None
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        if not self.nv:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "err", "no nvml")}
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": round(max(self.power), 1) if self.power else None}


def build_workload(ng: int):
    from paper_1609_08621_b200 import inputs
    t = time.time()
    p = inputs.config3(ng)
    return p, time.time() - t


def workload_config(p, ng):
    list_gb = (p.pp_idx.nbytes + p.pc_idx.nbytes + p.pp_off.nbytes + p.pc_off.nbytes) / 1e9
    return {"workload": f"configs[2]: N={ng}^3={p.n} Zel'dovich lattice (P(k)~k^-2, rms 0.3 cells), binary tree, "
                        f"bucket<=16, theta=0.7, order-4 multipoles, eps=1/(50*{ng})",
            "n_particles": p.n, "n_buckets": p.n_buckets, "n_cells": int(p.cells.shape[0]),
            "mean_bucket_occupancy": round(float(p.count.mean()), 3),
            "mean_L_pp": round(float(np.diff(p.pp_off).mean()), 2), "mean_L_pc": round(float(np.diff(p.pc_off).mean()), 2),
            "I_pp": p.I_pp, "I_pc": p.I_pc, "theta": 0.7, "eps": p.eps,
            "l2_policy": f"inputs larger than L2: lists {list_gb:.2f} GB + particles/cells "
                         f"{(p.xyzm.nbytes + p.cells.nbytes) / 1e9:.2f} GB are re-read every step (L2 = 126 MB)"}


def oracle_sample(p, target_s: float, seed: int = 0):
    """Time the oracle, as it stands, on an evenly spread sample of buckets sized for ~target_s."""
    import oracle
    nb = p.n_buckets
    n_probe = min(nb, 2048)   # large enough that thread start-up does not dominate the estimate
    probe = np.unique(np.linspace(0, nb - 1, n_probe).astype(np.int64))
    oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, sel=probe)
    t = time.perf_counter()   # second pass: threads and caches are warm
    oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, sel=probe)
    dt = max(time.perf_counter() - t, 1e-4)
    n = int(min(nb, max(64, len(probe) * target_s / dt)))
    sel = np.unique(np.linspace(0, nb - 1, n).astype(np.int64))
    inter = int(np.dot(p.count[sel].astype(np.int64), np.diff(p.pp_off)[sel] + np.diff(p.pc_off)[sel]))
    t = time.perf_counter()
    oracle.gravity_eval(p.xyzm, p.cells, p.first, p.count, p.pp_off, p.pp_idx, p.pc_off, p.pc_idx, p.eps, sel=sel)
    dt = time.perf_counter() - t
    return inter / dt, dt, len(sel), inter, oracle.num_threads()


def parallelism_string(world, scaling):
    """What `config.parallelism` says; the same text in both arms (the arms are compared on `config`)."""
    if world == 1:
        return "1 GPU"
    if scaling == "weak":
        return f"{world} independent replicas"
    return (f"{world} ranks, contiguous cost-balanced bucket ranges (shard.rank_piece), arrays replicated by one NCCL "
            f"broadcast, no data-path collective")


def run_reference(args, rank, world):
    if rank != 0:
        return
    p, gen_s = build_workload(args.ng)
    per_step = min(10.0, 150.0 / (args.steps + args.warmup))
    for _ in range(args.warmup):
        oracle_sample(p, per_step)
    tot_i, tot_t, nb_s, cores = 0, 0.0, 0, 1
    for _ in range(args.steps):
        rate, dt, nsel, inter, cores = oracle_sample(p, per_step)
        tot_i += inter; tot_t += dt; nb_s = nsel
    value = tot_i / tot_t
    sample = f"{nb_s} of {p.n_buckets} buckets (evenly spread in tree order) per step, ~{per_step:.1f} s of CPU work each"
    line = {"impl": "reference", "metric": "P-P+P-C interactions/s", "value": value, "unit": "interactions/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(workload_config(p, args.ng), parallelism=parallelism_string(world, args.scaling)),
            "cpu_baseline": {"value": value, "unit": "interactions/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def kernel_source_hash():
    """sha256 (first 16 hex digits) of the CUDA sources the evaluation kernel is built from, comments and white space
    removed: the key profiles/traffic.json is stamped with, so that a measured DRAM-traffic figure is dropped (null)
    as soon as the code it was measured on has changed."""
    import hashlib
    import re
    h = hashlib.sha256()
    for rel in ("paper_1609_08621_b200/csrc/pkdg_kernels.cuh", "paper_1609_08621_b200/csrc/pkdg.cu", "include/pkdg.h"):
        with open(os.path.join(ROOT, rel), "r") as f:
            text = f.read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        text = re.sub(r"//[^\n]*", "", text)
        h.update(re.sub(r"\s+", "", text).encode())
    return h.hexdigest()[:16]


def measured_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the evaluation kernel from the last ncu --set full
    capture (profiles/traffic.json), or None if that capture was taken on other kernel sources."""
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(tpath):
        return None, "no capture"
    with open(tpath) as f:
        t = json.load(f)
    if t.get("source_hash") != kernel_source_hash():
        return None, f"stale: captured on sources {t.get('source_hash')}, running {kernel_source_hash()}"
    return t.get(key), f"ncu capture {t.get('capture', '?')}"


def _leaf_lists(p):
    """The P-P lists of problem p with bucket references as entries (what the host generator gives with leaf form)."""
    from paper_1609_08621_b200 import inputs
    return inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)


def _max_over_ranks(x, dist, torch, dev):
    if dist is None:
        return x
    tt = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def _sum_over_ranks(x, dist, torch, dev):
    if dist is None:
        return x
    tt = torch.tensor([x], dtype=torch.int64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.SUM)
    return int(tt.item())


def run_ours(args, rank, world, local_rank):
    """One problem (config 3) on `world` GPUs.  world > 1, default --scaling strong: rank 0 builds the problem,
    multigpu.distribute broadcasts the read-only arrays over NCCL and every rank evaluates the bucket range
    shard.rank_piece gives it through pkdg_gravity_eval_range -- no collective on the data path; value =
    all interactions / max-over-ranks time.  --scaling weak: every rank evaluates its own full replica."""
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_1609_08621_b200 import binding, multigpu
    peaks, peak_kind = load_peaks()
    dev = torch.device("cuda", local_rank)
    strong = world > 1 and args.scaling != "weak"

    p, gen_s = (None, 0.0)
    if rank == 0 or not strong:
        p, gen_s = build_workload(args.ng)
    if strong:
        g, piece = multigpu.distribute(p, dist, rank, world, dev, torch)
    else:
        g, piece = multigpu.distribute(p, None, 0, 1, dev, torch)
    cfg = workload_config(p, args.ng) if p is not None else None
    n_particles = int(g.xyzm.shape[0])
    cnt_piece = piece.count.astype(np.int64)
    I_pp = int(np.dot(cnt_piece, np.diff(piece.pp_off))); I_pc = int(np.dot(cnt_piece, np.diff(piece.pc_off)))
    tot_pp = _sum_over_ranks(I_pp, dist if strong else None, torch, dev)
    tot_pc = _sum_over_ranks(I_pc, dist if strong else None, torch, dev)
    out = torch.zeros((n_particles, 4), dtype=torch.float32, device=dev)
    ctx = binding.Context(local_rank)
    flags = args.flags

    def step(fl=flags):
        ctx.gravity_eval_range(g.xyzm, g.cells, g.first, g.count, piece.b0, piece.b1, piece.d_pp_off, piece.pp_idx,
                               piece.d_pc_off, piece.pc_idx, g.eps, out, flags=fl)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, k):
        """K calls of fn between barriers, CUDA events on the launching stream; ms per call, max over ranks."""
        barrier()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(k):
            fn()
        e1.record()
        barrier()
        return _max_over_ranks(e0.elapsed_time(e1) / k, dist, torch, dev)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        step()
    barrier()
    ctx.profile_read()
    ctx.profile_enable(True)
    sampler = ClockSampler(torch, local_rank)
    launches0 = ctx.launch_count()
    sampler.start()
    ms_step = timed(step, args.steps)
    clocks = sampler.stop()
    sampler_x = ClockSampler(torch, local_rank)   # the extra keys below are timed too: their own clock record
    sampler_x.start()
    n_eval, eval_ms_total, fix_ms_total = ctx.profile_read()
    ctx.profile_enable(False)
    launches = (ctx.launch_count() - launches0) // args.steps
    stats = ctx.get_stats()
    assert stats["interactions_pp"] == I_pp and stats["interactions_pc"] == I_pc and stats["bad_entries"] == 0
    if not strong:
        tot_pp, tot_pc = world * I_pp, world * I_pc
    inter = tot_pp + tot_pc
    value = inter / (ms_step * 1e-3)
    flops = F_PP * tot_pp + F_PC * tot_pc
    fix_sinks = _sum_over_ranks(stats["fixup_sinks"], dist, torch, dev)
    # the cost of the conditioning-triggered fp64 fix-up: the same step without it
    ms_nofix = timed(lambda: step(flags | binding.NO_FIXUP), max(3, args.steps // 2))
    fixup = {"sinks": fix_sinks, "frac_of_sinks": fix_sinks / (n_particles * (1 if strong else world)),
             "kernel_ms": fix_ms_total / max(n_eval, 1), "step_ms_without_fixup_and_estimate": ms_nofix,
             "added_ms": ms_step - ms_nofix}
    shares = None
    if strong:
        sh = torch.zeros(world, dtype=torch.float64, device=dev)
        sh[rank] = piece.cost / max(piece.cost_total, 1)
        dist.all_reduce(sh)
        shares = [round(float(x), 4) for x in sh.tolist()]

    # ---- end to end: every buffer starts in pinned host memory, result read back every step
    e2e = None
    pin = lambda t_: t_.cpu().pin_memory()
    if not args.no_e2e:
        h = dict(xyzm=pin(g.xyzm), cells=pin(g.cells), first=pin(g.first), count=pin(g.count),
                 pp_off=torch.from_numpy(piece.pp_off).pin_memory(), pp_idx=pin(piece.pp_idx),
                 pc_off=torch.from_numpy(piece.pc_off).pin_memory(), pc_idx=pin(piece.pc_idx))
        out_h = torch.zeros((n_particles, 4), dtype=torch.float32).pin_memory()

        def e2e_step():
            ctx.gravity_eval_host_range(h["xyzm"], h["cells"], h["first"], h["count"], piece.b0, piece.b1, h["pp_off"],
                                        h["pp_idx"], h["pc_off"], h["pc_idx"], g.eps, out_h, n_streams=args.e2e_streams,
                                        max_entries_per_chunk=args.e2e_chunk, flags=flags)
        for _ in range(2):
            e2e_step()
        barrier()
        k2 = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k2):
            e2e_step()
        torch.cuda.synchronize()
        dt = _max_over_ranks((time.perf_counter() - t0) / k2, dist, torch, dev)
        rows = int(cnt_piece.sum())
        h2d = sum(int(v.numel() * v.element_size()) for v in h.values())
        e2e = {"value": inter / dt, "unit": "interactions/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": rows * 16, "ms_per_step": dt * 1e3, "steps": k2,
               "api": "pkdg_gravity_eval_host_range (pinned host buffers, lists streamed in chunks; bytes are this rank's)",
               "n_streams": args.e2e_streams, "max_entries_per_chunk": args.e2e_chunk}
        del h, out_h

    # ---- the same workload with the P-P lists in leaf form (PKDG_PP_LEAVES): extra key, N = 1
    leaves = None
    if not args.no_leaves and world == 1:
        from paper_1609_08621_b200 import inputs as _inputs
        lo, li = _inputs.pp_leaves(p.n, p.first, p.count, p.pp_off, p.pp_idx)
        lflags = flags | binding.PP_LEAVES
        d_lo, d_li = torch.from_numpy(lo).to(dev), torch.from_numpy(li).to(dev)

        def lstep():
            ctx.gravity_eval(g.xyzm, g.cells, g.first, g.count, d_lo, d_li, g.pc_off, g.pc_idx, g.eps, out, flags=lflags)
        for _ in range(3):
            lstep()
        barrier()
        ctx.profile_read(); ctx.profile_enable(True)
        lms = timed(lstep, args.steps)
        ln, lk, _ = ctx.profile_read(); ctx.profile_enable(False)
        lst = ctx.get_stats()
        assert lst["interactions_pp"] == p.I_pp and lst["interactions_pc"] == p.I_pc and lst["bad_entries"] == 0
        leaves = {"value": inter / (lms * 1e-3), "unit": "interactions/s", "ms_per_step": lms,
                  "kernel_ms": lk / max(ln, 1), "pp_list_entries": int(li.shape[0]), "frac_fp32_fma_peak_kernel": None}
        if not args.no_e2e:
            h = dict(xyzm=pin(g.xyzm), cells=pin(g.cells), first=pin(g.first), count=pin(g.count),
                     pp_off=torch.from_numpy(lo).pin_memory(), pp_idx=torch.from_numpy(li).pin_memory(),
                     pc_off=pin(g.pc_off), pc_idx=pin(g.pc_idx))
            out_h = torch.zeros((p.n, 4), dtype=torch.float32).pin_memory()

            def le2e():
                ctx.gravity_eval_host(h["xyzm"], h["cells"], h["first"], h["count"], h["pp_off"], h["pp_idx"],
                                      h["pc_off"], h["pc_idx"], g.eps, out_h, n_streams=args.e2e_streams,
                                      max_entries_per_chunk=args.e2e_chunk, flags=lflags)
            for _ in range(2):
                le2e()
            barrier()
            k2 = max(2, min(args.steps, 5))
            t0 = time.perf_counter()
            for _ in range(k2):
                le2e()
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / k2
            leaves["e2e"] = {"value": inter / dt, "unit": "interactions/s", "ms_per_step": dt * 1e3,
                             "h2d_bytes_per_step": sum(int(v.numel() * v.element_size()) for v in h.values()),
                             "d2h_bytes_per_step": int(out_h.numel() * 4)}
            del h, out_h
        del d_lo, d_li

    # ---- group-shared lists (g = 64) with leaf-form P-P entries: extra key, N = 1
    groups = None
    if not args.no_groups and world == 1:
        from paper_1609_08621_b200 import inputs as _inputs
        t0 = time.perf_counter()
        gc_, gf, gn = _inputs.build_groups(p, 64)
        gppo, gppi, gpco, gpci = _inputs.build_group_lists(p, gc_, p.theta, p.eps)
        glo, gli = _inputs.pp_leaves(p.n, p.first, p.count, gppo, gppi)
        g_gen = time.perf_counter() - t0
        gI_pp = int(np.dot(np.add.reduceat(p.count.astype(np.int64), gf), np.diff(gppo)))
        gI_pc = int(np.dot(np.add.reduceat(p.count.astype(np.int64), gf), np.diff(gpco)))
        gflags = flags | binding.PP_LEAVES
        T = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        dg = dict(gf=T(gf), gn=T(gn), lo=T(glo), li=T(gli), co=T(gpco), ci=T(gpci))

        def gstep():
            ctx.gravity_eval_groups(g.xyzm, g.cells, g.first, g.count, dg["gf"], dg["gn"], dg["lo"], dg["li"], dg["co"],
                                    dg["ci"], g.eps, out, flags=gflags)
        for _ in range(3):
            gstep()
        barrier()
        ctx.profile_read(); ctx.profile_enable(True)
        gms = timed(gstep, args.steps)
        gn_, gk, gfx = ctx.profile_read(); ctx.profile_enable(False)
        gst = ctx.get_stats()
        assert gst["interactions_pp"] == gI_pp and gst["interactions_pc"] == gI_pc and gst["bad_entries"] == 0
        ginter = gI_pp + gI_pc
        groups = {"n_groups": int(gf.shape[0]), "mean_buckets_per_group": float(gn.mean()),
                  "mean_L_pp_particles": gI_pp / p.n, "mean_L_pc": gI_pc / p.n, "I_pp": gI_pp, "I_pc": gI_pc,
                  "list_entries": int(gli.shape[0] + gpci.shape[0]),
                  "list_entries_per_bucket_lists": int(p.pp_idx.shape[0] + p.pc_idx.shape[0]),
                  "value": ginter / (gms * 1e-3), "unit": "interactions/s", "ms_per_step": gms, "kernel_ms": gk / max(gn_, 1),
                  "fixup_sinks": gst["fixup_sinks"], "host_list_build_s": round(g_gen, 1),
                  "frac_fp32_fma_peak_kernel": None,
                  "note": "one P-P (bucket references) and one P-C list per group of <= 64 particles; every sink of the group "
                          "evaluates the whole list, so there are more interactions per sink than with per-bucket lists"}
        if not args.no_e2e:
            P_ = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
            h = dict(xyzm=pin(g.xyzm), cells=pin(g.cells), first=pin(g.first), count=pin(g.count), gf=P_(gf), gn=P_(gn),
                     lo=P_(glo), li=P_(gli), co=P_(gpco), ci=P_(gpci))
            out_h = torch.zeros((p.n, 4), dtype=torch.float32).pin_memory()

            def ge2e():
                ctx.gravity_eval_host_groups(h["xyzm"], h["cells"], h["first"], h["count"], h["gf"], h["gn"], h["lo"], h["li"],
                                             h["co"], h["ci"], g.eps, out_h, n_streams=args.e2e_streams,
                                             max_entries_per_chunk=max(1, args.e2e_chunk // 8), flags=gflags)
            for _ in range(2):
                ge2e()
            barrier()
            k2 = max(2, min(args.steps, 5))
            t0 = time.perf_counter()
            for _ in range(k2):
                ge2e()
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) / k2
            groups["e2e"] = {"value": ginter / dt, "unit": "interactions/s", "ms_per_step": dt * 1e3,
                             "sinks_per_s": p.n / dt,
                             "h2d_bytes_per_step": sum(int(v.numel() * v.element_size()) for v in h.values()),
                             "d2h_bytes_per_step": int(out_h.numel() * 4)}
            del h, out_h
        del dg

    # ---- list construction on the device: walk time, and the end-to-end time it gives when
    #      particles, cells and the tree (not the lists) cross PCIe.  Extra key, N = 1.
    devlists = None
    if not args.no_device_lists and world == 1:
        tr = p.tree
        T = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        tree_h = {k: torch.from_numpy(np.ascontiguousarray(tr[k])).pin_memory() for k in ("first", "count", "end", "isleaf", "bblo", "bbhi")}
        sink_h = torch.from_numpy(np.ascontiguousarray(tr["leaf_cell"].astype(np.int32))).pin_memory()
        xy_h, ce_h = pin(g.xyzm), pin(g.cells)
        fb_h, cb_h = pin(g.first), pin(g.count)
        out_h = torch.zeros((p.n, 4), dtype=torch.float32).pin_memory()
        nb_ = p.n_buckets
        d_ppo = torch.empty(nb_ + 1, dtype=torch.int64, device=dev); d_pco = torch.empty(nb_ + 1, dtype=torch.int64, device=dev)
        d_ppi = torch.empty(p.pp_idx.shape[0], dtype=torch.int32, device=dev)
        d_pci = torch.empty(p.pc_idx.shape[0], dtype=torch.int32, device=dev)
        tree_d = {k: v.to(dev) for k, v in tree_h.items()}
        sink_d = sink_h.to(dev)

        def walk():
            npp, npc = ctx.build_lists_count(tree_d, g.cells, sink_d, p.theta, p.eps, d_ppo, d_pco)
            assert npp == p.pp_idx.shape[0] and npc == p.pc_idx.shape[0]
            ctx.build_lists_fill(tree_d, g.cells, sink_d, p.theta, p.eps, d_ppo, d_pco, d_ppi, d_pci)
        for _ in range(2):
            walk()
        walk_ms = timed(walk, max(3, args.steps // 2))
        same = bool(torch.equal(d_ppi, g.pp_idx) and torch.equal(d_pci, g.pc_idx) and torch.equal(d_ppo, g.pp_off))

        def dl_e2e():
            x = xy_h.to(dev, non_blocking=True); c = ce_h.to(dev, non_blocking=True)
            td = {k: v.to(dev, non_blocking=True) for k, v in tree_h.items()}
            sk = sink_h.to(dev, non_blocking=True); fb = fb_h.to(dev, non_blocking=True); cb = cb_h.to(dev, non_blocking=True)
            ctx.build_lists_count(td, c, sk, p.theta, p.eps, d_ppo, d_pco)
            ctx.build_lists_fill(td, c, sk, p.theta, p.eps, d_ppo, d_pco, d_ppi, d_pci)
            ctx.gravity_eval(x, c, fb, cb, d_ppo, d_ppi, d_pco, d_pci, g.eps, out, flags=flags)
            out_h.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        for _ in range(2):
            dl_e2e()
        k2 = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(k2):
            dl_e2e()
        dt = (time.perf_counter() - t0) / k2
        h2d = sum(int(v.numel() * v.element_size()) for v in list(tree_h.values()) + [sink_h, xy_h, ce_h, fb_h, cb_h])
        # the same with P-P entries as bucket references (PKDG_PP_LEAVES): 16 x fewer P-P entries to write and to read
        leaf_rank = (np.cumsum(tr["isleaf"] != 0) - 1).astype(np.int32)
        lr_h = torch.from_numpy(leaf_rank).pin_memory()
        tree_d["leaf_rank"] = lr_h.to(dev)
        lo_h, li_h = _leaf_lists(p)
        d_lli = torch.empty(li_h.shape[0], dtype=torch.int32, device=dev)
        lfl = flags | binding.PP_LEAVES

        def walk_leaf():
            npp, npc = ctx.build_lists_count(tree_d, g.cells, sink_d, p.theta, p.eps, d_ppo, d_pco, flags=binding.PP_LEAVES)
            assert npp == li_h.shape[0] and npc == p.pc_idx.shape[0]
            ctx.build_lists_fill(tree_d, g.cells, sink_d, p.theta, p.eps, d_ppo, d_pco, d_lli, d_pci, flags=binding.PP_LEAVES)
        for _ in range(2):
            walk_leaf()
        walk_leaf_ms = timed(walk_leaf, max(3, args.steps // 2))
        same_leaf = bool(torch.equal(d_lli.cpu(), torch.from_numpy(li_h)) and torch.equal(d_ppo.cpu(), torch.from_numpy(lo_h))
                         and torch.equal(d_pci, g.pc_idx))

        def dl_e2e_leaf():
            x = xy_h.to(dev, non_blocking=True); c = ce_h.to(dev, non_blocking=True)
            td = {k: v.to(dev, non_blocking=True) for k, v in tree_h.items()}
            td["leaf_rank"] = lr_h.to(dev, non_blocking=True)
            sk = sink_h.to(dev, non_blocking=True); fb = fb_h.to(dev, non_blocking=True); cb = cb_h.to(dev, non_blocking=True)
            ctx.build_lists_count(td, c, sk, p.theta, p.eps, d_ppo, d_pco, flags=binding.PP_LEAVES)
            ctx.build_lists_fill(td, c, sk, p.theta, p.eps, d_ppo, d_pco, d_lli, d_pci, flags=binding.PP_LEAVES)
            ctx.gravity_eval(x, c, fb, cb, d_ppo, d_lli, d_pco, d_pci, g.eps, out, flags=lfl)
            out_h.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        for _ in range(2):
            dl_e2e_leaf()
        t0 = time.perf_counter()
        for _ in range(k2):
            dl_e2e_leaf()
        dt_leaf = (time.perf_counter() - t0) / k2
        lst = ctx.get_stats()
        assert lst["interactions_pp"] == p.I_pp and lst["interactions_pc"] == p.I_pc and lst["bad_entries"] == 0

        # the same again with the copies overlapped: tree and cells first, the walk starts while the particles are
        # still crossing the bus; the evaluation runs in four bucket ranges (pkdg_gravity_eval_range) and the rows of a
        # range go back while the next range is evaluated.
        s1, s2 = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        n_rng = 4
        rb = [int(v) for v in np.linspace(0, p.n_buckets, n_rng + 1)]
        row_of = lambda b: int(p.first[b]) if b < p.n_buckets else int(p.first[-1] + p.count[-1])

        def dl_e2e_overlapped():
            with torch.cuda.stream(s1):
                c = ce_h.to(dev, non_blocking=True)
                td = {k: v.to(dev, non_blocking=True) for k, v in tree_h.items()}
                td["leaf_rank"] = lr_h.to(dev, non_blocking=True)
                sk = sink_h.to(dev, non_blocking=True); fb = fb_h.to(dev, non_blocking=True); cb = cb_h.to(dev, non_blocking=True)
            with torch.cuda.stream(s2):
                x = xy_h.to(dev, non_blocking=True)
                ev_x = s2.record_event()
            with torch.cuda.stream(s1):
                ctx.build_lists_count(td, c, sk, p.theta, p.eps, d_ppo, d_pco, flags=binding.PP_LEAVES, stream=s1)
                ctx.build_lists_fill(td, c, sk, p.theta, p.eps, d_ppo, d_pco, d_lli, d_pci, flags=binding.PP_LEAVES, stream=s1)
                s1.wait_event(ev_x)
                for r in range(n_rng):
                    b0, b1 = rb[r], rb[r + 1]
                    ctx.gravity_eval_range(x, c, fb, cb, b0, b1, d_ppo[b0:b1 + 1], d_lli, d_pco[b0:b1 + 1], d_pci, g.eps, out,
                                           flags=lfl, stream=s1)
                    ev = s1.record_event()
                    with torch.cuda.stream(s2):
                        s2.wait_event(ev)
                        r0, r1 = row_of(b0), row_of(b1)
                        out_h[r0:r1].copy_(out[r0:r1], non_blocking=True)
            s1.synchronize(); s2.synchronize()
        ref_rows = out_h.clone()     # the result of the plain sequence above: ranges give the same bits
        out_h.zero_()
        for _ in range(2):
            dl_e2e_overlapped()
        same_rows = bool(torch.equal(out_h, ref_rows))
        t0 = time.perf_counter()
        for _ in range(k2):
            dl_e2e_overlapped()
        dt_ovl = (time.perf_counter() - t0) / k2
        # the same sequence as ONE call of the library: pkdg_gravity_eval_tree_host
        tree_np = {k: v for k, v in tree_h.items()}
        out_t = torch.zeros((p.n, 4), dtype=torch.float32).pin_memory()

        def tree_call():
            ctx.gravity_eval_tree_host(xy_h, ce_h, tree_np, fb_h, cb_h, sink_h, p.theta, p.eps, out_t, flags=flags, n_ranges=4)
        for _ in range(2):
            tree_call()
        same_tree = bool(torch.equal(out_t, ref_rows))
        tst = ctx.get_stats()
        assert tst["interactions_pp"] == p.I_pp and tst["interactions_pc"] == p.I_pc and tst["bad_entries"] == 0
        t0 = time.perf_counter()
        for _ in range(k2):
            tree_call()
        dt_tree = (time.perf_counter() - t0) / k2
        devlists = {"walk_ms": walk_ms, "bit_identical_to_host_generator": same,
                    "tree_host_call": {"api": "pkdg_gravity_eval_tree_host (host buffers in, device-built leaf-form lists, 4 ranges)",
                                       "ms_per_step": dt_tree * 1e3, "value": inter / dt_tree, "unit": "interactions/s",
                                       "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(out_t.numel() * 4),
                                       "rows_equal_to_plain_sequence": same_tree},
                    "leaf_form": {"walk_ms": walk_leaf_ms, "bit_identical_to_host_generator": same_leaf,
                                  "list_entries": int(li_h.shape[0] + p.pc_idx.shape[0]),
                                  "e2e_ms_per_step": dt_leaf * 1e3, "e2e_value": inter / dt_leaf,
                                  "e2e_overlapped_ms_per_step": dt_ovl * 1e3, "e2e_overlapped_value": inter / dt_ovl,
                                  "e2e_overlapped_rows_complete": same_rows,
                                  "e2e_overlapped_api": "H2D of tree and cells, walk while the particles arrive, four "
                                                        "pkdg_gravity_eval_range calls, rows of a range copied back under the next",
                                  "h2d_bytes_per_step": h2d + int(lr_h.numel() * 4)},
                    "list_entries": int(p.pp_idx.shape[0] + p.pc_idx.shape[0]),
                    "e2e": {"value": inter / dt, "unit": "interactions/s", "ms_per_step": dt * 1e3, "h2d_bytes_per_step": h2d,
                            "d2h_bytes_per_step": int(out_h.numel() * 4),
                            "api": "H2D of particles, cells, tree; pkdg_build_lists_count + _fill; pkdg_gravity_eval; D2H"}}
        del tree_d, sink_d, d_ppo, d_pco, d_ppi, d_pci, d_lli, out_h

    # ---- FMM form of the path: four lists per bucket, C-C / C-P through the 5th-order local
    #      expansion.  Extra key, N = 1: the whole call and the local-expansion kernel alone.
    fmm = None
    if not args.no_fmm and world == 1:
        from paper_1609_08621_b200 import inputs as _inputs
        t0 = time.perf_counter()
        F = _inputs.build_fmm_lists(p, p.theta, p.eps)
        f_gen = time.perf_counter() - t0
        T = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        df = {k: (T(F[k][0]), T(F[k][1])) for k in ("pp", "pc", "cp", "cc")}
        d_centre = T(F["centre"])
        cnt_all = p.count.astype(np.int64)
        fI_pp = int(np.dot(cnt_all, np.diff(F["pp"][0]))); fI_pc = int(np.dot(cnt_all, np.diff(F["pc"][0])))
        n_cc, n_cp = int(F["cc"][1].shape[0]), int(F["cp"][1].shape[0])

        def fstep(near=True):
            n_ = df if near else {"pp": (None, None), "pc": (None, None)}
            ctx.gravity_eval_fmm(g.xyzm, g.cells, g.first, g.count, d_centre, n_["pp"][0], n_["pp"][1], n_["pc"][0],
                                 n_["pc"][1], df["cp"][0], df["cp"][1], df["cc"][0], df["cc"][1], g.eps, out, flags=flags)
        for _ in range(3):
            fstep()
        fms = timed(fstep, args.steps)
        fst = ctx.get_stats()
        assert fst["interactions_cc"] == n_cc and fst["interactions_cp"] == n_cp and fst["bad_entries"] == 0
        assert fst["interactions_pp"] == fI_pp and fst["interactions_pc"] == fI_pc
        for _ in range(2):
            fstep(False)
        lms = timed(lambda: fstep(False), args.steps)
        fl_loc = F_CC * n_cc + F_CP * n_cp + F_LOC_SINK * p.n + F_LOC_BUCKET * p.n_buckets
        fmm = {"lists_per_bucket": {k: F[k][1].shape[0] / p.n_buckets for k in ("pp", "pc", "cp", "cc")},
               "I_pp": fI_pp, "I_pc": fI_pc, "I_cc": n_cc, "I_cp": n_cp, "ms_per_step": fms,
               "sinks_per_s": p.n / (fms * 1e-3), "local_expansion_kernel_ms": lms,
               "flops_as_executed": {"cc": F_CC, "cp": F_CP, "per_sink_evaluation": F_LOC_SINK, "per_bucket_reduction": F_LOC_BUCKET},
               "local_expansion_tflops": fl_loc / (lms * 1e-3) / 1e12, "frac_fp32_fma_peak_local_kernel": None,
               "paper_convention_tflops_local": (PAPER_F_CC * n_cc + PAPER_F_CP * n_cp) / (lms * 1e-3) / 1e12,
               "fixup_sinks": fst["fixup_sinks"], "host_list_build_s": round(f_gen, 1),
               "speedup_vs_per_sink_lists": ms_step / fms,
               "note": "same tree, same theta: C-C where |COM_B - COM_k| > 1.5 RO_B + RO_k (PAPER.md:L69), else the per-sink "
                       "criterion; every bucket keeps its own local expansion (no hierarchical sink side)"}
        del df, d_centre

    clocks_x = sampler_x.stop()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (pkdg_evalb_kernel, this rank's launch): plain FP32 ALU (FFMA pipe) bound
    sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
    peak_tflops = sms * FP32_LANES_PER_SM * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    eval_ms = eval_ms_total / max(n_eval, 1)
    flops_rank = F_PP * I_pp + F_PC * I_pc
    achieved = flops_rank / (eval_ms * 1e-3) / 1e12
    probe_ms, probe_flops = ctx.fma_peak_probe(1 << 15)
    traffic, traffic_note = measured_traffic(f"cfg3_ng{args.ng}") if world == 1 else (None, "single-GPU capture only")
    roofline = {"bound": "alu", "kernel": "pkdg_evalb_kernel", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": traffic, "traffic_note": traffic_note,
                "peak_kind": f"{sms} SMs x 128 FP32 lanes x 2 x sm_max_mhz ({peak_kind} MEASURED_PEAKS.json clock)",
                "kernel_ms": eval_ms, "kernel_share_of_step": eval_ms / ms_step,
                "ffma_probe_tflops": probe_flops / (probe_ms * 1e-3) / 1e12,
                "flops_per_interaction": {"pp": F_PP, "pc": F_PC},
                "hbm_algorithmic_gbs": (piece.pp_idx.numel() * 4 + piece.pc_idx.numel() * 4 + 32 * int(cnt_piece.sum())
                                        + 32 * piece.n_buckets) / (eval_ms * 1e-3) / 1e9,
                "hbm_peak_gbs": peaks.get("hbm_gbs")}

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        rate, dt, nsel, inter_s, cores = oracle_sample(p, args.cpu_seconds)
        cpu_baseline = {"value": rate, "unit": "interactions/s", "cores": cores, "kind": "oracle",
                        "sample": f"{nsel} of {p.n_buckets} buckets evenly spread in tree order "
                                  f"({inter_s} interactions, {dt:.1f} s)"}

    # ---- the other BASELINE.json configs that fit a default run (north_star: "uniform and clustered particle sets"):
    # config 2 and three config-4 shapes through the resident call, kernel time from the library's CUDA events, each
    # with its own clock record and a bounded oracle sample.  Not the headline: parity-test configs, measured.
    configs = None
    if world == 1 and not args.no_configs:
        from paper_1609_08621_b200 import inputs as _inputs
        configs = []
        cases = [("configs[1]: N=2^20 Plummer mix, binary tree, theta=0.7", lambda: _inputs.config2()),
                 ("configs[3]: 65536 buckets, P-P only, L_pp=4096", lambda: _inputs.config4(65536, 4096, 0)),
                 ("configs[3]: 8192 buckets, P-C only, L_pc=2048", lambda: _inputs.config4(8192, 0, 2048)),
                 ("configs[3]: 16384 buckets, fused, L_pp=L_pc=512", lambda: _inputs.config4(16384, 512, 512))]
        keep = ("case", "n_particles", "n_buckets", "I_pp", "I_pc", "mean_L_pp", "mean_L_pc", "kernel_ms_median",
                "step_ms_median", "interactions_per_s", "frac_fp32_fma_peak", "fixup_sinks", "clocks", "max_rel_err_acc",
                "max_rel_err_pot", "n_sampled_particles", "oracle_sample")
        for name, make in cases:
            t0 = time.time()
            q = make()
            ln = report_case(name, q, ctx, torch, binding, peak_tflops, 40, flags, args.configs_cpu_seconds, quiet=True,
                             modes=False)
            c = {k: ln[k] for k in keep if k in ln}
            c["mean_bucket_occupancy"] = round(float(q.count.mean()), 2)
            c["gen_seconds"] = round(time.time() - t0 - 0.0, 1)
            configs.append(c)
            del q

    cfg["parallelism"] = parallelism_string(world, args.scaling)
    line = {"metric": "P-P+P-C interactions/s", "value": value, "unit": "interactions/s", "n_gpus": world,
            "steps": args.steps, "warmup": warm, "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "strong" if (strong or world == 1) else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cfg, "clocks": clocks, "clocks_extra_keys": clocks_x, "configs": configs, "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline, "cpu_baseline": cpu_baseline, "fixup": fixup, "rank_cost_shares": shares,
            "flops_per_s": flops / (ms_step * 1e-3), "frac_fp32_fma_peak": flops / (ms_step * 1e-3) / 1e12 / (peak_tflops * world),
            "paper_convention_tflops": (PAPER_F_PP * tot_pp + PAPER_F_PC * tot_pc) / (ms_step * 1e-3) / 1e12,
            "interactions_per_s": {"pp": tot_pp / (ms_step * 1e-3), "pc": tot_pc / (ms_step * 1e-3)},
            "gen_seconds": round(gen_s, 1), "flags": args.flags, "pp_leaves": leaves, "group_lists": groups,
            "device_lists": devlists, "fmm": fmm}
    # `e2e` stays the plain call on the headline lists (the slowest host-buffer path: 2.2 GB of lists cross PCIe every
    # step); the other host-buffer calls measured above move fewer bytes for the same forces -- name the fastest
    cands = [("e2e", e2e), ("pp_leaves.e2e", (leaves or {}).get("e2e")), ("group_lists.e2e", (groups or {}).get("e2e")),
             ("device_lists.tree_host_call", (devlists or {}).get("tree_host_call"))]
    cands = [(k, v) for k, v in cands if v]
    if cands:
        k_best, v_best = min(cands, key=lambda kv: kv[1]["ms_per_step"])
        line["e2e_best"] = {"key": k_best, "ms_per_step": v_best["ms_per_step"], "h2d_bytes_per_step": v_best.get("h2d_bytes_per_step"),
                            "note": "fastest of the library's host-buffer calls on this workload; every candidate's own key has the details"}
    if fmm is not None:
        fmm["frac_fp32_fma_peak_local_kernel"] = fmm["local_expansion_tflops"] / peak_tflops
    if groups is not None:
        groups["frac_fp32_fma_peak_kernel"] = (F_PP * groups["I_pp"] + F_PC * groups["I_pc"]) / (groups["kernel_ms"] * 1e-3) / 1e12 / peak_tflops
    if leaves is not None:
        leaves["frac_fp32_fma_peak_kernel"] = flops / (leaves["kernel_ms"] * 1e-3) / 1e12 / peak_tflops
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# --report: every BASELINE.json config through the resident call (kernel-only timing from the
# library's CUDA events, median of `reps`), the oracle timed and compared on a bounded sample of the
# same buckets.  One JSON line per case; not the driver's contract line (that is the default mode).
# ------------------------------------------------------------------------------------------------
def report_case(name, p, ctx, torch, binding, peak_tflops, reps, flags, cpu_seconds, note="", quiet=False, modes=True):
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    has_pc = p.cells is not None and p.cells.shape[0] > 0 and p.pc_off is not None
    d = dict(xyzm=t(p.xyzm), cells=t(p.cells) if has_pc else None, first=t(p.first), count=t(p.count),
             pp_off=t(p.pp_off), pp_idx=t(p.pp_idx), pc_off=t(p.pc_off) if has_pc else None,
             pc_idx=t(p.pc_idx) if has_pc else None)
    out = torch.zeros((p.n, 4), dtype=torch.float32, device=dev)
    step = lambda: ctx.gravity_eval(d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"],
                                    d["pc_off"], d["pc_idx"], p.eps, out, flags=flags)
    for _ in range(3):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(torch, torch.cuda.current_device())   # clocks and throttle reasons over this case's timed calls
    sampler.start()
    ctx.profile_read(); ctx.profile_enable(True)
    kms, sms_, fms = [], [], []
    for _ in range(reps):
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(); step(); e1.record(); torch.cuda.synchronize()
        n, ms, fx = ctx.profile_read()
        kms.append(ms / max(n, 1)); sms_.append(e0.elapsed_time(e1)); fms.append(fx / max(n, 1))
    ctx.profile_enable(False)
    st = ctx.get_stats()
    I_pp, I_pc = p.I_pp, (p.I_pc if has_pc else 0)
    assert st["interactions_pp"] == I_pp and st["interactions_pc"] == I_pc and st["bad_entries"] == 0
    k_med, k_best = float(np.median(kms)), float(min(kms))
    flops = F_PP * I_pp + F_PC * I_pc
    line = {"case": name, "n_particles": p.n, "n_buckets": p.n_buckets, "I_pp": I_pp, "I_pc": I_pc,
            "mean_L_pp": round(float(np.diff(p.pp_off).mean()), 1) if p.pp_off is not None else 0,
            "mean_L_pc": round(float(np.diff(p.pc_off).mean()), 1) if has_pc else 0,
            "kernel_ms_median": k_med, "kernel_ms_best": k_best, "step_ms_median": float(np.median(sms_)),
            "interactions_per_s": (I_pp + I_pc) / (k_med * 1e-3), "tflops": flops / (k_med * 1e-3) / 1e12,
            "frac_fp32_fma_peak": flops / (k_med * 1e-3) / 1e12 / peak_tflops,
            "paper_convention_tflops": (PAPER_F_PP * I_pp + PAPER_F_PC * I_pc) / (k_med * 1e-3) / 1e12, "note": note,
            "fixup_sinks": st["fixup_sinks"], "fixup_frac": st["fixup_sinks"] / max(1, int(p.count.sum())),
            "fixup_kernel_ms_median": float(np.median(fms))}
    line["frac_fp32_fma_peak_step"] = flops / (line["step_ms_median"] * 1e-3) / 1e12 / peak_tflops
    # the two other precision modes, timed whole-step (3 calls each): no fix-up at all; every sink in fp64
    for key, fl in ((("step_ms_no_fixup", flags | binding.NO_FIXUP), ("step_ms_fp64_all", flags | binding.FIXUP_ALL)) if modes else ()):
        ts = []
        for _ in range(3):
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.gravity_eval(d["xyzm"], d["cells"], d["first"], d["count"], d["pp_off"], d["pp_idx"], d["pc_off"],
                             d["pc_idx"], p.eps, out, flags=fl)
            e1.record(); torch.cuda.synchronize()
            ts.append(e0.elapsed_time(e1))
        line[key] = float(np.median(ts))
    step()            # leave the default-mode result in `out` for the comparison below
    torch.cuda.synchronize()
    line["clocks"] = sampler.stop()
    if cpu_seconds > 0:
        import oracle
        nb = p.n_buckets
        cost = p.count.astype(np.int64) * ((np.diff(p.pp_off) if p.pp_off is not None else 0) +
                                           (np.diff(p.pc_off) if has_pc else 0))
        per_bucket = max(float(cost.mean()), 1.0) / 3.0e6 * 1.0      # ~3e6 interactions/s per core-second guess
        n_s = int(min(nb, max(64, cpu_seconds * oracle.num_threads() / max(per_bucket, 1e-9))))
        sel = np.unique(np.linspace(0, nb - 1, n_s).astype(np.int64))
        args = (p.xyzm, p.cells if has_pc else None, p.first, p.count,
                p.pp_off if p.pp_off is not None else np.zeros(nb + 1, np.int64),
                p.pp_idx if p.pp_idx is not None else np.zeros(0, np.int32),
                p.pc_off if has_pc else np.zeros(nb + 1, np.int64), p.pc_idx if has_pc else np.zeros(0, np.int32), p.eps)
        t0 = time.perf_counter()
        ref = oracle.gravity_eval(*args, sel=sel)
        dt = time.perf_counter() - t0
        rows = np.concatenate([np.arange(p.first[b], p.first[b] + p.count[b]) for b in sel]).astype(np.int64)
        got = out[torch.from_numpy(rows).to(dev)].cpu().numpy().astype(np.float64)
        r = ref[rows]
        ea = np.linalg.norm(got[:, :3] - r[:, :3], axis=1) / np.linalg.norm(r[:, :3], axis=1)
        ep = np.abs(got[:, 3] - r[:, 3]) / np.abs(r[:, 3])
        S = oracle.contribution_norms(*args, sel=sel)   # conditioning of each sum
        kappa = S[rows] / np.linalg.norm(r[:, :3], axis=1)
        line.update({"kappa_max": float(kappa.max()), "kappa_median": float(np.median(kappa)),
                     "max_err_over_kappa": float((ea / kappa).max()), "n_sampled_particles": int(len(rows)),
                     "n_acc_err_above_2e-5": int((ea > 2e-5).sum())})
        line.update({"oracle_interactions_per_s": float(cost[sel].sum()) / dt, "oracle_cores": oracle.num_threads(),
                     "oracle_sample": f"{len(sel)} of {nb} buckets, {dt:.1f} s",
                     "max_rel_err_acc": float(ea.max()), "max_rel_err_pot": float(ep.max())})
    if not quiet:
        print(json.dumps(line), flush=True)
    del d, out
    torch.cuda.empty_cache()
    return line


def run_report(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --report: no CUDA device; the product path has no CPU fallback")
    from paper_1609_08621_b200 import binding, inputs
    peaks, _ = load_peaks()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    peak = sms * FP32_LANES_PER_SM * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    ctx = binding.Context(0)
    rc = lambda name, p, note="": report_case(name, p, ctx, torch, binding, peak, args.report_reps, args.flags,
                                              args.cpu_seconds, note)
    lines = []
    want = set(args.report.split(","))
    if "1" in want or "all" in want:
        lines.append(rc("cfg1 N=4096 uniform, octree", inputs.config1()))
    if "2" in want or "all" in want:
        lines.append(rc("cfg2 N=2^20 Plummer mix", inputs.config2()))
    if "3" in want or "all" in want:
        lines.append(rc(f"cfg3 N={args.ng}^3 Zel'dovich (headline)", inputs.config3(args.ng)))
    if "4" in want or "all" in want:
        nb = 65536
        for lpp in (32, 128, 512, 2048, 4096):
            lines.append(rc(f"cfg4 P-P only L_pp={lpp}", inputs.config4(nb, lpp, 0), "reuse 16"))
        for lpc, nbc in ((32, 65536), (128, 65536), (512, 16384), (2048, 8192)):
            lines.append(rc(f"cfg4 P-C only L_pc={lpc}", inputs.config4(nbc, 0, lpc), f"{nbc} buckets, reuse 16"))
        for l, nbc in ((32, 65536), (128, 65536), (512, 16384), (2048, 4096)):
            lines.append(rc(f"cfg4 fused L_pp=L_pc={l}", inputs.config4(nbc, l, l), f"{nbc} buckets, reuse 16"))
    for tok in sorted(want):   # one config-4 shape by itself: c4:<buckets>:<L_pp>:<L_pc> (what an ncu capture of one shape runs)
        if tok.startswith("c4:"):
            nbc, lpp, lpc = (int(v) for v in tok[3:].split(":"))
            lines.append(rc(f"cfg4 {nbc} buckets L_pp={lpp} L_pc={lpc}", inputs.config4(nbc, lpp, lpc), "reuse 16"))
    if "5" in want or "all" in want:
        # N = 2^26: a contiguous range of 2^20 buckets (lists built for that range), resident and streamed
        xyzm, eps = inputs.config5_particles()
        p = inputs.build_tree(xyzm, "binary", 16, name="cfg5")
        del xyzm
        b0 = p.n_buckets // 3; b1 = b0 + (1 << 20)
        pp_off, pp_idx, pc_off, pc_idx = inputs.build_lists(p, 0.55, eps, b0, b1)
        q = inputs.Problem(name="cfg5_range", xyzm=p.xyzm, cells=p.cells, first=np.ascontiguousarray(p.first[b0:b1]),
                           count=np.ascontiguousarray(p.count[b0:b1]), pp_off=pp_off, pp_idx=pp_idx, pc_off=pc_off,
                           pc_idx=pc_idx, eps=eps)
        ln = rc("cfg5 N=2^26 theta=0.55, 2^20 of %d buckets, resident" % p.n_buckets, q)
        lines.append(ln)
        dev = torch.device("cuda", 0)
        d_x = torch.from_numpy(q.xyzm).to(dev); d_c = torch.from_numpy(q.cells).to(dev)
        out = torch.zeros((q.n, 4), dtype=torch.float32, device=dev)
        pin = lambda a: torch.from_numpy(a).pin_memory()
        h = [pin(q.first), pin(q.count), pin(pp_off), pin(pp_idx), pin(pc_off), pin(pc_idx)]
        for ns, chunk in ((1, 1 << 24), (3, 1 << 24), (3, 1 << 26)):
            ts = []
            for _ in range(4):
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.gravity_eval_streamed(d_x, d_c, h[0], h[1], h[2], h[3], h[4], h[5], eps, out, n_streams=ns,
                                          max_entries_per_chunk=chunk, flags=args.flags)
                e1.record(); torch.cuda.synchronize()
                ts.append(e0.elapsed_time(e1))
            st = ctx.get_stats()
            ms = float(np.median(ts[1:]))
            sl = {"case": f"cfg5 streamed lists, {ns} stream(s), chunk {chunk} entries", "chunks": st["chunks"],
                  "ms": ms, "interactions_per_s": (q.I_pp + q.I_pc) / (ms * 1e-3),
                  "h2d_gb": (pp_idx.nbytes + pc_idx.nbytes + pp_off.nbytes + pc_off.nbytes + 8 * q.n_buckets) / 1e9,
                  "resident_kernel_ms": ln["kernel_ms_median"]}
            print(json.dumps(sl), flush=True)
            lines.append(sl)
    if "5full" in want:
        # the WHOLE of config 5 resident: lists are built range by range on the host and assembled on the device
        xyzm, eps = inputs.config5_particles()
        p = inputs.build_tree(xyzm, "binary", 16, name="cfg5")
        del xyzm
        dev = torch.device("cuda", 0)
        nb = p.n_buckets
        step_b = 1 << 20
        pp_offs, pc_offs, pp_parts, pc_parts = [np.zeros(1, np.int64)], [np.zeros(1, np.int64)], [], []
        t0 = time.perf_counter()
        for b0 in range(0, nb, step_b):
            po, pi, co, ci = inputs.build_lists(p, 0.55, eps, b0, min(nb, b0 + step_b))
            pp_offs.append(po[1:] + pp_offs[-1][-1]); pc_offs.append(co[1:] + pc_offs[-1][-1])
            pp_parts.append(torch.from_numpy(pi).to(dev)); pc_parts.append(torch.from_numpy(ci).to(dev))
        build_s = time.perf_counter() - t0
        pp_off = np.concatenate(pp_offs); pc_off = np.concatenate(pc_offs)
        d_ppi = torch.cat(pp_parts); del pp_parts
        d_pci = torch.cat(pc_parts); del pc_parts
        d_x = torch.from_numpy(p.xyzm).to(dev); d_c = torch.from_numpy(p.cells).to(dev)
        d_f = torch.from_numpy(p.first).to(dev); d_n = torch.from_numpy(p.count).to(dev)
        d_ppo = torch.from_numpy(pp_off).to(dev); d_pco = torch.from_numpy(pc_off).to(dev)
        out = torch.zeros((p.n, 4), dtype=torch.float32, device=dev)
        fl = args.flags
        step = lambda: ctx.gravity_eval(d_x, d_c, d_f, d_n, d_ppo, d_ppi, d_pco, d_pci, eps, out, flags=fl)
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        ctx.profile_read(); ctx.profile_enable(True)
        for _ in range(5):
            step()
        torch.cuda.synchronize()
        n_k, ms_k, _ = ctx.profile_read(); ctx.profile_enable(False)
        st = ctx.get_stats()
        cnt = p.count.astype(np.int64)
        I_pp, I_pc = int(np.dot(cnt, np.diff(pp_off))), int(np.dot(cnt, np.diff(pc_off)))
        assert st["interactions_pp"] == I_pp and st["interactions_pc"] == I_pc and st["bad_entries"] == 0
        k_ms = ms_k / n_k
        flops = F_PP * I_pp + F_PC * I_pc
        line = {"case": "cfg5 N=2^26 theta=0.55, ALL %d buckets resident" % nb, "n_particles": p.n, "n_buckets": nb,
                "I_pp": I_pp, "I_pc": I_pc, "mean_L_pp": round(float(np.diff(pp_off).mean()), 1),
                "mean_L_pc": round(float(np.diff(pc_off).mean()), 1), "list_gb": (d_ppi.numel() + d_pci.numel()) * 4 / 1e9,
                "kernel_ms_median": k_ms, "interactions_per_s": (I_pp + I_pc) / (k_ms * 1e-3),
                "tflops": flops / (k_ms * 1e-3) / 1e12, "frac_fp32_fma_peak": flops / (k_ms * 1e-3) / 1e12 / peak,
                "host_list_build_s": round(build_s, 1),
                "device_mem_gb": round(torch.cuda.max_memory_allocated() / 1e9, 1)}
        if args.cpu_seconds > 0:
            import oracle
            sel = np.unique(np.linspace(0, nb - 1, 3000).astype(np.int64))
            # the oracle needs host lists: rebuild them for the sampled buckets only (same generator, same result)
            rows_all, err_a, err_p = 0, 0.0, 0.0
            for b in sel[:: max(1, len(sel) // 300)]:
                po, pi, co, ci = inputs.build_lists(p, 0.55, eps, int(b), int(b) + 1)
                ref = oracle.gravity_eval(p.xyzm, p.cells, p.first[b:b + 1], p.count[b:b + 1], po, pi, co, ci, eps)
                r = np.arange(p.first[b], p.first[b] + p.count[b])
                got = out[int(r[0]):int(r[-1]) + 1].cpu().numpy().astype(np.float64)
                ea = np.linalg.norm(got[:, :3] - ref[r, :3], axis=1) / np.linalg.norm(ref[r, :3], axis=1)
                ep = np.abs(got[:, 3] - ref[r, 3]) / np.abs(ref[r, 3])
                err_a = max(err_a, float(ea.max())); err_p = max(err_p, float(ep.max())); rows_all += len(r)
            line.update({"max_rel_err_acc": err_a, "max_rel_err_pot": err_p, "n_sampled_particles": rows_all})
        print(json.dumps(line), flush=True)
        lines.append(line)
    ctx.close()
    return lines


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ng", type=int, default=256, help="lattice size per axis (256 = the headline 2^24 config)")
    ap.add_argument("--flags", type=lambda v: int(v, 0), default=0, help="extra PKDG_* flags for every evaluation call (e.g. 0x10 = PKDG_NO_FIXUP)")
    ap.add_argument("--scaling", default="strong", choices=["strong", "weak"], help="N > 1: one problem sharded (default) or N replicas")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-leaves", action="store_true", help="skip the extra PKDG_PP_LEAVES measurement")
    ap.add_argument("--no-groups", action="store_true", help="skip the extra group-shared-lists measurement")
    ap.add_argument("--no-fmm", action="store_true", help="skip the extra four-list (C-C / C-P local expansion) measurement")
    ap.add_argument("--no-device-lists", action="store_true", help="skip the extra device list-construction measurement")
    ap.add_argument("--no-configs", action="store_true", help="skip the extra `configs` key (config 2 and three config-4 shapes)")
    ap.add_argument("--configs-cpu-seconds", type=float, default=3.0, help="oracle sample per case of the `configs` key")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--e2e-streams", type=int, default=4)
    ap.add_argument("--e2e-chunk", type=int, default=1 << 23)
    ap.add_argument("--report", default="", help="comma list of configs (1,2,3,4,5,5full, all, or c4:<buckets>:<L_pp>:<L_pc>): per-case report lines "
                                                  "instead of the contract line")
    ap.add_argument("--report-reps", type=int, default=10)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.report:
        if rank == 0:
            run_report(args)
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
