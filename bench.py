#!/usr/bin/env python
"""bench.py -- throughput of the SL1M hot path on B200 (contract: see the task prompt / DESIGN.md).

A "step" is ONE FISTA iteration = one pass of the whole hot path:
forward A y, residual, adjoint A^H r, threshold + momentum update, objective partials -- issued
through the C ABI (`sl1m_solve`, n_iter = 1, warm-started from the previous step's image).
Default workload: BASELINE.json configs[4], the configuration the metric is quoted on
(1024^2 pixels x 406,400 visibilities, full w-term), synthetic seeded inputs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

N > 1 (torchrun): the path does not shard under north_star ("one GPU, no collectives"), so every
rank runs an independent replica of the workload; value = all ranks' terms / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import fista_lambda, make_workload  # noqa: E402

METRIC = "pixel_x_visibility_terms_per_s (A and A^H inside one FISTA iteration)"
UNIT = "terms/s"
MUFU_PER_SM_PER_CLK = 16      # 4 SFU lanes per SM sub-partition x 4 (measured 15.7, profiles/r1_microbench.md)
SM_COUNT = 148
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
# `ncu --set full` captures summarised under profiles/ (config, kernel) -> bytes
NCU_DRAM_BYTES_PER_LAUNCH = {(5, "fwd"): 100.70e6, (5, "adj"): 52.56e6, (4, "fwd"): 341.8e6, (4, "adj"): 328.0e6}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"sm_max_mhz": 1965.0, "hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            if not (t0 - 0.05 <= ts <= t1 + 0.25):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                smax.append(float(f[1]))
                power.append(float(f[2]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def _oracle_sample(wl, seconds: float):
    """Time the fp64 oracle (as it stands) on a bounded sample of the workload: forward for a few
    visibility rows on a dense image + adjoint for a few pixels, each a full-length sum."""
    import oracle
    o = oracle.Oracle.from_workload(wl)
    rng = np.random.default_rng(12345)
    x = rng.uniform(0, 1, wl.n_pix)
    r = (rng.standard_normal(wl.n_vis) + 1j * rng.standard_normal(wl.n_vis))
    cores = oracle.num_threads()
    # probe the rate on a small sample, then size the real one
    nr0 = max(cores, 8)
    t = time.perf_counter()
    o.forward(x, rows=rng.choice(wl.n_vis, min(nr0, wl.n_vis), replace=False))
    rate = min(nr0, wl.n_vis) * wl.n_pix / max(time.perf_counter() - t, 1e-9)
    n_rows = int(min(wl.n_vis, max(cores, rate * seconds / 2 / wl.n_pix)))
    n_cols = int(min(wl.n_pix, max(cores, rate * seconds / 2 / wl.n_vis)))
    for attempt in range(2):
        rows = rng.choice(wl.n_vis, n_rows, replace=False)
        cols = rng.choice(wl.n_pix, n_cols, replace=False)
        t = time.perf_counter()
        o.forward(x, rows=rows)
        o.adjoint(r, cols=cols)
        dt = time.perf_counter() - t
        # the small probe under-estimates the rate (thread start-up): if the sample came out much shorter
        # than asked for, size it again from its own rate, once
        grow = seconds / max(dt, 1e-9)
        if attempt == 0 and grow > 1.5 and (n_rows < wl.n_vis or n_cols < wl.n_pix):
            n_rows = int(min(wl.n_vis, n_rows * grow))
            n_cols = int(min(wl.n_pix, n_cols * grow))
            continue
        break
    terms = n_rows * wl.n_pix + n_cols * wl.n_vis
    return {"value": terms / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"forward of {n_rows} sampled visibility rows x all {wl.n_pix} pixels (dense image) + "
                      f"adjoint of {n_cols} sampled pixels x all {wl.n_vis} visibilities, {dt:.1f} s",
            "seconds": dt, "terms": terms}


def run_reference(args, rank: int):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    if rank != 0:
        return
    wl = make_workload(args.config)
    for _ in range(args.warmup):
        _oracle_sample(wl, 0.5)
    vals, secs = [], []
    for _ in range(args.steps):
        s = _oracle_sample(wl, args.ref_seconds)
        vals.append(s["terms"])
        secs.append(s["seconds"])
    value = sum(vals) / sum(secs)
    last = s
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{wl.name}", "n_pix": wl.n_pix, "n_vis": wl.n_vis,
                   "note": "each step = a bounded sample of the workload on the host cores"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": last["cores"], "kind": "oracle",
                         "sample": last["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def reduce_over_ranks(total_ms: float, e2e_ms: float, launches: int, world: int, device):
    """Replicas only: every rank ran the same workload on its own GPU, with no
    data-path collective.  The job's time is the MAX over ranks (device-timed), its launch count the
    SUM.  `device` is the rank's CUDA device under NCCL, or "cpu" under gloo (the CPU tests)."""
    if world <= 1:
        return total_ms, e2e_ms, launches
    import torch
    import torch.distributed as dist
    t = torch.tensor([total_ms, e2e_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ln = torch.tensor([launches], device=device, dtype=torch.int64)
    dist.all_reduce(ln, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), int(ln[0])


def aggregate_value(world: int, terms_per_step: float, steps: int, t_max_ms: float) -> float:
    """Whole-job throughput: the terms ALL ranks processed / the max-over-ranks time."""
    return world * terms_per_step * steps / (t_max_ms * 1e-3)


def run_ours(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    import paper_1310_2078_b200 as sl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the SL1M path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    sl.load_library()
    peaks, peaks_src = _peaks()

    wl = make_workload(args.config)
    t_plan = time.perf_counter()
    plan = sl.Plan.from_workload(wl, dense_forward=args.dense_forward)
    torch.cuda.synchronize()
    t_plan = time.perf_counter() - t_plan
    n_terms = float(wl.n_pix) * float(wl.n_vis)
    stream = torch.cuda.current_stream()

    # measured data through the product path: V = A x_true + noise
    x_true = torch.from_numpy(wl.x_true.astype(np.float32)).to(dev)
    V = plan.forward(x_true) + torch.from_numpy(wl.noise.astype(np.complex64)).to(dev)
    lam = fista_lambda(wl)
    if lam == 0.0:
        lam = 0.01 * float(plan.adjoint(V).abs().max())
    t0 = time.perf_counter()
    L = plan.max_eig(args.n_pow) * 1.05
    t_eig = time.perf_counter() - t0

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def ev():
        return torch.cuda.Event(enable_timing=True)

    # ---------------- device-resident steps ----------------
    x = torch.zeros(wl.n_pix, dtype=torch.float32, device=dev)
    x_next = torch.empty_like(x)
    for _ in range(args.warmup):
        plan.solve(V, lam, L=L, n_iter=1, x0=x, out=x_next, want_info=False)
        x, x_next = x_next, x
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    launches0 = plan.launch_count
    pairs = []
    nnz_steps = []          # non-zero pixels of each step's forward input (zero-skipping forward)
    t_wall0 = time.time()
    torch.cuda.synchronize()
    for _ in range(args.steps):
        nnz_steps.append(torch.count_nonzero(x))      # device scalar, queued before the flush; read after the loop
        flush.zero_()
        a, b = ev(), ev()
        a.record(stream)
        plan.solve(V, lam, L=L, n_iter=1, x0=x, out=x_next, want_info=False)
        b.record(stream)
        pairs.append((a, b))
        x, x_next = x_next, x
    torch.cuda.synchronize()
    t_wall1 = time.time()
    launches = plan.launch_count - launches0
    step_ms = [a.elapsed_time(b) for a, b in pairs]
    total_ms = sum(step_ms)
    clocks = sampler.stop(t_wall0, t_wall1)

    # ---------------- per-apply timings (dominant kernels), same flush discipline ----------------
    def time_call(fn, reps):
        ts = []
        for _ in range(reps):
            flush.zero_()
            a, b = ev(), ev()
            a.record(stream)
            fn()
            b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return ts
    # a DENSE positive image: every pixel non-zero, so the zero-skipping forward evaluates all N_p x N_v terms
    y = torch.rand(wl.n_pix, dtype=torch.float32, device=dev, generator=torch.Generator(device=dev).manual_seed(7)) + 0.5
    vis_out = torch.empty(wl.n_vis, dtype=torch.complex64, device=dev)
    img_out = torch.empty(wl.n_pix, dtype=torch.float32, device=dev)
    reps = max(3, min(args.steps, 5))
    plan.forward(y, out=vis_out); plan.adjoint(V, out=img_out)
    t_fwd = time_call(lambda: plan.forward(y, out=vis_out), reps)
    t_adj = time_call(lambda: plan.adjoint(V, out=img_out), reps)

    # ---------------- end-to-end: HOST buffers through the C ABI, copies inside the timed region ----
    V_host = V.cpu().pin_memory()
    x_host = x.cpu().pin_memory()
    out_host = torch.empty(wl.n_pix, dtype=torch.float32).pin_memory()
    plan.solve_host(V_host, lam, L, 1, out_host, x0_host=x_host, want_info=False)
    e2e_ms = []
    e2e_nnz = []
    for _ in range(max(2, min(args.steps, 5))):
        e2e_nnz.append(int(np.count_nonzero(x_host.numpy())))
        flush.zero_()
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(stream)
        plan.solve_host(V_host, lam, L, 1, out_host, x0_host=x_host, want_info=False)
        b.record(stream)
        torch.cuda.synchronize()
        e2e_ms.append(a.elapsed_time(b))
        x_host.copy_(out_host)
    h2d = 8 * wl.n_vis + 4 * wl.n_pix
    d2h = 4 * wl.n_pix

    # ---------------- reduce over ranks (replicas) ----------------
    e2e_mean = sum(e2e_ms) / len(e2e_ms)
    t_max, e2e_mean, launches = reduce_over_ranks(total_ms, e2e_mean, launches, world, dev)
    if rank != 0:
        plan.close()
        return

    # Terms EVALUATED per step: the adjoint takes all N_p x N_v; the forward only the pixels with y_k != 0
    # (zero-skipping, include/sl1m.h; the skipped terms are exactly zero) -- all of them when the plan does not skip.
    desc = plan.describe()
    skip = bool(desc["zero_skip"])
    nnz_list = [int(v) for v in nnz_steps] if skip else [wl.n_pix] * args.steps
    e2e_nnz = e2e_nnz if skip else [wl.n_pix] * len(e2e_nnz)
    terms_per_step = (float(wl.n_pix) + sum(nnz_list) / len(nnz_list)) * float(wl.n_vis)
    value = aggregate_value(world, terms_per_step, args.steps, t_max)
    e2e_value = aggregate_value(world, (float(wl.n_pix) + sum(e2e_nnz) / len(e2e_nnz)) * float(wl.n_vis), 1, e2e_mean)
    f_max = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    fwd_ms, adj_ms = statistics.median(t_fwd), statistics.median(t_adj)

    def bound(kind, per16, packed, clock_hz):
        """Issue-rate bound (terms/s) of one apply kernel (`kind` = "fwd" or "adj") for ITS OWN instruction mix
        (SASS-counted).  A fraction f = per16/16 of the terms takes an FMA-pipe polynomial
        (0 MUFU), the rest the MUFU path.  Three per-SM limits, each in terms/clk:
          MUFU pipe   16 results/clk            / (mufu_per_term * (1 - f))
          FMA pipe    128 fp32 lanes/clk        / lane-ops per term (an FFMA2 is 2 lane-ops)
          issue       4 warp-instr = 128 thread-instr/clk / issue slots per term
        peak = the smallest of the three.  The adjoint of a REAL image needs one cosine per term,
        Re(e^{iX} r) = |r| cos(X + arg r): 1 MUFU + 5 lane-ops (3 phase + FMUL.RZ + 1 accumulate)."""
        f = per16 / 16.0
        gauss, gains = int(desc["gaussian"]), bool(desc["gains"])   # gaussian: 0 delta, 1 per-pixel sigma, 2 per-tile sigma
        grouped = int(desc["gains"]) == 2            # one polar gain product per pixel per 8 samples
        m_term = desc["adj_mufu_per_term"] if kind == "adj" else desc["mufu_per_term_mufu_path"]
        one_cos = kind == "adj" and m_term == 1
        mufu = m_term * (1.0 - f)
        if one_cos:
            lane_mufu_path, lane_poly_path = 5.0, 12.0          # poly: 3 phase + 3 reduce + 1 + 4 cos + 1 accumulate
            extra = 1.5 if grouped else 0.0                      # + phase add per term, gain product per 8 terms
        else:
            lane_mufu_path = {0: 6.0, 1: 20.0, 2: (12.0 if kind == "adj" else 13.0) if packed else 16.0}[gauss]
            lane_poly_path = 18.0                    # 3 phase + 3 reduce + 1 + 5 sin + 4 cos + 2 accumulate
            extra = 0.5 if grouped else (10.0 if gains else 0.0)
        lanes = lane_mufu_path * (1.0 - f) + lane_poly_path * f + extra
        if packed:   # FFMA2 halves the issue slots of everything but FMUL.RZ and MUFU
            if one_cos:
                slots = 4.0 * (1.0 - f) + 7.5 * f + 0.25 + (1.0 if grouped else 0.0)
            else:
                slots = ((7.5 if kind == "adj" else 10.0) if gauss == 2 else 5.5) * (1.0 - f) + 11.0 * f + 0.25 \
                    + (2.2 if grouped else 0.0)      # gains: address arithmetic of 8 gain loads per 4 pixels
        else:
            slots = {0: 8.0, 1: 24.0, 2: 19.0}[gauss] * (1.0 - f) + 20.0 * f + 0.125 + (10.0 if gains else 0.0)
        b_mufu = SM_COUNT * MUFU_PER_SM_PER_CLK * clock_hz / mufu
        b_fma = SM_COUNT * 128.0 * clock_hz / lanes
        b_issue = SM_COUNT * 128.0 * clock_hz / slots
        return min(b_mufu, b_fma, b_issue), b_mufu, b_fma, b_issue

    pk_f, pk_f_mufu, pk_f_fma, pk_f_issue = bound("fwd", desc["fwd_poly_per16"], desc["fwd_packed_pairs"], f_max)
    pk_a, pk_a_mufu, pk_a_fma, pk_a_issue = bound("adj", desc["adj_poly_per16"], desc["adj_packed_pairs"], f_max)
    ach_f, ach_a = n_terms / (fwd_ms * 1e-3), n_terms / (adj_ms * 1e-3)
    # the dominant kernel of the TIMED STEP: the adjoint evaluates every term, the forward only the non-zero pixels
    step_ms_mean = t_max / args.steps
    dom_is_adj = adj_ms >= step_ms_mean - adj_ms
    m_dom = desc["adj_mufu_per_term"] if dom_is_adj else desc["mufu_per_term_mufu_path"]
    mufu_only = SM_COUNT * MUFU_PER_SM_PER_CLK * f_max / m_dom      # every term on the MUFU path
    # best any MUFU/FMA split of the dominant kernel's instruction set could do (delta pixels, unit gains):
    # MUFU time = FMA time, m (1-f)/16 = (a (1-f) + b f)/128 with (m, a, b) = (2, 6, 18) forward, (1, 5, 12) adjoint
    m_, a_, b_ = (1.0, 5.0, 12.0) if (dom_is_adj and m_dom == 1) else (2.0, 6.0, 18.0)
    f_bal = (8.0 * m_ - a_) / (8.0 * m_ - a_ + b_)
    balanced = (SM_COUNT * MUFU_PER_SM_PER_CLK * f_max / (m_ * (1.0 - f_bal))
                if not (desc["gaussian"] or desc["gains"]) else None)
    dom = "sl1m::adj_kernel" if dom_is_adj else "sl1m::fwd_kernel"
    if (desc["adj_packed_pairs"] if dom_is_adj else desc["fwd_packed_pairs"]):      # the packed R = 8 kernels
        if int(desc["gaussian"]) == 2:
            dom += "_gtx2"
        elif dom_is_adj and int(desc["gains"]) == 2:
            dom += "_g2x2"
        elif dom_is_adj and desc["adj_mufu_per_term"] == 1:
            dom += "_c1"
        else:
            dom += "_x2"
    achieved, peak = (ach_a, pk_a) if dom_is_adj else (ach_f, pk_f)
    traffic = NCU_DRAM_BYTES_PER_LAUNCH.get((args.config, "adj" if dom_is_adj else "fwd"))
    roof = {
        "bound": "alu", "kernel": dom, "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "Tterm/s",
        "frac": achieved / peak, "traffic": traffic,
        "peak_basis": f"min(MUFU pipe, FMA pipe, issue slots) for the kernel's own SASS instruction mix at "
                      f"{f_max/1e6:.0f} MHz (sm_max_mhz, {peaks_src}): {SM_COUNT} SMs x {MUFU_PER_SM_PER_CLK} MUFU/clk, "
                      f"x 128 fp32 lanes/clk, x 128 thread-instr/clk; fwd {desc['fwd_poly_per16']}/16 and adj "
                      f"{desc['adj_poly_per16']}/16 of the terms use FMA-pipe polynomials; MUFU per MUFU-path term: fwd "
                      f"{desc['mufu_per_term_mufu_path']}, adj {desc['adj_mufu_per_term']} (real image: one cosine per adjoint term)",
        "traffic_basis": "dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full "
                         "(profiles/, same kernel and workload; null = not captured); algorithmic bytes at config 5: ~30 MB in per apply "
                         "+ the split partials (37 x 3.25 MB forward, 15 x 4 MB adjoint, partly L2-resident)",
        "mufu_only_bound_Tterm_per_s": mufu_only / 1e12,
        "frac_vs_mufu_only_bound": achieved / mufu_only,
        "best_split_bound_Tterm_per_s": None if balanced is None else balanced / 1e12,
        "frac_vs_best_split_bound": None if balanced is None else achieved / balanced,
        "fwd": {"ms": fwd_ms, "Tterm_per_s": ach_f / 1e12, "peak": pk_f / 1e12, "frac": ach_f / pk_f,
                "mufu_bound": pk_f_mufu / 1e12, "fma_bound": pk_f_fma / 1e12, "issue_bound": pk_f_issue / 1e12},
        "adj": {"ms": adj_ms, "Tterm_per_s": ach_a / 1e12, "peak": pk_a / 1e12, "frac": ach_a / pk_a,
                "mufu_bound": pk_a_mufu / 1e12, "fma_bound": pk_a_fma / 1e12, "issue_bound": pk_a_issue / 1e12},
        "plan": desc,
        "note": "per-apply time = C-ABI call (main kernel + O(N) epilogues, < 0.1 % of it); "
                "not an HBM-bound path: the matrix is generated, never read",
    }
    if clocks.get("sm_mhz"):
        pk_c = bound("adj" if dom_is_adj else "fwd", desc["adj_poly_per16"] if dom_is_adj else desc["fwd_poly_per16"],
                     desc["adj_packed_pairs"] if dom_is_adj else desc["fwd_packed_pairs"], clocks["sm_mhz"] * 1e6)[0]
        roof["frac_at_sampled_clock"] = achieved / pk_c

    cpu = None
    if not args.no_cpu_baseline:
        cpu = _oracle_sample(wl, args.cpu_seconds)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{wl.name}", "n_pix": wl.n_pix, "n_vis": wl.n_vis,
                   "pixel_kind": "gaussian" if wl.sigma is not None else "delta",
                   "gains": wl.gains is not None, "lambda": lam, "L": L,
                   "l2_flush": "256 MiB device memset between timed steps",
                   "step": "one FISTA iteration via sl1m_solve(n_iter=1, x0=previous image); per-apply timings use a dense image",
                   "parallelism": "replicas" if world > 1 else "single-gpu"},
        "iters_per_s": world * args.steps / (t_max * 1e-3),
        "terms": {"counted": "evaluated terms: N_v x (N_p for A^H + pixels with y_k != 0 for A)",
                  "zero_skip": skip, "fwd_active_fraction": sum(nnz_list) / len(nnz_list) / wl.n_pix,
                  "fwd_active_pixels_per_step": nnz_list,
                  "dense_equivalent_terms_per_s": aggregate_value(world, 2.0 * n_terms, args.steps, t_max)},
        "step_ms": step_ms, "plan_create_s": t_plan, "max_eig_s": t_eig, "n_pow": args.n_pow,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_mean, "call": "sl1m_solve_host(n_iter=1) with pinned host V, x0, x_out"},
        "gpu_launches": launches, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
        "peaks_source": peaks_src,
    }
    print(json.dumps(line), flush=True)
    plan.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n-pow", type=int, default=4, dest="n_pow")
    ap.add_argument("--cpu-seconds", type=float, default=16.0, dest="cpu_seconds")
    ap.add_argument("--ref-seconds", type=float, default=8.0, dest="ref_seconds")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dense-forward", action="store_true", dest="dense_forward",
                    help="SL1M_DENSE_FORWARD: the forward evaluates every term, also where the image is zero (A/B of the zero-skipping forward)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl")
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
