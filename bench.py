#!/usr/bin/env python
"""bench.py -- throughput of the SL1M hot path on B200 (contract: see the task prompt / DESIGN.md).

A "step" is ONE FISTA iteration = one pass of the whole hot path:
forward A y, residual, adjoint A^H r, threshold + momentum update, objective partials -- issued
through the C ABI's stepping calls (`sl1m_fista_begin` once, then `sl1m_fista_step(1)` per step), so the
warm-up and timed steps are consecutive iterations of ONE continuing FISTA run from I_0 = 0 (momentum on).
The same run is also timed as a single `sl1m_solve(n_iter = warmup + steps)` call ("continuous_solve").
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
MUFU_PER_SM_PER_CLK = 16      # nominal: 4 SFU lanes per SM sub-partition x 4; the line's peaks use the MEASURED rate
SM_COUNT = 148
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the
# `ncu --set full` captures summarised under profiles/ (config, kernel) -> bytes
NCU_DRAM_BYTES_PER_LAUNCH = {(5, "fwd"): 100.95e6, (5, "adj"): 56.39e6, (4, "fwd"): 341.0e6, (4, "adj"): 326.0e6,
                             (2, "fwd"): 1.56e6, (2, "adj"): 1.72e6, (3, "fwd"): 1.90e6, (3, "adj"): 2.10e6}   # profiles/r2_ncu_full_config*.md


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
    wl = make_workload(args.config, **args.overrides)
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

    wl = make_workload(args.config, **args.overrides)
    if args.jitter_sigma and wl.sigma is not None:      # a sigma of its own per pixel: the per-pixel-sigma Gaussian kernels
        wl.sigma = wl.sigma * np.random.default_rng(777).uniform(0.7, 1.3, wl.n_pix)
    t_plan = time.perf_counter()
    plan = sl.Plan.from_workload(wl, dense_forward=args.dense_forward, no_persistent=args.no_persistent,
                                 phase_fp64=args.phase_fp64)
    torch.cuda.synchronize()
    t_plan = time.perf_counter() - t_plan
    n_terms = float(wl.n_pix) * float(wl.n_vis)
    stream = torch.cuda.current_stream()

    # measured data through the product path: V = A x_true + noise
    x_true = torch.from_numpy(wl.x_true.astype(np.float32)).to(dev)
    V = plan.forward(x_true) + torch.from_numpy(wl.noise.astype(np.complex64)).to(dev)
    if args.batch_stop > 0:
        # side measurement: C channels of this geometry, each solved to a tolerance in ONE call
        # (sl1m_plan_set_channels + sl1m_dirty_image + sl1m_solve_stop_batch), against the same channels one after
        # the other through sl1m_solve_stop on single-channel plans
        C = args.batch_stop
        scale = np.linspace(0.9, 1.1, C)
        lam0 = fista_lambda(wl)
        Vs, Ls, plans = [], [], []
        for c in range(C):
            pc = sl.Plan(wl.uvw * scale[c], wl.l, wl.m, wl.sigma, wl.ant_p, wl.ant_q, wl.gains, wl.gauss_model)
            Vs.append(pc.forward(x_true * (1.0 + 0.1 * c / C)) + torch.from_numpy(wl.noise.astype(np.complex64)).to(dev))
            Ls.append(pc.max_eig(args.n_pow) * 1.05)
            plans.append(pc)
        plan.set_channels(scale)
        Vb, Lb = torch.stack(Vs).contiguous(), np.array(Ls, np.float32)

        def timed(fn):
            best = 1e30
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); out = fn(); b.record(stream); torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b))
            return best, out
        kw = dict(max_iter=args.max_iter, tol=args.tol, check_every=args.check_every)
        t_b, (xb, infos) = timed(lambda: plan.solve_stop_batch(Vb, lam0, Lb, x0=plan.dirty_image(Vb), **kw))
        t_s, outs = timed(lambda: [plans[c].solve_stop(Vs[c], lam0, float(Lb[c]), x0=plans[c].dirty_image(Vs[c]), **kw) for c in range(C)])
        same = max(float((xb[c] - outs[c][0]).norm() / outs[c][0].norm().clamp_min(1e-30)) for c in range(C))
        if rank == 0:
            print(json.dumps({"batch_stop": True, "config": args.config, "n_chan": C, "tol": args.tol, "check_every": args.check_every,
                              "batched_ms": t_b, "one_after_the_other_ms": t_s, "speedup": t_s / t_b,
                              "iterations_per_channel": [i.n_iter_done for i in infos],
                              "iterations_per_channel_single_plans": [o[1].n_iter_done for o in outs],
                              "max_rel_l2_batched_vs_single": same,
                              "single_plans_persistent": plans[0].describe()["persistent"]}), flush=True)
        for pc in plans:
            pc.close()
        plan.close()
        return
    if args.applies_only:
        # profiling aid (ncu -k regex:fwd_kernel -s 1 / -k regex:adj_kernel): after the sparse forward above, three
        # forwards on a DENSE image and three adjoints, nothing else
        yd = torch.rand(wl.n_pix, dtype=torch.float32, device=dev, generator=torch.Generator(device=dev).manual_seed(7)) + 0.5
        ts = []
        for fn in (lambda: plan.forward(yd), lambda: plan.adjoint(V)):
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); fn(); b.record(stream); torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
        if rank == 0:
            print(json.dumps({"applies_only": True, "config": args.config, "fwd_ms": ts[:3], "adj_ms": ts[3:],
                              "plan": plan.describe()}), flush=True)
        plan.close()
        return
    lam = fista_lambda(wl)
    if lam == 0.0:
        lam = 0.01 * float(plan.adjoint(V).abs().max())
    t0 = time.perf_counter()
    L = plan.max_eig(args.n_pow) * 1.05
    t_eig = time.perf_counter() - t0

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def ev():
        return torch.cuda.Event(enable_timing=True)

    # ---------------- issue-rate peaks of THIS GPU, measured now (sl1m_measure_peaks, csrc/sl1m_peaks.cu) ----
    pk_meas = sl.measure_peaks() if rank == 0 else None

    # ---------------- device-resident steps: consecutive iterations of one FISTA run ----------------
    skip = bool(plan.describe()["zero_skip"])
    plan.fista_begin(V, lam, L)
    plan.fista_step(args.warmup)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    launches0 = plan.launch_count
    pairs = []
    nnz_steps = []          # pixels the step's forward streams (non-zeros of y_k, padded to 4 per tile)
    t_wall0 = time.time()
    torch.cuda.synchronize()
    for _ in range(args.steps):
        nnz_steps.append(plan.forward_active_pixels() if skip else wl.n_pix)   # synchronises: outside the events
        flush.zero_()
        a, b = ev(), ev()
        a.record(stream)
        plan.fista_step(1)
        b.record(stream)
        pairs.append((a, b))
    torch.cuda.synchronize()
    t_wall1 = time.time()
    launches = plan.launch_count - launches0
    step_ms = [a.elapsed_time(b) for a, b in pairs]
    total_ms = sum(step_ms)
    clocks = sampler.stop(t_wall0, t_wall1)
    x, k_done = plan.fista_image()
    assert k_done == args.warmup + args.steps

    # ---------------- the same run as ONE call: sl1m_solve(n_iter = warmup + steps), events around the call ----
    n_cont = args.cont_iters if args.cont_iters > 0 else args.warmup + args.steps
    trace = torch.zeros(3 * n_cont, dtype=torch.float64, device=dev)
    x_cont = torch.empty_like(x)
    flush.zero_()
    a, b = ev(), ev()
    a.record(stream)
    plan.solve(V, lam, L=L, n_iter=n_cont, out=x_cont, trace=trace, want_info=False)
    b.record(stream)
    torch.cuda.synchronize()
    cont_ms = a.elapsed_time(b)
    cont_same = bool(torch.equal(x_cont, x))
    tr = trace.cpu().numpy().reshape(n_cont, 3)

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
    reps = 10                                   # median of >= 10 timed applies after 3 warm-ups
    for _ in range(3):
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
    nnz_list = [int(v) for v in nnz_steps]
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

    # Measured denominators (sl1m_measure_peaks): MUFU results/s, FFMA2 fp32 lanes/s, SM clock of the probes.
    R_mufu, R_fma = pk_meas["mufu_per_s"], pk_meas["ffma2_lanes_per_s"]
    clk_meas = pk_meas["sm_clock_mhz"] * 1e6
    plain = not (desc["gaussian"] or desc["gains"])

    def fixed_ceiling(kind, m_term):
        """The fixed ceiling of a plan TYPE (it does not move with any tuning knob): the best the instruction set of
        the method allows when the share f of terms whose sin/cos (forward: 2 MUFU, adjoint: 1) is evaluated by the
        FMA-pipe polynomial is free in [0, 1].  ex2 / rcp of Gaussian pixels stay on the MUFU pipe (moving them was
        measured slower).  Lane-ops per term are the SASS counts of DESIGN.md section 6 (the same constants as
        bound()); gains add their amortised product, the fp64-phase kernels add 4 FP64-pipe ops per term (3 DFMA + the
        magic-number DADD) against the DFMA rate measured in this run.  Returns (terms/s, binding pipe, f)."""
        gauss, gains_k = int(desc["gaussian"]), int(desc["gains"])
        movable = 1.0 if kind == "adj" else 2.0                 # MUFU per term that a polynomial can replace
        movable = min(movable, float(m_term))
        if kind == "adj":
            a_ = {0: 5.0, 1: 19.0, 2: 12.0}[gauss]
            b_ = a_ + 7.0                                       # cos polynomial instead of MUFU.COS: + 3 reduce + 4 Horner
            extra = {0: 0.0, 1: 10.0, 2: 1.5}[gains_k]
        else:
            a_ = {0: 6.0, 1: 20.0, 2: 13.0}[gauss]
            b_ = a_ + 12.0                                      # sincos polynomial: + 3 reduce + 5 sin + 4 cos
            extra = {0: 0.0, 1: 10.0, 2: 0.5}[gains_k]
        R_f64 = pk_meas.get("dfma_per_s") or SM_COUNT * 64.0 * clk_meas
        best, pipe, f_at = 0.0, "", 0.0
        for i in range(0, 257):
            f = i / 256.0
            mufu = m_term - movable * f
            t = {"mufu": mufu / R_mufu if mufu > 0 else 0.0, "fma": (a_ * (1.0 - f) + b_ * f + extra) / R_fma}
            if desc["phase_fp64"]:
                t["fp64"] = 4.0 / R_f64
            worst = max(t, key=t.get)
            if 1.0 / t[worst] > best:
                best, pipe, f_at = 1.0 / t[worst], worst, f
        return best, pipe, f_at

    def kernel_entry(kind, ms, per16, packed, name):
        """Roofline of one apply kernel on a DENSE image (every N_p x N_v term evaluated).
        own_mix: min(MUFU pipe, FMA pipe, issue slots) for the kernel's SASS instruction mix, with the measured
                 pipe rates -- moves with the polynomial share the kernel was tuned to (context);
        mufu_only: every term on the MUFU path, measured MUFU rate / MUFU per term (SURVEY.md 8(d) as written);
        best_split: the best ANY MUFU/FMA split of this instruction set allows: MUFU time = FMA time,
                 m (1-f)/R_mufu = (a (1-f) + b f)/R_fma, (m, a, b) = (2, 6, 18) forward, (1, 5, 12) one-cosine adjoint
                 -- the fixed hardware ceiling the headline frac is quoted against (delta pixels, unit gains)."""
        ach = n_terms / (ms * 1e-3)
        own, b_mufu, b_fma, b_issue = bound(kind, per16, packed, clk_meas)
        scale_m, scale_f = R_mufu / (SM_COUNT * MUFU_PER_SM_PER_CLK * clk_meas), R_fma / (SM_COUNT * 128.0 * clk_meas)
        own = min(b_mufu * scale_m, b_fma * scale_f, b_issue)
        m_term = desc["adj_mufu_per_term"] if kind == "adj" else desc["mufu_per_term_mufu_path"]
        mufu_only = R_mufu / m_term
        best, best_pipe, best_f = fixed_ceiling(kind, m_term)
        e = {"kernel": name, "ms": ms, "Tterm_per_s": ach / 1e12, "poly_per16": per16,
             "own_mix_bound": own / 1e12, "frac_vs_own_mix": ach / own,
             "mufu_only_bound": mufu_only / 1e12, "frac_vs_mufu_only": ach / mufu_only,
             "best_split_bound": best / 1e12, "frac_vs_best_split": ach / best,
             "best_split_binding_pipe": best_pipe, "best_split_poly_fraction": best_f,
             "own_mix_pipes": {"mufu": b_mufu * scale_m / 1e12, "fma": b_fma * scale_f / 1e12, "issue": b_issue / 1e12}}
        if plain and not desc["phase_fp64"]:
            # fourth denominator: what the kernel's OWN mix reaches in the co-issue micro-benchmark (MUFU beside a packed
            # FMA stream, sl1m_peaks.cu): measured MUFU results/s under co-issue / MUFU per term at the kernel's split
            co = pk_meas["coissue_adj_mufu_per_clk_sm" if (kind == "adj" and m_term == 1) else "coissue_mufu_per_clk_sm"]
            co_bound = co * SM_COUNT * clk_meas / (m_term * (1.0 - per16 / 16.0))
            e["coissue_bound"] = co_bound / 1e12
            e["frac_vs_coissue"] = ach / co_bound
        return e, ach, best

    def kname(kind):
        nm = "sl1m::adj_kernel" if kind == "adj" else "sl1m::fwd_kernel"
        if desc["phase_fp64"]:
            return nm + "_p64"
        if (desc["adj_packed_pairs"] if kind == "adj" else desc["fwd_packed_pairs"]):      # the packed R = 8 kernels
            if int(desc["gaussian"]) == 2:
                nm += "_gtx2"
            elif kind == "adj" and int(desc["gains"]) == 2:
                nm += "_g2x2"
            elif kind == "adj" and desc["adj_mufu_per_term"] == 1:
                nm += "_c1"
            else:
                nm += "_x2"
        return nm

    ent_f, ach_f, pk_f = kernel_entry("fwd", fwd_ms, desc["fwd_poly_per16"], desc["fwd_packed_pairs"], kname("fwd"))
    ent_a, ach_a, pk_a = kernel_entry("adj", adj_ms, desc["adj_poly_per16"], desc["adj_packed_pairs"], kname("adj"))
    # headline kernel: the one with the LARGER time on a dense image (stable run to run; both are first-class below)
    dom_is_adj = adj_ms > fwd_ms
    dom_e, achieved, peak = (ent_a, ach_a, pk_a) if dom_is_adj else (ent_f, ach_f, pk_f)
    traffic = NCU_DRAM_BYTES_PER_LAUNCH.get((args.config, "adj" if dom_is_adj else "fwd"))
    roof = {
        "bound": "alu", "kernel": dom_e["kernel"], "achieved": achieved / 1e12, "peak": peak / 1e12, "unit": "Tterm/s",
        "frac": achieved / peak, "traffic": traffic,
        "peak_basis": "fixed ceiling of the plan type: the best split of sin/cos between the MUFU pipe and an FMA-pipe "
                      "polynomial that the kernel's instruction set allows (ex2/rcp of Gaussian pixels stay on MUFU; gains add "
                      "their amortised product; fp64-phase kernels add 4 FP64-pipe ops per term), binding pipe "
                      f"'{dom_e['best_split_binding_pipe']}', from the MUFU, FFMA2 and DFMA rates measured in this run by "
                      "sl1m_measure_peaks (peak_measured); kernels.fwd / kernels.adj carry every denominator (own mix, MUFU "
                      "only, fixed ceiling, co-issue micro-benchmark) for both apply kernels",
        "peak_measured": pk_meas,
        "kernels": {"fwd": ent_f, "adj": ent_a},
        "traffic_basis": "dram__bytes_read.sum + dram__bytes_write.sum of one launch, ncu --set full "
                         "(profiles/, same kernel and workload; null = not captured); algorithmic bytes at config 5: ~30 MB in per apply "
                         "+ the split partials (37 x 3.25 MB forward, 15 x 4 MB adjoint, partly L2-resident)",
        "plan": desc,
        "note": "per-apply time = C-ABI call on a dense image (main kernel + O(N) epilogues, < 0.1 % of it); "
                "not an HBM-bound path: the matrix is generated, never read",
    }

    cpu = None
    if not args.no_cpu_baseline:
        cpu = _oracle_sample(wl, args.cpu_seconds)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}:{wl.name}" + (f" overrides={args.overrides}" if args.overrides else ""),
                   "n_pix": wl.n_pix, "n_vis": wl.n_vis,
                   "pixel_kind": ("gaussian-per-pixel-sigma" if args.jitter_sigma else "gaussian") if wl.sigma is not None else "delta",
                   "flags": {"dense_forward": args.dense_forward, "no_persistent": args.no_persistent,
                             "phase_fp64": args.phase_fp64},
                   "gains": wl.gains is not None, "lambda": lam, "L": L,
                   "l2_flush": "256 MiB device memset between timed steps",
                   "step": "one FISTA iteration via sl1m_fista_step(1): warm-up and timed steps are consecutive iterations "
                           "of one run from I_0 = 0 (momentum carried); per-apply timings use a dense image; the e2e leg "
                           "is sl1m_solve_host(n_iter=1, x0=previous image), which restarts the momentum on every call",
                   "parallelism": "replicas" if world > 1 else "single-gpu"},
        "iters_per_s": world * args.steps / (t_max * 1e-3),
        "terms": {"counted": "evaluated terms: N_v x (N_p for A^H + pixels with y_k != 0 for A)",
                  "zero_skip": skip, "fwd_active_fraction": sum(nnz_list) / len(nnz_list) / wl.n_pix,
                  "fwd_active_pixels_per_step": nnz_list,
                  "dense_equivalent_terms_per_s": aggregate_value(world, 2.0 * n_terms, args.steps, t_max)},
        "step_ms": step_ms, "plan_create_s": t_plan, "max_eig_s": t_eig, "n_pow": args.n_pow,
        "continuous_solve": {"call": f"sl1m_solve(n_iter={n_cont}) from I_0 = 0, trace on, CUDA events around the call",
                             "n_iter": n_cont, "ms_total": cont_ms, "ms_per_iter": cont_ms / n_cont,
                             "iters_per_s": 1e3 * n_cont / cont_ms,
                             "nnz_I_k": [int(v) for v in tr[:: max(1, n_cont // 50), 2]],
                             "image_bit_identical_to_stepped_run": cont_same if n_cont == args.warmup + args.steps else None},
        "dense_forward_step_ms": fwd_ms + adj_ms,
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
    ap.add_argument("--no-persistent", action="store_true", dest="no_persistent",
                    help="SL1M_NO_PERSISTENT: small problems keep the multi-launch loop (A/B of the persistent kernel)")
    ap.add_argument("--phase-fp64", action="store_true", dest="phase_fp64", help="SL1M_PHASE_FP64: the fp64-phase kernels")
    ap.add_argument("--jitter-sigma", action="store_true", dest="jitter_sigma",
                    help="Gaussian configs: multiply every sigma_k by a seeded U(0.7, 1.3) draw (per-pixel-sigma kernels)")
    ap.add_argument("--batch-stop", type=int, default=0, dest="batch_stop", metavar="C",
                    help="side measurement: C channels (uvw scaled 0.9..1.1) solved to --tol in one sl1m_solve_stop_batch call")
    ap.add_argument("--tol", type=float, default=1e-6)
    ap.add_argument("--max-iter", type=int, default=7000, dest="max_iter")
    ap.add_argument("--check-every", type=int, default=10, dest="check_every")
    ap.add_argument("--applies-only", action="store_true", dest="applies_only",
                    help="profiling aid: plan, one sparse forward, then 3 dense forwards and 3 adjoints; no solver, no bench line")
    ap.add_argument("--cont-iters", type=int, default=0, dest="cont_iters",
                    help="iterations of the continuous_solve leg (default: warmup + steps, the stepped run's length)")
    ap.add_argument("--override", action="append", default=[], metavar="KEY=VALUE",
                    help="workloads.make_workload override for side measurements, e.g. n_steps=2 (config 4 with 2 samples per "
                         "baseline: per-term gain kernels); the default line uses none")
    args = ap.parse_args()
    args.overrides = {k: (float(v) if "." in v else int(v)) for k, v in (o.split("=", 1) for o in args.override)}
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
