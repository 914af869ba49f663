#!/usr/bin/env python
"""bench.py -- likelihood evaluations per second on BASELINE.json's dense-contraction config.

One *step* = one pass of the whole hot path (coefficients -> reweighted MC spectrum -> response
fold -> Poisson -2lnL) over one batch of the config's scan points.  Headline workload: config 4
("cfg4_dense": 16384 recoil bins x 8192 reconstructed bins, 1.07 GB FP64 response, 65536 points),
the configuration the batched-throughput metric is quoted on.  The same JSON line also carries, inside
`roofline`, the other regimes of that config (single evaluation: HBM-bound; 2..64 points: the ridge) and a
short run of every other BASELINE config (`per_config`), each with its parity maxima against the CPU oracle.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config NAME]
                  [--scaling weak|strong] [--quick]

N > 1: one rank per GPU under torch.distributed.run (bench.py re-executes itself under it when it was
started as a plain process); the points are sharded, the tables replicated, there is no data-path
collective.  weak: every rank folds its own 65536-point batch; strong: one scan is split with
sharding.shard_range and the -2lnL slices are gathered.
`--impl reference` times the CPU oracle (oracle/) on the box's host cores -- a deliberately slow,
plain program; see DESIGN.md section 6.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "likelihood evals/sec (batched)"
UNIT = "evals/s"
L2_BYTES = 126e6

NCU_CSV = os.path.join("profiles", "r03_folds_raw.csv")
REGIME_POINTS = (2, 3, 8, 12, 16, 17, 24, 32, 33, 40, 48, 56, 64, 65, 72, 96, 127, 128, 192, 300)
DETAIL_FILE = "bench_detail.json"      # everything measured, prose included; the stdout line names it
LINE_LIMIT = 4096                      # bytes of the contract line (the driver keeps only a tail of stdout)


def load_ncu_traffic(path=None):
    """kernel -> dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed reduction of an
    `ncu --set full` capture of `bench.py --tour` on config 4 (profiles/r03_folds.md names the command).  NOT measured in
    this run: bench.py cannot run under ncu.  Of a kernel's captures inside plain rw_eval_batch calls (rows whose `call`
    names no flag), the longest one with a DRAM figure counts: the main launch of a chunk (ncu returned no counters for
    the 1.6 ms split-K tail launches of k_fold_gemm<8>).  Missing file or kernel: no traffic figure."""
    import csv
    path = path or os.path.join(ROOT, NCU_CSV)
    res, best = {}, {}
    if not os.path.exists(path):
        return res
    with open(path, newline="") as f:
        for row in csv.DictReader(f):
            call = row.get("call", "rw_eval_batch")
            if not call.startswith("rw_eval_batch") or "RW_" in call:
                continue
            try:
                t, tr = float(row["time_ms"]), float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
            except (KeyError, ValueError):
                continue
            if t >= best.get(row["kernel"], 0.0):
                best[row["kernel"]], res[row["kernel"]] = t, tr
    return res


NCU_TRAFFIC = load_ncu_traffic()


def _clean(x, digits=6):
    """JSON-safe copy: non-finite floats -> None, floats rounded to `digits` significant digits, numpy scalars unwrapped."""
    if isinstance(x, dict):
        return {str(k): _clean(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_clean(v, digits) for v in x]
    if isinstance(x, (bool, np.bool_)):
        return bool(x)
    if isinstance(x, (int, np.integer)):
        return int(x)
    if isinstance(x, (float, np.floating)):
        x = float(x)
        if x != x or x in (float("inf"), float("-inf")):
            return None
        return float("%.*g" % (digits, x))
    return x


def contract_line(full):
    """The ONE line the driver parses: built from the dict of everything measured (`full`, which goes to
    bench_detail.json as it is), numbers only, no prose, at most LINE_LIMIT bytes, strict JSON.
    roofline.regimes rows: [points, kernel, bound, ms_per_call, frac]; roofline.per_config values:
    [evals_per_s, bound, frac, single_eval_ms, mu_rel_max, m2lnl_err_over_bound_max, parity pass]."""
    def pick(d, keys):
        return {k: d.get(k) for k in keys if d is not None and k in d} if d else None

    line = {k: full.get(k) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                                      "higher_is_better", "scaling", "vs_baseline", "dtype", "data")}
    cfg = full.get("config") or {}
    line["config"] = dict(cfg)
    line["gpu_launches"] = full.get("gpu_launches")
    line["clocks"] = pick(full.get("clocks"), ("sm_mhz", "sm_max_mhz", "reasons"))
    line["e2e"] = pick(full.get("e2e"), ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step",
                                         "matches_device_path"))
    rf = full.get("roofline") or {}
    roof = pick(rf, ("bound", "kernel", "achieved", "peak", "unit", "frac", "call_frac", "traffic", "avg_launch_ms",
                     "launches_timed", "kernel_share_of_step", "ridge_points"))
    if rf.get("regimes"):
        roof["regimes"] = [[r.get("points"), r.get("kernel"), r.get("bound"), r.get("ms_per_call"), r.get("frac")]
                           for r in rf["regimes"]]
    if rf.get("per_config"):
        pc = {}
        for name, r in rf["per_config"].items():
            par = r.get("parity") or {}
            pc[name] = [r.get("evals_per_s"), r.get("bound"), r.get("frac"), r.get("single_eval_ms"),
                        par.get("mu_rel_max"), par.get("m2lnl_err_over_bound_max"), par.get("pass")] \
                if "unavailable" not in r else None
        roof["per_config"] = pc
    line["roofline"] = roof
    cpu = full.get("cpu_baseline")
    if cpu:
        line["cpu_baseline"] = pick(cpu, ("value", "unit", "cores", "kind", "sample"))
        if cpu.get("single_thread"):
            line["cpu_baseline"]["single_thread_value"] = cpu["single_thread"].get("value")
    else:
        line["cpu_baseline"] = None
    line["parity"] = pick(full.get("parity"), ("points", "mu_rel_max", "m2lnl_abs_max", "m2lnl_err_over_bound_max", "pass"))
    line["all_finite"] = full.get("all_finite")
    line["bench_wall_s"] = full.get("bench_wall_s")
    line["detail"] = full.get("detail")
    if full.get("errors"):
        line["errors"] = len(full["errors"])
    text = json.dumps(_clean(line, 7), allow_nan=False, separators=(",", ":"))
    if len(text) > LINE_LIMIT:                       # never let context take the contract down: drop it, largest first
        for key in ("regimes", "per_config"):
            if line["roofline"] and key in line["roofline"]:
                del line["roofline"][key]
                text = json.dumps(_clean(line, 7), allow_nan=False, separators=(",", ":"))
                if len(text) <= LINE_LIMIT:
                    break
    return text


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=p["hbm_gbs"], bf16=p["bf16_tflops"], bf16_sus=p.get("bf16_tflops_sustained"),
                    source="measured")
    return dict(hbm_gbs=6650.0, bf16=1590.0, bf16_sus=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        out = self.proc.communicate()[0]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def workload_config(name, inp, P, n_gpus, max_batch=0, scaling="weak"):
    """The `config` object of the line; both arms (ours and --impl reference) print exactly this."""
    D, n_T, n_rec = inp["R"].shape
    if scaling == "strong":
        par = "one scan split over %d GPU(s), tables replicated, -2lnL slices gathered" % n_gpus
    else:
        par = "points sharded over %d GPU(s), tables replicated, no collective" % n_gpus
    return {"workload": name, "n_E": int(inp["E"].size), "n_T": int(n_T), "n_rec": int(n_rec), "n_periods": int(D),
            "points_per_step_per_gpu": int(P), "response_bytes": int(D * n_T * n_rec * 8),
            "library_slice_points": int(max_batch) if max_batch else int(P), "parallelism": par,
            # working set beyond 2 x the 126 MB L2: nothing survives between steps, no flush needed; else a 256 MB buffer
            # is rewritten between timed steps
            "l2_flush": bool(D * n_T * n_rec * 8 + 8.0 * P * n_T <= 2 * L2_BYTES)}


def default_max_batch(name, P):
    return 16384 if name == "cfg5_joint6" else P            # BASELINE.json: config 5 is streamed in batches of 16384


def run_reference(args, rank, world):
    """CPU oracle arm: rank 0 alone works; each step folds a bounded sample of the config."""
    if rank != 0:
        return
    from oracle import rw_oracle as orc
    from paper_2607_00488_b200 import workloads as wl
    orc.build()
    cores = os.cpu_count() or 1
    name = args.config
    inp = wl.make(name)
    params, kinds = wl.scan_points(name)
    P = params.shape[0]
    n_sample = max(1, min(P, cores))                       # one point per core and step
    for w in range(args.warmup):
        orc.eval_batch(inp, params[:n_sample], kinds, nthreads=cores)
    t0 = time.perf_counter()
    for s in range(args.steps):
        lo = (s * n_sample) % max(1, P - n_sample + 1)
        orc.eval_batch(inp, params[lo:lo + n_sample], kinds, nthreads=cores)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = "%d scan points per step (of %d), OpenMP over points on %d threads" % (n_sample, P, cores)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": workload_config(name, inp, P, args.gpus, max_batch=default_max_batch(name, P), scaling=args.scaling),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(_clean(line, 9), allow_nan=False), flush=True)


# ------------------------------------------------------------------------------------------------ helpers (GPU arm)
class Timer:
    """Device timing with CUDA events on the current stream; an L2 flush (256 MB rewrite, untimed) before every
    timed call when the working set could stay in the 126 MB L2."""

    def __init__(self, torch, dev, need_flush):
        self.torch, self.need_flush = torch, need_flush
        self.e0, self.e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if need_flush else None

    def total_ms(self, fn, reps):
        t = self.torch
        t.cuda.synchronize()
        if not self.need_flush:
            self.e0.record()
            for _ in range(reps):
                fn()
            self.e1.record()
            t.cuda.synchronize()
            return self.e0.elapsed_time(self.e1)
        total = 0.0
        for _ in range(reps):
            self.flush_buf.zero_()
            self.e0.record()
            fn()
            self.e1.record()
            t.cuda.synchronize()
            total += self.e0.elapsed_time(self.e1)
        return total

    def per_call_ms(self, fn, reps, warm=2):
        for _ in range(warm):
            fn()
        return self.total_ms(fn, reps) / reps


def policy_kernel(P, inp=None):
    """The fold kernel RW_MODE_AUTO picks for a call of P points (label only; mirrors rw_api.cu).  With `inp` the label
    also names the ridge-kernel tail of a batch that is not a multiple of 128 points."""
    if P <= 1:
        return "k_fold_stream<1>"
    if P <= 64:
        return "k_fold_ridge<%d>" % ((P + 7) // 8)               # one instantiation per multiple of 8 points
    if inp is not None and 0 < P % 128 <= 96:           # fold_slice() in rw_api.cu: where the tail pays
        D, n_T, n_rec = inp["R"].shape
        if (P <= 16384 and n_T * n_rec >= 4e7) or (P <= 256 and n_T * n_rec * D >= 4e6):
            return ("k_fold_gemm<8>+" if P >= 128 else "") + "k_fold_ridge[last %d]" % (P % 128)
    return "k_fold_gemm<8>"


def parity_indices(name, P, max_batch, n):
    """Seeded oracle sample: batch / chunk edges plus random points (configs 1-2: every point)."""
    if name in ("cfg1_tiny_nsi", "cfg2_mm_lowE"):
        return np.arange(P)
    edges = {0, P - 1}
    for b in (max_batch, 32768):                                       # library slice and contraction chunk edges
        for q in (b - 1, b, (P // b) * b - 1, (P // b) * b):
            if 0 <= q < P:
                edges.add(int(q))
    rng = np.random.default_rng(20260705)
    extra = [int(x) for x in rng.choice(P, size=min(P, n), replace=False) if int(x) not in edges]
    idx = sorted(edges) + extra
    return np.array(sorted(idx[:max(n, len(edges))]))


def parity_block(orc, wl, torch, ctx, name, inp, params, kinds, out_scan, dev, max_batch, n_sample, cores):
    """Raw error maxima of the timed scan against the CPU oracle on a sample: -2lnL from the timed scan's own output,
    mu from 256-point RW_MODE_AUTO calls (the mode the scan ran in) that contain the sample points.
    Returns (dict, oracle seconds, points)."""
    P = params.shape[0]
    idx = parity_indices(name, P, max_batch, n_sample)
    t0 = time.perf_counter()
    ref, mu_ref, ab = orc.eval_batch(inp, params[idx], kinds, want_mu=True, want_abs=True, nthreads=cores)
    secs = time.perf_counter() - t0
    got = out_scan[idx]
    err = np.abs(got - ref)
    bound = 1e-9 + 1e-12 * ab
    mu_max, mu_pts = None, 0
    for lo in range(0, idx.size, 256):                                 # mu of the sample points, 256 at a time
        sel = idx[lo:lo + 256]
        pad = np.setdiff1d(np.arange(min(P, 512)), sel)[:max(0, min(P, 256) - sel.size)]
        batch = np.concatenate([sel, pad]).astype(np.int64)
        _, mu = ctx.eval_batch(torch.from_numpy(params[batch]).to(dev), kinds, want_mu=True, mode="auto")
        torch.cuda.synchronize()
        rel = np.abs(mu.cpu().numpy()[:sel.size] - mu_ref[lo:lo + sel.size]) / np.abs(mu_ref[lo:lo + sel.size])
        mu_max = float(rel.max()) if mu_max is None else max(mu_max, float(rel.max()))
        mu_pts += int(sel.size)
    res = {"points": int(idx.size), "mu_rel_max": mu_max, "mu_bar": 1e-12,
           "m2lnl_abs_max": float(err.max()), "m2lnl_bound_max": float(bound.max()),
           "m2lnl_err_over_bound_max": float((err / bound).max()), "m2lnl_rel_max": float((err / np.abs(ref)).max()),
           "m2lnl_abs_ref_max": float(np.abs(ref).max()),
           "pure_1e-9_met": bool(err.max() <= 1e-9),
           "bar": "|d(-2lnL)| <= 1e-9 + 1e-12 * sum_k 2|term_k| (DESIGN.md reading T); mu 1e-12 relative",
           "pass": bool(np.all(err <= bound) and mu_max <= 1e-12),
           "source": "-2lnL: the timed scan's own output at the sampled indices; mu: 256-point calls of the same "
                     "kernel family containing them; oracle = oracle/rw_oracle.c (long double)"}
    return res, secs, int(idx.size)


def single_eval_block(torch, ctx, timer, param_dev, kinds, dev, r_bytes, peaks, reps=30):
    """P = 1: ms per evaluation (call level), kernel time from the library's event hooks, CUDA-graph replay."""
    one = param_dev[:1].contiguous()
    out1 = torch.empty(1, dtype=torch.float64, device=dev)
    fn = lambda: ctx.eval_batch(one, kinds, out=out1)                   # RW_MODE_AUTO: the one-launch streaming kernel
    for _ in range(5):
        fn()
    ms = timer.total_ms(fn, reps) / reps                               # call level: without the library's event hooks
    ctx.profile_begin()                                                 # (they cost ~5 us per call on the stream)
    timer.total_ms(fn, reps)
    k_ms, k_n = ctx.profile_end()
    k_ms = k_ms / max(1, k_n)
    graph_us = None
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fn()
        graph_us = timer.per_call_ms(g.replay, reps, warm=5) * 1e3
    except Exception as exc:                                  # capture is a convenience, not part of the metric
        graph_us = "unavailable: %s" % str(exc)[:80]
    cold = r_bytes > 2 * L2_BYTES or timer.need_flush
    blk = {"regime": "single_eval", "points": 1, "kernel": "k_fold_stream<1>", "ms_per_call": ms,
           "avg_launch_ms": k_ms, "graph_replay_us_per_eval": graph_us, "algorithmic_bytes": int(r_bytes),
           "achieved_gbs": r_bytes / (k_ms * 1e-3) / 1e9, "peak_gbs": peaks["hbm_gbs"],
           "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peaks["source"]}
    if r_bytes > 2 * L2_BYTES:
        blk["bound"] = "hbm"
        blk["frac"] = blk["achieved_gbs"] / peaks["hbm_gbs"]
        blk["call_frac"] = r_bytes / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"]
        blk["note"] = ("one launch does a1-a4; R (%.2f GB) >> L2, every evaluation reads it from HBM once; kernel time "
                       "includes the last-CTA reduction; call_frac divides by the call-level time" % (r_bytes / 1e9))
        tr = NCU_TRAFFIC.get("k_fold_stream<1>")
        if tr and r_bytes == 1073741824:
            blk["traffic"], blk["traffic_source"] = tr, NCU_CSV + " (ncu capture, not measured in this run)"
    else:
        blk["bound"] = "l2/latency"
        blk["frac"] = None
        blk["note"] = ("R (%.1f MB) fits the 126 MB L2; L2 flushed before every timed call (%s), so achieved_gbs is a "
                       "cold read, launch-latency dominated: no HBM fraction is claimed" % (r_bytes / 1e6, cold))
    return blk


def fold_flops(inp, P):
    D, n_T, n_rec = inp["R"].shape
    return 2.0 * n_T * n_rec * D * P


def ridge_regimes(torch, ctx, timer, param_dev, kinds, dev, inp, peaks, dmma_peak, P_list):
    """2..64 points per call: the regime around the ridge P* = 4 F / BW of the roofline.  bound_ms = max(R bytes / HBM
    peak, 2 N_T N_rec P / DMMA peak); frac = bound_ms / call-level ms (the stricter reading), kernel_frac = the same
    with the fold kernel's own time."""
    D, n_T, n_rec = inp["R"].shape
    r_bytes = D * n_T * n_rec * 8
    res = []
    for Pb in P_list:
        if Pb > param_dev.shape[0]:
            break
        pb = param_dev[:Pb].contiguous()
        ob = torch.empty(Pb, dtype=torch.float64, device=dev)
        fn = lambda: ctx.eval_batch(pb, kinds, out=ob)
        for _ in range(3):
            fn()
        ms = timer.total_ms(fn, 20) / 20                                # call level: without the library's event hooks
        ctx.profile_begin()
        timer.total_ms(fn, 20)
        k_ms, k_n = ctx.profile_end()
        k_ms = k_ms / 20                                               # all fold launches of one call
        hbm_ms = r_bytes / (peaks["hbm_gbs"] * 1e9) * 1e3
        ten_ms = fold_flops(inp, Pb) / (dmma_peak * 1e12) * 1e3
        bound_ms = max(hbm_ms, ten_ms)
        blk = {"regime": "ridge" if Pb <= 64 else "small batch", "points": Pb, "kernel": policy_kernel(Pb, inp),
               "bound": "hbm" if hbm_ms >= ten_ms else "tensor", "bound_ms": bound_ms, "ms_per_call": ms,
               "fold_kernel_ms": k_ms, "frac": bound_ms / ms, "kernel_frac": bound_ms / k_ms if k_ms > 0 else None,
               "evals_per_s": Pb / ms * 1e3, "fold_tflops": fold_flops(inp, Pb) / ms / 1e9,
               "response_gbs": r_bytes / ms / 1e6}
        tr = NCU_TRAFFIC.get(blk["kernel"])
        if tr and r_bytes == 1073741824:
            blk["traffic"], blk["traffic_source"] = tr, NCU_CSV + " (ncu capture, not measured in this run)"
        res.append(blk)
    return res


def bench_config(name, dev, steps, warmup, peaks, dmma_peak, cores, quick):
    """A short run of one BASELINE config: batched scan (device-resident and host-buffer e2e), fold-kernel roofline,
    single evaluation, parity maxima.  Used for the configs that are not the headline."""
    import torch
    from oracle import rw_oracle as orc
    from paper_2607_00488_b200 import binding, workloads as wl
    inp = wl.make(name)
    D, n_T, n_rec = inp["R"].shape
    params, kinds = wl.scan_points(name)
    P, k = params.shape
    max_batch = default_max_batch(name, P)
    r_bytes = D * n_T * n_rec * 8
    dev_inp = {key: torch.from_numpy(np.ascontiguousarray(inp[key])).to(dev)
               for key in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev_inp["f_tau"] = inp["f_tau"]
    ctx = binding.Reweighter(dev_inp, max_batch=max_batch, device=dev)
    param_dev = torch.from_numpy(params).to(dev)
    out_dev = torch.empty(P, dtype=torch.float64, device=dev)
    param_pin = torch.from_numpy(params).pin_memory()
    out_pin = torch.empty(P, dtype=torch.float64).pin_memory()
    need_flush = r_bytes + 8.0 * min(P, max_batch) * n_T <= 2 * L2_BYTES
    timer = Timer(torch, dev, need_flush)
    scan = lambda: ctx.eval_batch(param_dev, kinds, out=out_dev)
    big = P * n_T * n_rec * D > 2e15                                   # config 5: a scan takes seconds
    n_warm = 1 if big else warmup
    n_steps = 1 if big else steps
    if big:                                                            # warm up on three library slices only
        ctx.eval_batch(param_dev[:3 * max_batch].contiguous(), kinds)
    else:
        for _ in range(n_warm):
            scan()
    launches0 = ctx.launch_count()
    ctx.profile_begin()
    ms = timer.total_ms(scan, n_steps) / n_steps
    fold_ms, fold_n = ctx.profile_end()
    launches = (ctx.launch_count() - launches0) // n_steps
    ms_e2e, same = None, None
    if not big:                                                        # (config 5: one timed scan only, a scan takes seconds)
        ctx.eval_batch(param_pin, kinds, out=out_pin)
        ms_e2e = timer.total_ms(lambda: ctx.eval_batch(param_pin, kinds, out=out_pin), n_steps) / n_steps
        torch.cuda.synchronize()
        same = bool(np.array_equal(out_pin.numpy(), out_dev.cpu().numpy()))
    achieved = fold_flops(inp, P) * n_steps / (fold_ms * 1e-3) / 1e12
    launch_bound = fold_flops(inp, P) < 5e10                            # < ~1.5 us of DMMA work per SM
    res = {"points": P, "k": k, "n_T": n_T, "n_rec": n_rec, "n_periods": D, "response_bytes": int(r_bytes),
           "library_slice_points": int(max_batch), "steps": n_steps, "warmup": "3 library slices" if big else n_warm,
           "evals_per_s": P / ms * 1e3, "ms_per_scan": ms, "e2e_evals_per_s": P / ms_e2e * 1e3 if ms_e2e else None, "e2e_ms_per_scan": ms_e2e,
           "e2e_h2d_bytes": int(P * k * 8), "e2e_d2h_bytes": int(P * 8), "e2e_matches_device_path": same,
           "gpu_launches_per_scan": int(launches), "l2_flush_between_steps": bool(need_flush),
           "dominant_kernel": policy_kernel(min(P, max_batch)), "fold_launches_per_scan": int(fold_n // n_steps),
           "fold_kernel_share_of_scan": fold_ms / n_steps / ms, "achieved": achieved, "peak": dmma_peak, "unit": "TFLOP/s"}
    if launch_bound:
        res["bound"] = "launch"
        res["frac"] = None
        res["note"] = ("%.1e flop per scan is microseconds of tensor work: the scan is bound by its %d kernel launches; "
                       "no roofline fraction is claimed" % (fold_flops(inp, P), launches))
        try:                                   # the same scan replayed from a CUDA graph: launch gaps gone, kernels remain
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                scan()
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                scan()
            g_ms = timer.per_call_ms(g.replay, 20, warm=5)
            res["graph_replay_ms_per_scan"] = g_ms
            res["graph_replay_evals_per_s"] = P / g_ms * 1e3
            res["graph_replay_call_frac"] = fold_flops(inp, P) / (g_ms * 1e-3) / 1e12 / dmma_peak
        except Exception as exc:               # noqa: BLE001
            res["graph_replay_ms_per_scan"] = "unavailable: %s" % str(exc)[:80]
    else:
        res["bound"] = "tensor"
        res["frac"] = achieved / dmma_peak
        res["call_frac"] = fold_flops(inp, P) / (ms * 1e-3) / 1e12 / dmma_peak
        if need_flush:
            res["note"] = "R fits the L2 (flushed between steps); the fold kernel is timed by events inside the library"
    res["single_eval"] = single_eval_block(torch, ctx, timer, param_dev, kinds, dev, r_bytes, peaks, reps=10 if quick else 30)
    res["single_eval_ms"] = res["single_eval"]["ms_per_call"]
    n_par = {"cfg3_nsi4": 32, "cfg5_joint6": 16}.get(name, 16)
    res["parity"], _, _ = parity_block(orc, wl, torch, ctx, name, inp, params, kinds, out_dev.cpu().numpy(), dev,
                                       max_batch, n_par, cores)
    ctx.close()
    del dev_inp, param_dev
    torch.cuda.empty_cache()
    return res


def kernel_tour(torch, ctx, param_dev, kinds, inp, dev, max_batch):
    """Two calls (the first warms caches, clocks and lazily loaded modules) of every regime and entry point on the
    context the bench times: the launches an `ncu --set full -k regex:...` capture picks from.  Nothing is timed."""
    P, k = param_dev.shape
    calls = []

    def twice(label, fn):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        calls.append(label)

    for Pb in (1, 2, 8, 16, 32, 64):
        pb = param_dev[:Pb].contiguous()
        twice("rw_eval_batch P=%d auto -> %s" % (Pb, policy_kernel(Pb)), lambda: ctx.eval_batch(pb, kinds))
    twice("rw_eval_batch P=%d auto -> %s" % (P, policy_kernel(min(P, max_batch))), lambda: ctx.eval_batch(param_dev, kinds))
    twice("rw_eval_batch P=%d RW_SLICED -> k_slice_A + k_fold_i8" % P, lambda: ctx.eval_batch(param_dev, kinds, sliced=True))
    twice("rw_eval_batch P=%d RW_SLICED_FAST" % P, lambda: ctx.eval_batch(param_dev, kinds, sliced="fast"))
    twice("rw_eval_batch P=%d RW_MODE_COLLAPSED -> k_collapsed" % P, lambda: ctx.eval_batch(param_dev, kinds, mode="collapsed"))
    Pp = int(min(P, max_batch, 4096))
    pp = param_dev[:Pp].contiguous()
    twice("rw_eval_profile P=%d -> fold + k_profile" % Pp, lambda: ctx.eval_profile(pp, kinds, s0=1.0, sigma=0.05))
    Pg = int(min(P, max(1, min(max_batch, 4096) // (1 + k))))
    pg = param_dev[:Pg].contiguous()
    twice("rw_eval_grad P=%d -> k_coef_grad + fold + k_grad" % Pg, lambda: ctx.eval_grad(pg, kinds))
    if all(int(x) < 7 for x in kinds):
        Pe = int(min(P, max_batch, 1024))
        pe = param_dev[:Pe].contiguous()
        tab = torch.from_numpy(np.ascontiguousarray(inp["P_e"])).to(dev)[None, :].repeat(Pe, 1).contiguous()
        twice("rw_eval_pee P=%d n_E=%d -> k_pee_scan + fold" % (Pe, tab.shape[1]), lambda: ctx.eval_pee(pe, kinds, tab))
    return calls


def self_launch(args):
    """Started as a plain process with --gpus N > 1: re-execute under torch.distributed.run, one rank per GPU."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")            # NCCL_DEBUG=INFO from the caller is passed through (communicator lines)
    raise SystemExit(subprocess.call(cmd, env=env))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4_dense")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tour", action="store_true",
                    help="no timing: two calls of every entry point / regime on the bench context, for `ncu -k ...` captures "
                         "(profiles/*.md name the command); prints the list of calls")
    ap.add_argument("--quick", action="store_true", help="headline, e2e and rooflines only: no other configs")
    ap.add_argument("--full", action="store_true",
                    help="also time the opt-in legs (batch sweep, collapsed, FP32, sliced + certificate, profile / gradient / P_ee, "
                         "library DGEMM); they go to bench_detail.json only, never into the stdout line")
    ap.add_argument("--detail", default=DETAIL_FILE, help="where everything measured is written (JSON, relative to the repo root)")
    ap.add_argument("--max-batch", type=int, default=0,
                    help="points per library slice (default: the whole scan; 16384 for cfg5_joint6, as BASELINE.json says)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        self_launch(args)

    import torch
    import torch.distributed as dist
    from paper_2607_00488_b200 import binding, probe, sharding, workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d has no GPU (%d visible)" % (local_rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    binding.load_library()
    t_start = time.perf_counter()
    name = args.config
    inp = wl.make(name)
    D, n_T, n_rec = inp["R"].shape
    strong = args.scaling == "strong" and world > 1
    if strong:
        params_all, kinds = wl.scan_points(name)
        lo, hi = sharding.shard_range(params_all.shape[0], rank, world)
        params = np.ascontiguousarray(params_all[lo:hi])
        P_job = params_all.shape[0]
    else:
        params, kinds = sharding.rank_points(name, rank)
        P_job = params.shape[0] * world
    P, k = params.shape
    lite = args.quick or world > 1          # multi-rank runs time the headline and e2e legs only
    extras = (args.full or args.tour) and not lite         # opt-in legs (sliced / fp32 / collapsed / profile / gradient / P_ee / DGEMM): detail file only

    # tables resident in HBM before anything is timed (R is borrowed by the context, not copied)
    dev_inp = {key: torch.from_numpy(np.ascontiguousarray(inp[key])).to(dev)
               for key in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev_inp["f_tau"] = inp["f_tau"]
    max_batch = args.max_batch or default_max_batch(name, params.shape[0] if not strong else P_job)
    max_batch = min(max_batch, max(P, 1))
    ctx = binding.Reweighter(dev_inp, max_batch=max_batch, device=dev, fp32=extras, sliced=extras)   # + operand copies for the opt-in legs
    param_dev = torch.from_numpy(params).to(dev)
    out_dev = torch.empty(P, dtype=torch.float64, device=dev)
    param_pin = torch.from_numpy(params).pin_memory()
    out_pin = torch.empty(P, dtype=torch.float64).pin_memory()
    peaks = load_peaks()
    r_bytes = D * n_T * n_rec * 8
    if args.tour:
        assert world == 1, "--tour is a single-GPU profiling aid"
        calls = kernel_tour(torch, ctx, param_dev, kinds, inp, dev, max_batch)
        print(json.dumps({"tour": calls, "config": name, "launches": int(ctx.launch_count())}))
        ctx.close()
        return

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def maxreduce(x):
        return sharding.max_over_ranks(x, dev, world)

    dmma_peak0 = probe.fp64_peak(1)
    dfma_peak0 = probe.fp64_peak(0)

    gathered = None
    if strong:
        shard_max = sharding.shard_pad(P_job, world)
        pad = torch.zeros(shard_max, dtype=torch.float64, device=dev)
        gathered = torch.empty(world * shard_max, dtype=torch.float64, device=dev)

    def step_dev():
        ctx.eval_batch(param_dev, kinds, out=out_dev)
        if strong:                            # the caller wants the whole scan: gather the slices (8 P_job bytes)
            sharding.gather_shards(out_dev, pad, gathered, P_job, world)

    def step_host():
        ctx.eval_batch(param_pin, kinds, out=out_pin)

    # ---------------------------------------------------------------- device-resident throughput
    for _ in range(args.warmup):
        step_dev()
    barrier()
    sampler = ClockSampler("GPU-" + str(torch.cuda.get_device_properties(dev).uuid))
    if rank == 0:
        sampler.start()
    need_flush = r_bytes + 8.0 * min(P, max_batch) * n_T <= 2 * L2_BYTES      # working set could stay in the 126 MB L2
    timer = Timer(torch, dev, need_flush)
    launches0 = ctx.launch_count()
    ctx.profile_begin()
    barrier()
    ms = maxreduce(timer.total_ms(step_dev, args.steps))
    barrier()
    fold_ms, fold_launches = ctx.profile_end()
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    value = P_job * args.steps / (ms * 1e-3)
    finite = bool(torch.isfinite(out_dev).all().item())

    # ---------------------------------------------------------------- end to end with host buffers
    for _ in range(2):
        step_host()
    barrier()
    # H2D params, kernels, D2H -2lnL: all on the stream, inside the timed region
    ms_e2e = maxreduce(timer.total_ms(step_host, args.steps))
    barrier()
    e2e_value = P_job * args.steps / (ms_e2e * 1e-3)
    same = bool(np.array_equal(out_pin.numpy(), out_dev.cpu().numpy()))
    out_scan = out_dev.cpu().numpy()

    # everything measured goes into `full` (-> bench_detail.json); the stdout line is contract_line(full).  From here on
    # no leg may take the line down: each runs under guard() and a failure is recorded in full["errors"].
    sec = {"headline+e2e": time.perf_counter() - t_start}
    full = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(name, inp, P_job if strong else P, world,
                                      max_batch=default_max_batch(name, P_job if strong else P),
                                      scaling="strong" if strong else "weak"),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(P * k * 8),
                    "d2h_bytes_per_step": int(P * 8), "ms_per_step": ms_e2e / args.steps, "matches_device_path": same},
            "gpu_launches": int(launches), "clocks": clocks, "all_finite": finite, "errors": [],
            "detail": args.detail if rank == 0 else None, "section_wall_s": sec}
    if rank == 0:       # insurance for a human reader if a later leg hangs: the headline so far, on stderr (stdout carries ONE line)
        sys.stderr.write("bench.py headline so far: " + contract_line(full) + "\n")
        sys.stderr.flush()

    def guard(label, fn):
        t0 = time.perf_counter()
        try:
            return fn()
        except Exception as exc:               # noqa: BLE001
            full["errors"].append("%s: %s" % (label, str(exc)[:200]))
            return None
        finally:
            sec[label] = time.perf_counter() - t0

    # ---------------------------------------------------------------- roofline of the dominant kernel + the other regimes
    def tprobe(kind, prev):
        return max(prev, probe.fp64_peak(kind))
    dmma_peak = tprobe(1, dmma_peak0)
    dfma_peak = tprobe(0, dfma_peak0)
    flops_timed = fold_flops(inp, P) * args.steps              # algorithmic: 2 N_T N_rec per point and period
    achieved = flops_timed / (fold_ms * 1e-3) / 1e12
    dom = policy_kernel(min(P, max_batch))
    tr = NCU_TRAFFIC.get(dom) if name == "cfg4_dense" else None
    roofline = {"bound": "tensor", "kernel": dom, "achieved": achieved, "peak": dmma_peak, "unit": "TFLOP/s",
                "frac": achieved / dmma_peak, "traffic": tr,
                "traffic_source": (NCU_CSV + " (ncu --set full capture of this kernel on this workload; not measured in this run)") if tr else None,
                "peak_source": "FP64 DMMA.8x8x4 issue-rate probe measured live (librw_probe.so); DFMA probe %.2f; "
                               "bf16 %s peak x nominal FP64/bf16 ratio (45/2250) = %.1f burst / %.1f sustained"
                               % (dfma_peak, peaks["source"], peaks["bf16"] * 0.02, (peaks["bf16_sus"] or 0) * 0.02),
                "launches_timed": int(fold_launches), "avg_launch_ms": fold_ms / max(1, fold_launches),
                "flops_per_launch": flops_timed / max(1, fold_launches),
                "kernel_share_of_step": fold_ms / ms,
                "call_frac": flops_timed / (ms * 1e-3) / 1e12 / dmma_peak,
                "ridge_points": 4.0 * dmma_peak * 1e12 / (peaks["hbm_gbs"] * 1e9)}
    full["roofline"] = roofline
    single = None
    if rank == 0 and world == 1:
        single = guard("single_eval", lambda: single_eval_block(torch, ctx, timer, param_dev, kinds, dev, r_bytes, peaks))
        regimes = [single] if single else []
        regimes += guard("regimes", lambda: ridge_regimes(torch, ctx, timer, param_dev, kinds, dev, inp, peaks, dmma_peak,
                                                          REGIME_POINTS)) or []
        regimes.append({"regime": "batched", "points": P, "kernel": dom, "bound": "tensor", "achieved_tflops": achieved,
                        "peak_tflops": dmma_peak, "frac": achieved / dmma_peak, "avg_launch_ms": roofline["avg_launch_ms"],
                        "flops_per_launch": roofline["flops_per_launch"], "ms_per_call": ms / args.steps})
        roofline["regimes"] = regimes

    # ---------------------------------------------------------------- parity maxima + CPU oracle beside it
    cores = os.cpu_count() or 1
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        def cpu_leg():
            from oracle import rw_oracle as orc
            orc.build()
            n_par = min(P, 2 * cores)
            parity, secs, n_done = parity_block(orc, wl, torch, ctx, name, inp, params, kinds, out_scan, dev, max_batch,
                                                n_par, cores)
            full["parity"] = parity
            cpu = {"value": n_done / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": "%d of %d scan points, %d threads, %.1f s" % (n_done, P, cores, secs),
                   "sample_detail": "the parity sample (slice/chunk edges + seeded draws), OpenMP over points, mu and "
                                    "conditioning scale returned"}
            full["cpu_baseline"] = cpu
            n1 = 1 if fold_flops(inp, 1) > 1e8 else min(P, 64)
            t0 = time.perf_counter()
            orc.eval_batch(inp, params[:n1], kinds, nthreads=1)
            s1 = time.perf_counter() - t0
            cpu["single_thread"] = {"value": n1 / s1, "unit": UNIT, "cores": 1,
                                    "sample": "first %d scan points on one thread, %.1f s wall" % (n1, s1)}
        guard("parity+cpu_baseline", cpu_leg)

    # ---------------------------------------------------------------- other regimes of the same path (context lines)
    def timed(fn, reps):
        return timer.per_call_ms(fn, reps)

    sweep, collapsed, fp32_leg, sliced_leg, next_rows, lib_dgemm = None, None, None, None, None, None
    t_extras = time.perf_counter()
    if extras:
        sweep = []
        for Pb in (1, 4, 16, 64, 192, 256, 300, 2048):
            if Pb > P:
                break
            pb = param_dev[:Pb].contiguous()
            ob = torch.empty(Pb, dtype=torch.float64, device=dev)
            t = timed(lambda: ctx.eval_batch(pb, kinds, out=ob), 20 if Pb <= 256 else 5)
            sweep.append({"points": Pb, "ms_per_call": t, "evals_per_s": Pb / t * 1e3, "kernel": policy_kernel(Pb, inp),
                          "fold_tflops": fold_flops(inp, Pb) / t / 1e9, "response_gbs": r_bytes / t / 1e6})
        # opt-in rank-K collapsed mode: exact, O(11 n_rec) per point, FP64-ALU bound; never mixed into `value`
        out_c = torch.empty(P, dtype=torch.float64, device=dev)
        t_c = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_c, mode="collapsed"), 5)
        dmax = float((out_c - out_dev).abs().max().item())
        collapsed = {"ms_per_call": t_c, "evals_per_s": P / t_c * 1e3, "bound": "alu",
                     "algorithmic_gflops": 2.0 * 11 * n_rec * D * P / t_c / 1e6,
                     "max_abs_diff_vs_dense_fold": dmax,
                     "note": "2*11*n_rec*D flop per point plus one log1p per bin (FP64 ALU)"}

        # opt-in RW_FP32 contraction: 1e-5 relative on mu; never mixed into `value`
        try:                                   # a context leg must never take the bench line down with it
            if P > 4:
                out_f = torch.empty(P, dtype=torch.float64, device=dev)
                t_f = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_f, fp32=True), 5)
                ns = min(P, 128)
                # accuracy of the contraction RW_FP32 runs (top four slices) WITHOUT the strict recomputation: with mu asked
                # for, a chunk holding one uncertified point is recomputed wholly in FP64 and the comparison would be
                # FP64 against FP64 (round 2's 0.0)
                _, mu32 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm", sliced="fast")
                _, mu64 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm")
                rel = ((mu32 - mu64).abs() / mu64.abs())
                fp32_leg = {"ms_per_call": t_f, "evals_per_s": P / t_f * 1e3,
                            "what": "RW_FP32 = RW_SLICED_FAST | RW_SLICED_STRICT at 1e-5 (one stream synchronisation per chunk; "
                                    "the TF32 x 3 kernel of round 1 is gone: slower and less accurate than this)",
                            "strict_fallback_points": ctx.strict_fallback_count(),
                            "effective_fold_tflops": fold_flops(inp, P) / t_f / 1e9,
                            "mu_rel_err_vs_fp64_max": float(rel.max().item()), "mu_rel_err_vs_fp64_mean": float(rel.mean().item()),
                            "mu_rel_err_of": "the fast sliced contraction itself (RW_SLICED_FAST, no strict recomputation), %d points" % ns}
        except Exception as exc:               # noqa: BLE001
            fp32_leg = {"unavailable": str(exc)[:160]}

        # opt-in RW_SLICED contraction: FP64 by slicing on the INT8 tensor cores, exact int32 accumulation,
        # same 1e-12 bar as the DMMA path; a context line, never mixed into `value`
        try:
            if P > 4:
                out_s = torch.empty(P, dtype=torch.float64, device=dev)
                ctx.profile_begin()
                t_s = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_s, sliced=True), 5)
                k_ms, k_n = ctx.profile_end()
                ns = min(P, 128)
                _, mu8 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm", sliced=True)
                _, mu64 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm")
                rel = ((mu8 - mu64).abs() / mu64.abs())
                # RW_SLICED_FAST: the top four slices of the same operands (10 products), the FP32 bar
                out_f = torch.empty(P, dtype=torch.float64, device=dev)
                t_f = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_f, sliced="fast"), 5)
                _, muf = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm", sliced="fast")
                relf = ((muf - mu64).abs() / mu64.abs())
                fast_leg = {"ms_per_call": t_f, "evals_per_s": P / t_f * 1e3,
                            "effective_fold_tflops": fold_flops(inp, P) / t_f / 1e9,
                            "mu_rel_err_vs_fp64_max": float(relf.max().item()), "int8_products_per_k_step": 10}
                # certificate: rigorous per-point bound on max_k |mu~ - mu| / mu, and the strict call that enforces the bar
                _, bnd = ctx.eval_certified(param_dev, kinds, sliced=True)
                _, bnd_f = ctx.eval_certified(param_dev, kinds, sliced="fast")
                fb0 = ctx.strict_fallback_count()
                out_st = torch.empty(P, dtype=torch.float64, device=dev)
                t_st = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_st, sliced="strict"), 3)
                fb_calls = 5                                                # timed(): 2 warm-up + 3 timed calls
                cert = {"bound_max": float(bnd.max().item()), "bound_median": float(bnd.median().item()),
                        "points_over_1e-12": int((bnd > 1e-12).sum().item()), "points": P,
                        "fast_bound_max": float(bnd_f.max().item()), "fast_points_over_1e-5": int((bnd_f > 1e-5).sum().item()),
                        "strict_ms_per_call": t_st, "strict_evals_per_s": P / t_st * 1e3,
                        "strict_fallback_points_per_call": (ctx.strict_fallback_count() - fb0) / fb_calls,
                        "strict_max_abs_diff_m2lnL_vs_dmma": float((out_st - out_dev).abs().max().item()),
                        "note": "rw_eval_certified; strict = RW_SLICED | RW_SLICED_STRICT: points over the bar are recomputed by the DMMA path"}
                n_sl = 8 if n_T <= 2048 else 7                              # balanced 8-bit slices per operand (rw_fold_i8.cu)
                n_prod = n_sl * (n_sl + 1) // 2
                sliced_leg = {"ms_per_call": t_s, "evals_per_s": P / t_s * 1e3, "bound": "tensor (int8)",
                              "effective_fold_tflops": fold_flops(inp, P) / t_s / 1e9,
                              "kernel_effective_fold_tflops": fold_flops(inp, P) * 7 / (k_ms * 1e-3) / 1e12 if k_ms > 0 else None,
                              "executed_int8_tops": n_prod * fold_flops(inp, P) / t_s / 1e9,
                              "mu_rel_diff_vs_dmma_max": float(rel.max().item()),
                              "max_abs_diff_m2lnL_vs_dmma": float((out_s - out_dev).abs().max().item()),
                              "slices": n_sl, "int8_products_per_k_step": n_prod, "fast": fast_leg, "certificate": cert,
                              "note": "%d balanced 8-bit slices per operand, %d tcgen05.mma.kind::i8 products per k-step with exact "
                                      "int32 accumulation in TMEM; FP64 DMMA peak is %.1f TFLOP/s" % (n_sl, n_prod, dmma_peak)}
        except Exception as exc:               # noqa: BLE001
            sliced_leg = {"unavailable": str(exc)[:160]}

        # the other entry points of the same path, timed on a slice of the same scan: context only
        try:
            if P > 4:
                kin = [int(x) for x in kinds]
                nr = {}
                Pp = int(min(P, max_batch, 4096))
                pp = param_dev[:Pp].contiguous()
                t = timed(lambda: ctx.eval_profile(pp, kinds, s0=1.0, sigma=0.05), 3)
                nr["profile"] = {"points": Pp, "ms_per_call": t, "evals_per_s": Pp / t * 1e3,
                                 "note": "rw_eval_profile: fold with mu to a scratch + Newton per point (k_profile)"}
                Pg = int(min(P, max(1, min(max_batch, 4096) // (1 + k))))
                pg = param_dev[:Pg].contiguous()
                t = timed(lambda: ctx.eval_grad(pg, kinds), 3)
                nr["gradient"] = {"points": Pg, "fold_rows": Pg * (1 + k), "ms_per_call": t, "evals_per_s": Pg / t * 1e3,
                                  "note": "rw_eval_grad: 1 + k fold rows per point, then k_grad"}
                t = timed(lambda: ctx.eval_grad(param_dev[:1].contiguous(), kinds), 10)
                nr["gradient_single_point"] = {"fold_rows": 1 + k, "ms_per_call": t,
                                               "note": "a minimiser's call: value + %d derivative rows in one %s launch" % (k, policy_kernel(1 + k))}
                if all(x < 7 for x in kin) and "P_mu" not in inp and int(inp.get("n_comp", 1) or 1) == 1:
                    Pe = int(min(P, max_batch, 1024))
                    pe = param_dev[:Pe].contiguous()
                    tab = torch.from_numpy(np.ascontiguousarray(inp["P_e"])).to(dev)[None, :].repeat(Pe, 1).contiguous()
                    t = timed(lambda: ctx.eval_pee(pe, kinds, tab), 3)
                    nr["per_point_pee"] = {"points": Pe, "n_E": int(tab.shape[1]), "ms_per_call": t, "evals_per_s": Pe / t * 1e3,
                                           "note": "rw_eval_pee: spectrum on the (E x T) grid per point, then the dense fold"}
                next_rows = nr
        except Exception as exc:                   # noqa: BLE001
            next_rows = {"unavailable": str(exc)[:160]}

        # library DGEMM of the shape of one chunk of the fold (cuBLAS FP64 as a reference point for the
        # denominator).  Context only: no N' generation, no Poisson epilogue, no reduction, and mu goes to HBM.
        if P > 4:
            Pl = int(min(P, max_batch, 32768))
            try:
                gen = torch.Generator(device=dev).manual_seed(7)
                A_l = torch.rand((Pl, n_T), dtype=torch.float64, device=dev, generator=gen)
                B_l = torch.rand((n_T, n_rec), dtype=torch.float64, device=dev, generator=gen)
                C_l = torch.empty((Pl, n_rec), dtype=torch.float64, device=dev)
                t_l = timed(lambda: torch.matmul(A_l, B_l, out=C_l), 3)
                lib_dgemm = {"shape": [Pl, n_T, n_rec], "ms": t_l, "tflops": 2.0 * Pl * n_T * n_rec / t_l / 1e9,
                             "note": "torch.matmul float64 (cuBLAS DGEMM), one period, operands resident; not on the product path"}
                del A_l, B_l, C_l
            except RuntimeError as exc:                                  # out of memory on a crowded box: context only
                lib_dgemm = {"unavailable": str(exc)[:120]}

    sec["extras"] = time.perf_counter() - t_extras
    ctx.close()
    del dev_inp, param_dev
    torch.cuda.empty_cache()

    # ---------------------------------------------------------------- every other BASELINE config, briefly
    if not lite and rank == 0:
        per_config = {name: {"see": "top level of this line (value, e2e, roofline, parity)", "evals_per_s": value,
                             "ms_per_scan": ms / args.steps, "dominant_kernel": dom, "bound": "tensor", "achieved": achieved,
                             "peak": dmma_peak, "unit": "TFLOP/s", "frac": achieved / dmma_peak,
                             "single_eval_ms": single["ms_per_call"] if single else None, "parity": full.get("parity")}}
        for other in wl.CONFIG_NAMES:
            if other == name:
                continue
            r = guard(other, lambda: bench_config(other, dev, min(args.steps, 5), 3, peaks, dmma_peak, cores, True))
            per_config[other] = r if r is not None else {"unavailable": full["errors"][-1]}
        roofline["per_config"] = per_config

    if rank == 0:
        full.update({"single_eval": single, "batch_sweep": sweep, "collapsed_mode": collapsed, "fp32_mode": fp32_leg,
                     "sliced_mode": sliced_leg, "library_dgemm": lib_dgemm, "next_rows": next_rows,
                     "bench_wall_s": time.perf_counter() - t_start,
                     "paper_context": "PAPER.md Table I: 86.8 ms (RTX 3080 Ti) / 52.4 ms (A30X) per single evaluation of "
                                      "the authors' own multi-component model; other hardware and inputs, not comparable"})
        full.setdefault("cpu_baseline", None)
        full.setdefault("parity", None)
        if full["detail"]:
            try:
                with open(os.path.join(ROOT, args.detail), "w") as f:
                    json.dump(_clean(full, 9), f, indent=1, allow_nan=False)
            except OSError as exc:
                full["detail"] = None
                full["errors"].append("detail file: %s" % exc)
        sys.stdout.flush()
        print(contract_line(full), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
