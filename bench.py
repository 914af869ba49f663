#!/usr/bin/env python
"""bench.py -- likelihood evaluations per second on BASELINE.json's dense-contraction config.

One *step* = one pass of the whole hot path (coefficients -> reweighted MC spectrum -> response
fold -> Poisson -2lnL) over one batch of the config's scan points.  Default workload: config 4
("cfg4_dense": 16384 recoil bins x 8192 reconstructed bins, 1.07 GB FP64 response, 65536 points),
the configuration the batched-throughput metric is quoted on; the others are parity cases.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config NAME]

N > 1 is launched by torchrun (one rank per GPU); the points are sharded, the tables replicated,
there is no data-path collective (weak scaling: every rank folds its own 65536-point batch).
`--impl reference` times the CPU oracle (oracle/) on the box's host cores -- a deliberately slow,
plain program; see DESIGN.md section 8.
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

# dram__bytes_read.sum + dram__bytes_write.sum per k_fold_gemm launch from the committed
# `ncu --set full` capture (profiles/r01c_fold_gemm_full.md: the fused launch over the 110 full waves of one
# 32768-point chunk), or None if not captured.
NCU_TRAFFIC_BYTES_PER_LAUNCH = {"cfg4_dense": 69.584991e9 + 0.032040e9}
# the same for the single-evaluation kernel k_fold_stream<1> (profiles/r01e_fold_stream_full.md)
NCU_TRAFFIC_BYTES_SINGLE_EVAL = {"cfg4_dense": 1.075726e9 + 0.0112768e9}


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


def oracle_sample_run(name, n_points, nthreads, repeats=1):
    """Times the oracle as it stands on the first n_points scan points; returns (evals/s, seconds)."""
    from oracle import rw_oracle as orc
    from paper_2607_00488_b200 import workloads as wl
    inp = wl.make(name)
    params, kinds = wl.scan_points(name)
    sample = params[:n_points]
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        orc.eval_batch(inp, sample, kinds, nthreads=nthreads)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return n_points / best, best


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
    n_sample = max(1, min(params.shape[0], cores))        # one point per core and step
    for w in range(args.warmup):
        orc.eval_batch(inp, params[:n_sample], kinds, nthreads=cores)
    t0 = time.perf_counter()
    for s in range(args.steps):
        lo = (s * n_sample) % max(1, params.shape[0] - n_sample + 1)
        orc.eval_batch(inp, params[lo:lo + n_sample], kinds, nthreads=cores)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    sample = "%d scan points per step (of %d), OpenMP over points on %d threads" % (n_sample, params.shape[0], cores)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(name, inp, params.shape[0], args.gpus, sample=sample),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(name, inp, P, n_gpus, sample=None, max_batch=0):
    D, n_T, n_rec = inp["R"].shape
    cfg = {"workload": name, "n_E": int(inp["E"].size), "n_T": int(n_T), "n_rec": int(n_rec), "n_periods": int(D),
           "points_per_step_per_gpu": int(P), "response_bytes": int(D * n_T * n_rec * 8),
           "library_slice_points": int(max_batch) if max_batch else int(P),
           "parallelism": "points sharded over %d GPU(s), tables replicated, no collective" % n_gpus,
           "l2": ("response (%.2f GB) and reweighted spectrum exceed the 126 MB L2: no flush needed" % (D * n_T * n_rec * 8 / 1e9))
                 if D * n_T * n_rec * 8 + 8.0 * P * n_T > 252e6 else
                 "working set fits the 126 MB L2: a 256 MB buffer is rewritten between timed steps (L2 flush)"}
    if sample:
        cfg["sample"] = sample
    return cfg


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4_dense")
    ap.add_argument("--no-cpu-baseline", action="store_true")
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

    import torch
    import torch.distributed as dist
    from paper_2607_00488_b200 import binding, sharding, workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    binding.load_library()
    name = args.config
    inp = wl.make(name)
    D, n_T, n_rec = inp["R"].shape
    params, kinds = sharding.rank_points(name, rank)
    P, k = params.shape

    # tables resident in HBM before anything is timed (R is borrowed by the context, not copied)
    dev_inp = {key: torch.from_numpy(np.ascontiguousarray(inp[key])).to(dev)
               for key in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev_inp["f_tau"] = inp["f_tau"]
    max_batch = args.max_batch or (16384 if name == "cfg5_joint6" else P)
    sliced_ok = True
    ctx = binding.Reweighter(dev_inp, max_batch=max_batch, device=dev, fp32=True, sliced=sliced_ok)   # + operand copies for the opt-in legs
    param_dev = torch.from_numpy(params).to(dev)
    out_dev = torch.empty(P, dtype=torch.float64, device=dev)
    param_pin = torch.from_numpy(params).pin_memory()
    out_pin = torch.empty(P, dtype=torch.float64).pin_memory()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def maxreduce(x):
        return sharding.max_over_ranks(x, dev, world)

    dmma_peak0 = binding.probe_fp64_peak(1)
    dfma_peak0 = binding.probe_fp64_peak(0)

    # ---------------------------------------------------------------- device-resident throughput
    for _ in range(args.warmup):
        ctx.eval_batch(param_dev, kinds, out=out_dev)
    barrier()
    sampler = ClockSampler("GPU-" + str(torch.cuda.get_device_properties(dev).uuid))
    if rank == 0:
        sampler.start()
    launches0 = ctx.launch_count()
    ctx.profile_begin()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    need_flush = D * n_T * n_rec * 8 + 8.0 * P * n_T <= 252e6      # working set could stay in the 126 MB L2
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if need_flush else None

    def timed_steps(fn):
        """K steps timed on the device; with an L2 flush (256 MB rewrite, untimed) before each one if needed."""
        barrier()
        if not need_flush:
            e0.record()
            for _ in range(args.steps):
                fn()
            e1.record()
            barrier()
            return e0.elapsed_time(e1)
        total = 0.0
        for _ in range(args.steps):
            flush_buf.zero_()
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            total += e0.elapsed_time(e1)
        barrier()
        return total

    ms = maxreduce(timed_steps(lambda: ctx.eval_batch(param_dev, kinds, out=out_dev)))
    fold_ms, fold_launches = ctx.profile_end()
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    value = sharding.whole_job_value(world, P, args.steps, ms)
    finite = bool(torch.isfinite(out_dev).all().item())

    # ---------------------------------------------------------------- end to end with host buffers
    for _ in range(2):
        ctx.eval_batch(param_pin, kinds, out=out_pin)
    # H2D params, kernels, D2H -2lnL: all on the stream, inside the timed region
    ms_e2e = maxreduce(timed_steps(lambda: ctx.eval_batch(param_pin, kinds, out=out_pin)))
    e2e_value = sharding.whole_job_value(world, P, args.steps, ms_e2e)
    same = bool(np.array_equal(out_pin.numpy(), out_dev.cpu().numpy()))

    # ---------------------------------------------------------------- single evaluation (HBM-bound regime)
    one = param_dev[:1].contiguous()
    out1 = torch.empty(1, dtype=torch.float64, device=dev)
    for _ in range(5):
        ctx.eval_batch(one, kinds, out=out1, mode="stream")
    torch.cuda.synchronize()
    reps = 30
    ctx.profile_begin()
    e0.record()
    for _ in range(reps):
        ctx.eval_batch(one, kinds, out=out1, mode="stream")
    e1.record()
    torch.cuda.synchronize()
    single_ms = e0.elapsed_time(e1) / reps
    sfold_ms, sfold_n = ctx.profile_end()
    # the same single evaluation replayed from a CUDA graph: device-side latency without the Python/ctypes call
    graph_us = None
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            ctx.eval_batch(one, kinds, out=out1, mode="stream")
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            ctx.eval_batch(one, kinds, out=out1, mode="stream")
        for _ in range(5):
            g.replay()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            g.replay()
        e1.record()
        torch.cuda.synchronize()
        graph_us = e0.elapsed_time(e1) / reps * 1e3
    except Exception as exc:                                  # capture is a convenience, not part of the metric
        graph_us = "unavailable: %s" % exc
    peaks = load_peaks()
    r_bytes = D * n_T * n_rec * 8
    single = {"ms_per_eval": single_ms, "graph_replay_us_per_eval": graph_us, "fold_kernel_ms": sfold_ms / max(1, sfold_n),
              "hbm_gbs": r_bytes / (sfold_ms / max(1, sfold_n) * 1e-3) / 1e9,
              "hbm_peak_gbs": peaks["hbm_gbs"]}
    if r_bytes > 252e6:
        single["note"] = ("P=1, one-launch streaming path (fold + likelihood); R (%.2f GB) >> L2, so every eval reads it "
                          "from HBM; kernel time includes the last-CTA reduction" % (r_bytes / 1e9))
        single["hbm_frac"] = single["hbm_gbs"] / peaks["hbm_gbs"]
        single["algorithmic_bytes"] = r_bytes
        single["traffic"] = NCU_TRAFFIC_BYTES_SINGLE_EVAL.get(name)
    else:
        single["note"] = ("P=1, one-launch streaming path; R (%.1f MB) stays in the 126 MB L2 between back-to-back "
                          "evaluations: latency-bound, no HBM fraction is claimed" % (r_bytes / 1e6))
        single["hbm_frac"] = None

    # ---------------------------------------------------------------- other regimes of the same path (context lines)
    def timed(fn, reps):
        fn(); fn()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    sweep = []
    for Pb in (1, 4, 16, 64, 256, 2048):
        if Pb > P:
            break
        pb = param_dev[:Pb].contiguous()
        ob = torch.empty(Pb, dtype=torch.float64, device=dev)
        t = timed(lambda: ctx.eval_batch(pb, kinds, out=ob), 20 if Pb <= 256 else 5)
        sweep.append({"points": Pb, "ms_per_call": t, "evals_per_s": Pb / t * 1e3,
                      "fold_tflops": 2.0 * n_T * n_rec * D * Pb / t / 1e9, "response_gbs": r_bytes / t / 1e6})
    # opt-in rank-K collapsed mode: exact, O(11 n_rec) per point, FP64-ALU bound; never mixed into `value`
    out_c = torch.empty(P, dtype=torch.float64, device=dev)
    t_c = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_c, mode="collapsed"), 5)
    dmax = float((out_c - out_dev).abs().max().item())
    collapsed = {"ms_per_call": t_c, "evals_per_s": P / t_c * 1e3, "bound": "alu",
                 "algorithmic_gflops": 2.0 * 11 * n_rec * D * P / t_c / 1e6,
                 "max_abs_diff_vs_dense_fold": dmax,
                 "note": "2*11*n_rec*D flop per point plus one log1p per bin; see profiles/ for the FP64-pipe utilisation"}

    # opt-in RW_FP32 contraction: TF32 x 3 on tcgen05, 1e-5 relative on mu; never mixed into `value`
    fp32_leg = None
    try:                                   # a context leg must never take the bench line down with it
        if P > 4:
            out_f = torch.empty(P, dtype=torch.float64, device=dev)
            t_f = timed(lambda: ctx.eval_batch(param_dev, kinds, out=out_f, fp32=True), 5)
            ns = min(P, 128)
            _, mu32 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm", fp32=True)
            _, mu64 = ctx.eval_batch(param_dev[:ns].contiguous(), kinds, want_mu=True, mode="gemm")
            rel = ((mu32 - mu64).abs() / mu64.abs())
            fp32_leg = {"ms_per_call": t_f, "evals_per_s": P / t_f * 1e3, "bound": "tensor (tf32) / L2",
                        "effective_fold_tflops": 2.0 * n_T * n_rec * D * P / t_f / 1e9,
                        "executed_tf32_tflops": 6.0 * n_T * n_rec * D * P / t_f / 1e9,
                        "mu_rel_err_vs_fp64_max": float(rel.max().item()), "mu_rel_err_vs_fp64_mean": float(rel.mean().item()),
                        "note": "three tcgen05.mma.kind::tf32 products per k-step (hi*hi, hi*lo, lo*hi), FP32 accumulation in "
                                "128-bin TMEM chunks; the three-fold executed flops are not counted in effective_fold_tflops"}
    except Exception as exc:               # noqa: BLE001
        fp32_leg = {"unavailable": str(exc)[:160]}

    # opt-in RW_SLICED contraction: FP64 by slicing on the INT8 tensor cores, exact int32 accumulation,
    # same 1e-12 bar as the DMMA path; a context line, never mixed into `value`
    sliced_leg = None
    try:
        if P > 4 and sliced_ok:
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
                        "effective_fold_tflops": 2.0 * n_T * n_rec * D * P / t_f / 1e9,
                        "mu_rel_err_vs_fp64_max": float(relf.max().item()), "int8_products_per_k_step": 10}
            n_sl = 8 if n_T <= 2048 else 7                              # balanced 8-bit slices per operand (rw_fold_i8.cu)
            n_prod = n_sl * (n_sl + 1) // 2
            sliced_leg = {"ms_per_call": t_s, "evals_per_s": P / t_s * 1e3, "bound": "tensor (int8)",
                          "effective_fold_tflops": 2.0 * n_T * n_rec * D * P / t_s / 1e9,
                          "kernel_effective_fold_tflops": 2.0 * n_T * n_rec * D * P * 7 / (k_ms * 1e-3) / 1e12 if k_ms > 0 else None,
                          "executed_int8_tops": 2.0 * n_prod * n_T * n_rec * D * P / t_s / 1e9,
                          "mu_rel_diff_vs_dmma_max": float(rel.max().item()),
                          "max_abs_diff_m2lnL_vs_dmma": float((out_s - out_dev).abs().max().item()),
                          "slices": n_sl, "int8_products_per_k_step": n_prod, "fast": fast_leg,
                          "note": "%d balanced 8-bit slices per operand, %d tcgen05.mma.kind::i8 products per k-step with exact "
                                  "int32 accumulation in TMEM; FP64 DMMA peak is %.1f TFLOP/s" % (n_sl, n_prod, dmma_peak0)}
    except Exception as exc:               # noqa: BLE001
        sliced_leg = {"unavailable": str(exc)[:160]}

    # the other entry points of the same path, timed on a slice of the same scan: context only
    next_rows = None
    try:
        if P > 4 and rank == 0:
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
            if ctx.n_periods >= 1 and all(x < 7 for x in kin) and "P_mu" not in inp and int(inp.get("n_comp", 1) or 1) == 1:
                Pe = int(min(P, max_batch, 1024))
                pe = param_dev[:Pe].contiguous()
                tab = torch.from_numpy(np.ascontiguousarray(inp["P_e"])).to(dev)[None, :].repeat(Pe, 1).contiguous()
                t = timed(lambda: ctx.eval_pee(pe, kinds, tab), 3)
                nr["per_point_pee"] = {"points": Pe, "n_E": int(tab.shape[1]), "ms_per_call": t, "evals_per_s": Pe / t * 1e3,
                                       "note": "rw_eval_pee: spectrum on the (E x T) grid per point (FP64 ALU), then the dense fold"}
            next_rows = nr
    except Exception as exc:                   # noqa: BLE001
        next_rows = {"unavailable": str(exc)[:160]}

    # library DGEMM of the shape of one chunk of the fold (cuBLAS FP64 as a reference point for the
    # denominator).  Context only: no N' generation, no Poisson epilogue, no reduction, and mu goes to HBM.
    lib_dgemm = None
    if P > 4 and rank == 0:
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

    # ---------------------------------------------------------------- roofline of the dominant kernel
    # the probe is taken before the timed region and again here; the higher reading is the denominator (a probe
    # right after the TF32 leg can catch a lower clock)
    dmma_peak = max(dmma_peak0, binding.probe_fp64_peak(1))
    dfma_peak = max(dfma_peak0, binding.probe_fp64_peak(0))
    flops_timed = 2.0 * n_T * n_rec * D * P * args.steps           # algorithmic: 2 N_T N_rec per point and period
    achieved = flops_timed / (fold_ms * 1e-3) / 1e12
    traffic = NCU_TRAFFIC_BYTES_PER_LAUNCH.get(name)
    roofline = {"bound": "tensor", "kernel": "k_fold_gemm", "achieved": achieved, "peak": dmma_peak, "unit": "TFLOP/s",
                "frac": achieved / dmma_peak, "traffic": traffic,
                "peak_source": "FP64 DMMA.8x8x4 issue-rate probe measured live (rw_probe_fp64_peak); DFMA probe %.2f; "
                               "bf16 %s peak x nominal FP64/bf16 ratio (45/2250) = %.1f burst / %.1f sustained"
                               % (dfma_peak, peaks["source"], peaks["bf16"] * 0.02, (peaks["bf16_sus"] or 0) * 0.02),
                "launches_timed": int(fold_launches), "avg_launch_ms": fold_ms / max(1, fold_launches),
                "flops_per_launch": flops_timed / max(1, fold_launches),
                "kernel_share_of_step": fold_ms / ms}

    # ---------------------------------------------------------------- CPU oracle beside it
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import rw_oracle as orc
        orc.build()
        cores = os.cpu_count() or 1
        n_sample = min(P, 4 * cores)
        v, secs = oracle_sample_run(name, n_sample, cores)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "first %d of %d scan points, OpenMP over points on %d threads, %.1f s wall" % (n_sample, P, cores, secs)}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": workload_config(name, inp, P, world, max_batch=max_batch),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(P * k * 8),
                        "d2h_bytes_per_step": int(P * 8), "ms_per_step": ms_e2e / args.steps,
                        "matches_device_path": same},
                "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu, "single_eval": single,
                "batch_sweep": sweep, "collapsed_mode": collapsed, "fp32_mode": fp32_leg, "sliced_mode": sliced_leg,
                "library_dgemm": lib_dgemm, "next_rows": next_rows, "clocks": clocks, "all_finite": finite,
                "paper_context": "PAPER.md Table I: 86.8 ms (RTX 3080 Ti) / 52.4 ms (A30X) per single evaluation of "
                                 "the authors' own multi-component model; other hardware and inputs, not comparable"}
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
