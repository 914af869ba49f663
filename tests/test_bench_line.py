"""The stdout contract line of bench.py: small, strict JSON, numbers only -- whatever the legs produced.
(Round 2's line had grown to ~30 KB and the driver could not parse it; everything else now goes to bench_detail.json.)"""
import json
import math

import bench


def _canned_full():
    regimes = [{"regime": "single_eval", "points": 1, "kernel": "k_fold_stream<1>", "bound": "hbm",
                "ms_per_call": 0.17512345678, "frac": 0.9712345678, "note": "prose " * 40}]
    for P in bench.REGIME_POINTS:
        regimes.append({"regime": "ridge", "points": P, "kernel": bench.policy_kernel(P), "bound": "tensor" if P > 22 else "hbm",
                        "ms_per_call": 0.1798765432 + 0.007 * P, "frac": 0.8123456789, "kernel_frac": 0.9,
                        "traffic_source": "x" * 80})
    regimes.append({"regime": "batched", "points": 65536, "kernel": "k_fold_gemm<8>", "bound": "tensor",
                    "ms_per_call": 487.123456, "frac": 0.97123456})
    parity = {"points": 32, "mu_rel_max": 1.2345678e-15, "mu_bar": 1e-12, "m2lnl_abs_max": 2.98e-8,
              "m2lnl_bound_max": 1.6e-5, "m2lnl_err_over_bound_max": 0.0019, "pass": True, "bar": "prose " * 30,
              "source": "prose " * 30}
    per_config = {}
    for name in ("cfg1_tiny_nsi", "cfg2_mm_lowE", "cfg3_nsi4", "cfg4_dense", "cfg5_joint6"):
        per_config[name] = {"evals_per_s": 1234567.891, "bound": "tensor", "frac": float("nan"), "single_eval_ms": 0.0234567,
                            "parity": parity, "note": "prose " * 50, "single_eval": regimes[0]}
    per_config["cfg2_mm_lowE"] = {"unavailable": "CUDA error: " + "x" * 150}
    return {"metric": bench.METRIC, "value": 134567.8912345, "unit": bench.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
            "ms_per_step": 487.0123456, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "cfg4_dense", "n_E": 4096, "n_T": 16384, "n_rec": 8192, "n_periods": 1,
                       "points_per_step_per_gpu": 65536, "response_bytes": 1073741824, "library_slice_points": 65536,
                       "parallelism": "points sharded over 1 GPU(s), tables replicated, no collective", "l2_flush": False},
            "e2e": {"value": 134500.123, "unit": bench.UNIT, "h2d_bytes_per_step": 3670016, "d2h_bytes_per_step": 524288,
                    "ms_per_step": 487.3, "matches_device_path": True},
            "gpu_launches": 260, "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "samples": 50, "reasons": ["sw_power_cap"]},
            "all_finite": True, "errors": ["fp32 leg: boom"], "detail": bench.DETAIL_FILE,
            "roofline": {"bound": "tensor", "kernel": "k_fold_gemm<8>", "achieved": 36.123456789, "peak": 37.1, "unit": "TFLOP/s",
                         "frac": 0.9737, "call_frac": 0.9701, "traffic": 64.55e9, "traffic_source": "prose " * 20,
                         "peak_source": "prose " * 40, "launches_timed": 80, "avg_launch_ms": 121.7,
                         "flops_per_launch": 4.4e15, "kernel_share_of_step": 0.9991, "ridge_points": 22.6,
                         "regimes": regimes, "per_config": per_config},
            "cpu_baseline": {"value": 2.83, "unit": bench.UNIT, "cores": 16, "kind": "oracle", "sample": "32 of 65536 scan points, 16 threads, 11.3 s",
                             "sample_detail": "prose " * 30, "single_thread": {"value": 0.21, "sample": "prose"}},
            "parity": parity, "bench_wall_s": 101.2, "single_eval": regimes[0],
            "sliced_mode": {"note": "prose " * 100, "inf": math.inf}, "paper_context": "prose " * 30}


def test_contract_line_is_small_strict_json_with_every_required_key():
    full = _canned_full()
    text = bench.contract_line(full)
    assert "\n" not in text and len(text) < bench.LINE_LIMIT, len(text)
    assert "NaN" not in text and "Infinity" not in text
    line = json.loads(text, parse_constant=lambda c: (_ for _ in ()).throw(ValueError(c)))   # strict: no NaN / Infinity
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "e2e", "gpu_launches", "clocks", "roofline", "cpu_baseline", "parity"):
        assert key in line, key
    assert line["value"] > 0 and line["config"]["workload"] == "cfg4_dense"
    assert set(line["e2e"]) >= {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
    roof = line["roofline"]
    assert set(roof) >= {"bound", "achieved", "peak", "unit", "frac", "traffic", "regimes", "per_config"}
    assert abs(roof["frac"] - roof["achieved"] / roof["peak"]) < 1e-3
    assert len(roof["regimes"]) == len(bench.REGIME_POINTS) + 2 and roof["regimes"][1][0] == 2
    assert roof["per_config"]["cfg2_mm_lowE"] is None and roof["per_config"]["cfg3_nsi4"][2] is None   # NaN -> null
    assert set(line["cpu_baseline"]) >= {"value", "unit", "cores", "kind", "sample", "single_thread_value"}
    assert line["parity"]["pass"] is True and line["detail"] == bench.DETAIL_FILE and line["errors"] == 1
    assert "prose" not in text                                   # notes, bars and sources stay in the detail file
    # the full dict itself serialises strictly for the detail file
    json.dumps(bench._clean(full, 9), allow_nan=False)


def test_contract_line_sheds_context_rather_than_exceed_the_limit():
    full = _canned_full()
    full["roofline"]["regimes"] = full["roofline"]["regimes"] * 12
    text = bench.contract_line(full)
    line = json.loads(text)
    assert len(text) < bench.LINE_LIMIT and "regimes" not in line["roofline"] and line["value"] > 0


def test_ncu_traffic_is_read_from_the_committed_csv(tmp_path):
    p = tmp_path / "t.csv"
    p.write_text("call,kernel,time_ms,dram_read_bytes,dram_write_bytes\n"
                 "rw_eval_batch P=8,k_a,1.0,100,5\nrw_eval_batch P=8,k_b,2.0,,1\nrw_eval_batch P=8,k_a,1.1,200,7\n"
                 "rw_eval_batch P=8,k_a,0.1,,\nrw_eval_batch P=8 RW_SLICED,k_a,9.0,1,1\nrw_eval_pee P=4,k_a,9.0,2,2\n")
    assert bench.load_ncu_traffic(str(p)) == {"k_a": 207.0}
    real = bench.load_ncu_traffic()                     # the committed capture (profiles/r03_folds_raw.csv)
    assert 1.07e9 < real["k_fold_stream<1>"] < 1.10e9 and real["k_fold_gemm<8>"] > 1e10
    assert bench.load_ncu_traffic(str(tmp_path / "missing.csv")) == {}
