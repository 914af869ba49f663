"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(device-resident tables, R borrowed, mode auto, whole scan in one rw_eval_batch call), checked on
sampled outputs the oracle computes one by one."""
import os

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 4


def _device_ctx(binding, inp, max_batch, sliced=False):
    import torch
    dev_inp = {k: torch.from_numpy(np.ascontiguousarray(inp[k])).cuda()
               for k in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev_inp["f_tau"] = inp["f_tau"]
    return binding.Reweighter(dev_inp, max_batch=max_batch, sliced=sliced)


def _full_vs_sample(orc, name, sample_idx, max_batch, mu_check=True, sliced=False):
    import torch
    from paper_2607_00488_b200 import binding
    inp = wl.make(name)
    params, kinds = wl.scan_points(name)
    P = params.shape[0]
    ctx = _device_ctx(binding, inp, max_batch, sliced=sliced)
    out = ctx.eval_batch(torch.from_numpy(params).cuda(), kinds)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert out.shape == (P,) and np.all(np.isfinite(out)) and np.all(out >= 0)
    idx = np.unique(np.clip(np.asarray(sample_idx), 0, P - 1))
    ref, mu_ref, scale = orc.eval_batch(inp, params[idx], kinds, want_mu=True, want_abs=True, nthreads=CORES)
    err = np.abs(out[idx] - ref)
    assert np.all(err <= 1e-9 + 1e-12 * scale), "max err %.3e at -2lnL %.6e" % (err.max(), ref[err.argmax()])
    if mu_check:
        _, mu = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm")
        torch.cuda.synchronize()
        rel = np.abs(mu.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        assert rel.max() <= 1e-12, "mu rel err %.3e" % rel.max()
        # the same points through the streaming fold agree with the contraction to rounding
        out_s = ctx.eval_batch(torch.from_numpy(params[idx[:8]]).cuda(), kinds, mode="stream")
        torch.cuda.synchronize()
        assert np.all(np.abs(out_s.cpu().numpy() - ref[:8]) <= 1e-9 + 1e-12 * scale[:8])
    if sliced:      # the INT8-sliced contraction on the sampled points: same FP64 bars
        out_i8, mu_i8 = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm", sliced=True)
        torch.cuda.synchronize()
        rel = np.abs(mu_i8.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        assert rel.max() <= 1e-12, "sliced mu rel err %.3e" % rel.max()
        assert np.all(np.abs(out_i8.cpu().numpy() - ref) <= 1e-9 + 1e-12 * scale)
        # their top four slices only (RW_SLICED_FAST): the FP32 bar
        _, mu_f = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm", sliced="fast")
        torch.cuda.synchronize()
        rel = np.abs(mu_f.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        assert rel.max() <= 1e-5, "fast sliced mu rel err %.3e" % rel.max()
    ctx.close()
    return err.max()


def test_config3_full_scan_sampled(orc):
    rng = np.random.default_rng(303)
    idx = np.concatenate([[0, 9999, 8191, 8192], rng.integers(0, 10000, 28)])
    _full_vs_sample(orc, "cfg3_nsi4", idx, max_batch=10000, sliced=True)


def test_config4_bench_configuration_sampled(orc):
    """65536 points, 16384 x 8192 response: exactly what bench.py times (8 chunks of 8192 points)."""
    rng = np.random.default_rng(404)
    idx = np.concatenate([[0, 65535, 8191, 8192, 32767, 32768], rng.integers(0, 65536, 18)])
    _full_vs_sample(orc, "cfg4_dense", idx, max_batch=65536, sliced=True)


def test_config5_streamed_in_batches_of_16384(orc):
    """10^6 Latin-hypercube points, 8 periods; the library slices the call into 61 batches of 16384 and
    one of 576 (max_batch = 16384).  Samples include first/last points of several batches."""
    rng = np.random.default_rng(505)
    edges = [0, 16383, 16384, 61 * 16384 - 1, 61 * 16384, 999999, 100 * 16384 // 2]
    idx = np.concatenate([edges, rng.integers(0, 1000000, 17)])
    _full_vs_sample(orc, "cfg5_joint6", idx, max_batch=16384, mu_check=False, sliced=True)
