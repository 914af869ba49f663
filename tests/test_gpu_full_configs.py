"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(device-resident tables, R borrowed, mode auto, whole scan in one rw_eval_batch call), checked on
sampled outputs the oracle computes one by one: 64 seeded random points of each scan plus the first and last point
of library slices / contraction chunks, and the SM point with its sign-flip partner.  Every test
prints the raw maxima it saw (run with -s)."""
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


def _sm_and_partner(orc, ctx, inp, kinds, name):
    """theta = 0 and its sign-flip partner g~ -> -g~ (eps = -2 g for every scanned chiral coupling): Eq. (4) is even in
    (g~_L, g~_R) jointly, so the two points have the same spectrum; against the oracle and against each other."""
    import torch
    k = len(kinds)
    pts = np.zeros((2, k))
    g_L, g_R = orc.sm_couplings()
    for a, kind in enumerate(kinds):
        if kind < 6:
            pts[1, a] = -2.0 * (g_L if kind % 2 == 0 else g_R)[kind // 2]
    flavours = {int(kd) // 2 for kd in kinds if kd < 6}
    both = all((2 * f in kinds) and (2 * f + 1 in kinds) for f in flavours)
    ref, scale = orc.eval_batch(inp, pts, kinds, want_abs=True, nthreads=2)
    out = ctx.eval_batch(torch.from_numpy(pts).cuda(), kinds).cpu().numpy()
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-12 * scale)
    if both:
        assert abs(out[0] - out[1]) <= 1e-9 + 1e-12 * scale[0], "%s: sign-flip partner differs by %.3e" % (name, abs(out[0] - out[1]))
    print("%s: SM point -2lnL %.6f, sign-flip partner %.6f (oracle %.6f, %.6f)" % (name, out[0], out[1], ref[0], ref[1]))


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
    print("%s: %d sampled points of %d (max_batch %d): max |d(-2lnL)| %.3e, max |d|/sum|terms| %.3e" % (
        name, idx.size, P, max_batch, err.max(), (err / scale).max()))
    assert np.all(err <= 1e-9 + 1e-12 * scale), "max err %.3e at -2lnL %.6e" % (err.max(), ref[err.argmax()])
    _sm_and_partner(orc, ctx, inp, kinds, name)
    if mu_check:
        _, mu = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm")
        torch.cuda.synchronize()
        rel = np.abs(mu.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        print("%s: max relative error of mu over %d points x bins: %.3e" % (name, idx.size, rel.max()))
        assert rel.max() <= 1e-12, "mu rel err %.3e" % rel.max()
        # the same points through the streaming fold agree with the contraction to rounding
        out_s = ctx.eval_batch(torch.from_numpy(params[idx[:8]]).cuda(), kinds, mode="stream")
        torch.cuda.synchronize()
        assert np.all(np.abs(out_s.cpu().numpy() - ref[:8]) <= 1e-9 + 1e-12 * scale[:8])
    if sliced:      # the INT8-sliced contraction on the sampled points: same FP64 bars
        out_i8, mu_i8 = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm", sliced=True)
        torch.cuda.synchronize()
        rel = np.abs(mu_i8.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        print("%s: RW_SLICED max relative error of mu: %.3e" % (name, rel.max()))
        assert rel.max() <= 1e-12, "sliced mu rel err %.3e" % rel.max()
        assert np.all(np.abs(out_i8.cpu().numpy() - ref) <= 1e-9 + 1e-12 * scale)
        # their top four slices only (RW_SLICED_FAST): the FP32 bar
        _, mu_f = ctx.eval_batch(torch.from_numpy(params[idx]).cuda(), kinds, want_mu=True, mode="gemm", sliced="fast")
        torch.cuda.synchronize()
        rel = np.abs(mu_f.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        print("%s: RW_SLICED_FAST max relative error of mu: %.3e" % (name, rel.max()))
        assert rel.max() <= 1e-5, "fast sliced mu rel err %.3e" % rel.max()
    ctx.close()
    return err.max()


def test_config3_full_scan_sampled(orc):
    rng = np.random.default_rng(303)
    idx = np.concatenate([[0, 9999, 8191, 8192], rng.integers(0, 10000, 64)])
    _full_vs_sample(orc, "cfg3_nsi4", idx, max_batch=10000, sliced=True)


def test_config4_bench_configuration_sampled(orc):
    """65536 points, 16384 x 8192 response: exactly what bench.py times (one library slice of 65536 points, cut by the
    library into two contraction chunks of 32768)."""
    rng = np.random.default_rng(404)
    idx = np.concatenate([[0, 65535, 8191, 8192, 32767, 32768], rng.integers(0, 65536, 64)])
    _full_vs_sample(orc, "cfg4_dense", idx, max_batch=65536, sliced=True)


def test_config5_streamed_in_batches_of_16384(orc):
    """10^6 Latin-hypercube points, 8 periods; the library slices the call into 61 batches of 16384 and
    one of 576 (max_batch = 16384, what bench.py's per_config leg uses).  64 random points + the first and last point
    of every 10th batch and of the ragged last one."""
    rng = np.random.default_rng(505)
    B = 16384
    edges = [e for b in list(range(0, 62, 10)) + [60, 61] for e in (b * B, min((b + 1) * B, 1000000) - 1)]
    idx = np.concatenate([edges, rng.integers(0, 1000000, 64)])
    _full_vs_sample(orc, "cfg5_joint6", idx, max_batch=B, mu_check=False, sliced=True)


def test_config5_small_library_slices_every_100th_batch(orc):
    """The same scan through a context with max_batch = 2048: 488 full batches and one of 576 points, each a single
    contraction with its own tile-height choice.  First and last point of every 100th batch."""
    B = 2048
    n_b = (1000000 + B - 1) // B
    edges = [e for b in list(range(0, n_b, 100)) + [n_b - 1] for e in (b * B, min((b + 1) * B, 1000000) - 1)]
    _full_vs_sample(orc, "cfg5_joint6", edges, max_batch=B, mu_check=False)
