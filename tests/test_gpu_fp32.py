"""Opt-in RW_FP32 variant of the batched contraction (TF32 x 3 on tcgen05) against the FP64 oracle.
Bar (BASELINE.json north_star): mu within 1e-5 relative; -2lnL within the first-order propagation of that
bound, sum_k 2 |1 - n_k/mu_k| * 1e-5 mu_k (+ 1e-9), computed from the oracle's mu."""
import os

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 4
MU_RTOL = 1e-5


def _cuda(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _check(orc, inp, params, kinds, max_batch=None):
    import torch
    from paper_2607_00488_b200 import binding
    ref, mu_ref = orc.eval_batch(inp, params, kinds, want_mu=True, nthreads=CORES)
    ctx = binding.Reweighter(inp, max_batch=max_batch or params.shape[0], fp32=True)
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="gemm", fp32=True)
    out64 = ctx.eval_batch(_cuda(params), kinds, mode="gemm")
    torch.cuda.synchronize()
    out, mu, out64 = out.cpu().numpy(), mu.cpu().numpy(), out64.cpu().numpy()
    ctx.close()
    rel = np.abs(mu - mu_ref) / np.abs(mu_ref)
    assert rel.max() <= MU_RTOL, "fp32 mu rel err %.3e" % rel.max()
    counts = np.asarray(inp["counts"], float).reshape(mu_ref.shape[1:])
    tol = 1e-9 + (2.0 * np.abs(1.0 - counts[None] / mu_ref) * MU_RTOL * mu_ref).sum(axis=(1, 2))
    assert np.all(np.abs(out - ref) <= tol), "fp32 -2lnL err %.3e (tol %.3e)" % (np.abs(out - ref).max(), tol.min())
    assert np.all(np.abs(out64 - ref) <= 1e-9 + 1e-11 * np.abs(ref))      # the FP64 path of the same context is intact
    return rel.max()


def test_fp32_small_ragged(orc):
    """n_T = 203 (partial 32-bin stage, 2 chunks), n_rec = 330 (3 column tiles, ragged), 2 periods, 300 points."""
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=330, n_periods=2, seed=61, dead_fraction=0.1)
    params, kinds = wl.random_points(300, list(range(7)), seed=62)
    _check(orc, inp, params, kinds)


def test_fp32_long_contraction(orc):
    """n_T = 3000: 24 accumulation chunks per tile, several tiles per CTA (TMEM double buffering wraps)."""
    inp = wl.make_custom(n_E=24, n_T=3000, n_rec=200, n_periods=1, seed=63)
    params, kinds = wl.random_points(150, [wl.EPS_EE_L, wl.EPS_EE_R, wl.MU_NU], seed=64)
    _check(orc, inp, params, kinds, max_batch=64)


def test_fp32_config2_all_points(orc):
    inp = wl.make("cfg2_mm_lowE")
    params, kinds = wl.scan_points("cfg2_mm_lowE")
    _check(orc, inp, params, kinds)


def test_fp32_needs_the_create_flag(orc):
    from paper_2607_00488_b200 import binding
    inp = wl.make_custom(n_E=20, n_T=64, n_rec=40, seed=65)
    params, kinds = wl.random_points(8, [wl.EPS_EE_L], seed=66)
    ctx = binding.Reweighter(inp, max_batch=8)
    with pytest.raises(binding.RwError):
        ctx.eval_batch(_cuda(params), kinds, mode="gemm", fp32=True)
    ctx.close()
