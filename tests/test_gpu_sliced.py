"""Opt-in RW_SLICED contraction (FP64 by slicing on the INT8 tensor cores, exact int32 accumulation) against the
oracle at the FP64 bars of the main path: mu 1e-12 relative, -2lnL 1e-9 + 1e-12 * sum 2|term| (reading T)."""
import os

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 4


def _cuda(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _check(inp, params, kinds, ref, mu_ref, scale, max_batch=None):
    import torch
    from paper_2607_00488_b200 import binding
    ctx = binding.Reweighter(inp, max_batch=max_batch or params.shape[0], sliced=True)
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="gemm", sliced=True)
    out64 = ctx.eval_batch(_cuda(params), kinds, mode="gemm")
    torch.cuda.synchronize()
    out, mu, out64 = out.cpu().numpy(), mu.cpu().numpy(), out64.cpu().numpy()
    ctx.close()
    rel = np.abs(mu - mu_ref) / np.abs(mu_ref)
    assert rel.max() <= 1e-12, "sliced mu rel err %.3e" % rel.max()
    err = np.abs(out - ref)
    assert np.all(err <= 1e-9 + 1e-12 * scale), "sliced -2lnL err %.3e" % err.max()
    assert np.all(np.abs(out64 - ref) <= 1e-9 + 1e-12 * scale)
    return rel.max()


def test_sliced_small_ragged(orc):
    """n_T = 203 (7 k-blocks of 32, ragged), n_rec = 330 (6 column tiles of 64, ragged), 2 periods, 300 points
    (3 point tiles, ragged), all seven parameter kinds, dead bins."""
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=330, n_periods=2, seed=111, dead_fraction=0.1)
    params, kinds = wl.random_points(300, list(range(7)), seed=112)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)


def test_sliced_long_contraction_and_chunks(orc):
    """n_T = 3000 (94 k-blocks; the smem ring wraps many times), several tiles per CTA, P > max_batch."""
    inp = wl.make_custom(n_E=24, n_T=3000, n_rec=200, n_periods=1, seed=113)
    params, kinds = wl.random_points(150, [wl.EPS_EE_L, wl.EPS_EE_R, wl.MU_NU], seed=114)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale, max_batch=64)


def test_sliced_eight_slices_at_their_largest_size(orc):
    """n_T = 2048: the longest contraction that still takes eight balanced 8-bit slices (36 products per k-step)."""
    inp = wl.make_custom(n_E=24, n_T=2048, n_rec=130, n_periods=1, seed=117, tail=0.0)
    params, kinds = wl.random_points(140, [wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU], seed=118)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)


def test_sliced_seven_slices(orc):
    """n_T = 8300: seven balanced 8-bit slices (28 products per k-step, 55 bits below the row / column scale), as for
    every n_T > 2048 (n_T = 3000 and config 2's dead-bin-heavy 1000 x 500 are covered above and below)."""
    inp = wl.make_custom(n_E=24, n_T=8300, n_rec=100, n_periods=1, seed=119, tail=0.0)
    params, kinds = wl.random_points(130, [wl.EPS_EE_L, wl.EPS_MM_R, wl.MU_NU], seed=120)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)


def test_sliced_config2_all_points(orc):
    """Config 2: exact zeros in R, 867 dead recoil bins, mu_nu over two decades."""
    inp = wl.make("cfg2_mm_lowE")
    params, kinds = wl.scan_points("cfg2_mm_lowE")
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)


def test_sliced_components_rates_and_bad_points(orc):
    import torch
    from paper_2607_00488_b200 import binding
    inp = wl.make_components(n_comp=3, n_E=33, n_T=160, n_rec=140, n_periods=2, seed=115)
    kinds = np.array([wl.EPS_EE_L, wl.MU_NU, 7, 9], np.int32)
    params, _ = wl.random_points(70, kinds, seed=116)
    ref, mu_ref, scale = orc.eval_components(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)
    bad = params.copy()
    bad[5, 0] = np.nan
    ctx = binding.Reweighter(inp, max_batch=70, sliced=True)
    out = ctx.eval_batch(_cuda(bad), kinds, mode="gemm", sliced=True)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert np.isnan(out[5]) and np.all(np.isfinite(np.delete(out, 5)))
    plain = binding.Reweighter(inp, max_batch=8)
    with pytest.raises(binding.RwError):
        plain.eval_batch(_cuda(params[:8]), kinds, mode="gemm", sliced=True)
    plain.close()
    ctx.close()


def test_sliced_weights_profile_and_pee(orc):
    """RW_SLICED through the other entry points that feed the dense fold non-negative rows: rw_eval_weights
    (N' = w N_mc sliced from caller weights, a zero-weight stretch and an all-zero row included), rw_eval_profile
    (mu of the sliced fold into the profiling kernel) and rw_eval_pee; rw_eval_grad refuses it (derivative rows
    change sign)."""
    import torch
    from paper_2607_00488_b200 import binding
    inp = wl.make_custom(n_E=300, n_T=203, n_rec=330, n_periods=2, seed=121, dead_fraction=0.1)
    ctx = binding.Reweighter(inp, max_batch=160, sliced=True)
    # weights
    P = 150
    w = np.random.default_rng(122).uniform(0.0, 3.0, size=(P, 203))
    w[0, :7] = 0.0
    w[3] = 0.0
    ref, mu_ref, scale = orc.eval_weights(inp, w, want_mu=True, want_abs=True, nthreads=CORES)
    out, mu = ctx.eval_weights(_cuda(w), want_mu=True, mode="gemm", sliced=True)
    torch.cuda.synchronize()
    out, mu = out.cpu().numpy(), mu.cpu().numpy()
    assert (np.abs(mu - mu_ref) <= 1e-12 * np.abs(mu_ref)).all(), (np.abs(mu - mu_ref) / np.abs(mu_ref)).max()
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-12 * scale)
    # profiled normalisation with a pull
    params, kinds = wl.random_points(45, [wl.EPS_EE_L, wl.EPS_EE_R, wl.EPS_TT_L, wl.MU_NU], seed=123)
    ref, sc_ref, scale = orc.eval_profile(inp, params, kinds, s0=1.0, sigma=0.05, want_abs=True, nthreads=CORES)
    out, sc = ctx.eval_profile(_cuda(params), kinds, s0=1.0, sigma=0.05, mode="gemm", sliced=True)
    torch.cuda.synchronize()
    out, sc = out.cpu().numpy(), sc.cpu().numpy()
    assert np.all(np.abs(sc - sc_ref) <= 1e-10 * np.maximum(sc_ref, 1e-3)), np.abs(sc - sc_ref).max()
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-12 * (scale + np.abs(ref)))
    # survival-probability table per point
    rng = np.random.default_rng(124)
    Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.25, 0.25, size=(45, 300)), 0.0, 1.0)
    ref, mu_ref, scale = orc.eval_pee(inp, params, kinds, Pp, want_mu=True, want_abs=True, nthreads=CORES)
    out, mu = ctx.eval_pee(_cuda(params), kinds, _cuda(Pp), want_mu=True, mode="gemm", sliced=True)
    torch.cuda.synchronize()
    out, mu = out.cpu().numpy(), mu.cpu().numpy()
    assert (np.abs(mu - mu_ref) <= 1e-12 * np.abs(mu_ref)).all(), (np.abs(mu - mu_ref) / np.abs(mu_ref)).max()
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-12 * scale)
    # negative weights cannot be sliced: that point is NaN, the others are unaffected
    wneg = w[:20].copy()
    wneg[4, 10] = -0.5
    out = ctx.eval_weights(_cuda(wneg), mode="gemm", sliced=True)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert np.isnan(out[4]) and np.all(np.isfinite(np.delete(out, 4)))
    # the gradient accepts the sliced contraction (tests/test_gpu_next_rows.py) but not its strict form or RW_FP32
    for bad in ("strict", "fast-strict"):
        with pytest.raises(binding.RwError, match="RW_SLICED_STRICT"):
            ctx.eval_grad(_cuda(params), kinds, sliced=bad)
    ctx.close()


# ------------------------------------------------------------------------------------- RW_SLICED_FAST (FP32 bar)
def _check_fast(orc, inp, params, kinds, max_batch=None, components=False):
    """Top four slices only: mu within 1e-5 relative, -2lnL within the first-order propagation of that bound
    (the bar of tests/test_gpu_fp32.py)."""
    import torch
    from paper_2607_00488_b200 import binding
    fn = orc.eval_components if components else orc.eval_batch
    ref, mu_ref = fn(inp, params, kinds, want_mu=True, nthreads=CORES)
    ctx = binding.Reweighter(inp, max_batch=max_batch or params.shape[0], sliced=True)
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="gemm", sliced="fast")
    torch.cuda.synchronize()
    out, mu = out.cpu().numpy(), mu.cpu().numpy()
    with pytest.raises(binding.RwError):
        ctx.eval_batch(_cuda(params), kinds, mode="gemm", fp32=True, sliced="fast")
    ctx.close()
    rel = np.abs(mu - mu_ref) / np.abs(mu_ref)
    assert rel.max() <= 1e-5, "fast sliced mu rel err %.3e" % rel.max()
    counts = np.asarray(inp["counts"], float).reshape(mu_ref.shape[1:])
    tol = 1e-9 + (2.0 * np.abs(1.0 - counts[None] / mu_ref) * 1e-5 * mu_ref).sum(axis=(1, 2))
    assert np.all(np.abs(out - ref) <= tol), "fast sliced -2lnL err %.3e (tol %.3e)" % (np.abs(out - ref).max(), tol.min())
    return rel.max()


def test_sliced_fast_small_ragged(orc):
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=330, n_periods=2, seed=131, dead_fraction=0.1)
    params, kinds = wl.random_points(300, list(range(7)), seed=132)
    _check_fast(orc, inp, params, kinds)


def test_sliced_fast_long_contraction_seven_slice_layout(orc):
    """n_T = 8300: the operands are stored as 7 slices, the fast mode reads the first 4 of each k-block."""
    inp = wl.make_custom(n_E=24, n_T=8300, n_rec=100, n_periods=1, seed=133, tail=0.0)
    params, kinds = wl.random_points(130, [wl.EPS_EE_L, wl.EPS_MM_R, wl.MU_NU], seed=134)
    _check_fast(orc, inp, params, kinds, max_batch=64)


def test_sliced_fast_config2_and_components(orc):
    inp = wl.make("cfg2_mm_lowE")
    params, kinds = wl.scan_points("cfg2_mm_lowE")
    _check_fast(orc, inp, params, kinds)
    inp = wl.make_components(n_comp=3, n_E=33, n_T=160, n_rec=140, n_periods=2, seed=135)
    kinds = np.array([wl.EPS_EE_L, wl.MU_NU, 7, 9], np.int32)
    params, _ = wl.random_points(70, kinds, seed=136)
    _check_fast(orc, inp, params, kinds, components=True)


def test_sliced_agrees_with_the_dmma_path_on_odd_shapes():
    """Shape sweep around every boundary of the sliced kernels (k-blocks of 32 bins, tiles of 128 points x 128 bins,
    64-column epilogue halves, chunked batches, several periods).  The DMMA path is held to the oracle elsewhere;
    here the sliced, fast-sliced, sliced-weights and sliced-profile results are held to it."""
    import torch
    from paper_2607_00488_b200 import binding
    rng = np.random.default_rng(151)
    shapes = [(1, 1, 5, 1), (2, 3, 6, 2), (31, 63, 17, 1), (32, 64, 127, 3), (33, 65, 128, 1), (64, 127, 129, 2),
              (65, 128, 255, 1), (255, 129, 256, 1), (256, 130, 300, 2), (257, 255, 17, 3), (1000, 256, 128, 1),
              (2047, 257, 129, 1), (2048, 500, 300, 1), (2049, 700, 127, 2)]
    for n_T, n_rec, P, D in shapes:
        inp = wl.make_custom(n_E=int(rng.integers(3, 40)), n_T=n_T, n_rec=n_rec, n_periods=D,
                             seed=int(rng.integers(1, 10**6)), dead_fraction=float(rng.choice([0.0, 0.1])))
        params, kinds = wl.random_points(P, [wl.EPS_EE_L, wl.EPS_EE_R, wl.EPS_TT_L, wl.MU_NU], seed=int(rng.integers(1, 10**6)))
        ctx = binding.Reweighter(inp, max_batch=int(rng.choice([P, max(5, P // 2), 64])), sliced=True)
        p = _cuda(params)
        w = _cuda(rng.uniform(0.0, 2.0, size=(P, n_T)))
        o64, m64 = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm")
        o8, m8 = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced=True)
        _, mf = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced="fast")
        _, mw64 = ctx.eval_weights(w, want_mu=True, mode="gemm")
        _, mw8 = ctx.eval_weights(w, want_mu=True, mode="gemm", sliced=True)
        _, s64 = ctx.eval_profile(p, kinds, mode="gemm")
        _, s8 = ctx.eval_profile(p, kinds, mode="gemm", sliced=True)
        torch.cuda.synchronize()
        tag = "n_T %d n_rec %d P %d D %d" % (n_T, n_rec, P, D)
        assert ((m8 - m64).abs() <= 2e-12 * m64.abs()).all(), tag
        assert ((mf - m64).abs() <= 1e-5 * m64.abs()).all(), tag
        assert ((mw8 - mw64).abs() <= 2e-12 * mw64.abs()).all(), tag
        assert ((o8 - o64).abs() <= 1e-9 + 1e-10 * o64.abs()).all() and bool(torch.isfinite(o8).all()), tag
        assert ((s8 - s64).abs() <= 1e-9 * s64.abs().clamp_min(1e-3)).all(), tag
        ctx.close()


@pytest.mark.parametrize("n_T,n_rec,P,D", [(1, 1, 5, 1), (33, 65, 129, 2), (257, 129, 130, 1)])
def test_sliced_degenerate_and_boundary_shapes_against_the_oracle(orc, n_T, n_rec, P, D):
    """One recoil bin and one reconstructed bin; one bin / one point past a k-block, a tile row and a tile column."""
    inp = wl.make_custom(n_E=9, n_T=n_T, n_rec=n_rec, n_periods=D, seed=161 + n_T)
    params, kinds = wl.random_points(P, [wl.EPS_EE_L, wl.EPS_MM_L, wl.MU_NU], seed=162 + n_T)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)


def test_sliced_contraction_longer_than_one_int32_segment(orc):
    """n_T = 20000 > 16384: the int32 accumulators are drained after 512 k-blocks (16384 bins: 7 pairs x 129 x 128 x
    16384 < 2^31) and the segments are summed in FP64 in the epilogue's registers; both passes, and the fast mode."""
    inp = wl.make_custom(n_E=24, n_T=20000, n_rec=70, n_periods=1, seed=171, tail=0.0)
    params, kinds = wl.random_points(130, [wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU], seed=172)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    _check(inp, params, kinds, ref, mu_ref, scale)
    _check_fast(orc, inp, params, kinds)
