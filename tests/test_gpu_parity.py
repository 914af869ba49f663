"""GPU parity: the CUDA path through the C ABI vs the CPU oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): mu within 1e-12 relative,
-2lnL within 1e-9 absolute + 1e-12 x sum_k 2|term_k| (conditioning-aware bound, reading T)."""
import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu

MU_RTOL = 1e-12


def m2lnl_tol(abs_scale):
    return 1e-9 + 1e-12 * abs_scale


@pytest.fixture(scope="module")
def rw():
    import torch
    from paper_2607_00488_b200 import binding
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    binding.load_library()
    return binding


def _check(rw, orc, inp, params, kinds, mode, nthreads=8, mu_rows=None, max_batch=None):
    import torch
    P = params.shape[0]
    ref, mu_ref, ab = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=nthreads)
    ctx = rw.Reweighter(inp, max_batch=max_batch or max(1, P))
    out, mu = ctx.eval_batch(torch.from_numpy(params).cuda(), kinds, want_mu=True, mode=mode)
    torch.cuda.synchronize()
    out, mu = out.cpu().numpy(), mu.cpu().numpy()
    ctx.close()
    rel = np.abs(mu - mu_ref) / np.abs(mu_ref)
    assert np.all(rel <= MU_RTOL), "mu rel err max %.3e" % rel.max()
    err = np.abs(out - ref)
    assert np.all(err <= m2lnl_tol(ab)), "-2lnL abs err max %.3e (ref %.6e)" % (err.max(), ref[err.argmax()])
    return err.max(), rel.max()


@pytest.mark.parametrize("mode", ["stream", "gemm", "auto"])
def test_small_ragged_problem(rw, orc, mode):
    """Odd sizes everywhere: n_E=31, n_T=77 (not a multiple of 16), n_rec=53 (odd: padded copy of R),
    2 periods, 37 points (ragged last 16-group / partial 128-row tile), 3 parameter kinds."""
    inp = wl.make_custom(n_E=31, n_T=77, n_rec=53, n_periods=2, seed=5)
    params, kinds = wl.random_points(37, [wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU], seed=6)
    _check(rw, orc, inp, params, kinds, mode)


@pytest.mark.parametrize("mode", ["stream", "gemm"])
def test_multi_tile_problem(rw, orc, mode):
    """Several contraction tiles in every direction with ragged tails: 300 points (3 m-tiles),
    n_rec = 330 (3 n-tiles, last one partial), n_T = 203 (13 k-stages, last partial), dead bins."""
    inp = wl.make_custom(n_E=40, n_T=203, n_rec=330, n_periods=1, seed=7, dead_fraction=0.2)
    params, kinds = wl.random_points(300, list(range(7)), seed=8)
    _check(rw, orc, inp, params, kinds, mode)


@pytest.mark.parametrize("P", [5, 16, 17, 32, 50, 64, 100, 129])
def test_contraction_tile_heights_and_split_k(rw, orc, P):
    """Every tile height of the DMMA contraction (16/32/64/128 points) with a contraction long enough to be
    split into k-ranges (n_T = 1500: 94 stage-iterations, ragged last one), 3 column tiles with a ragged tail,
    2 periods: the parked accumulators of the k-ranges must add up to the oracle's mu."""
    inp = wl.make_custom(n_E=24, n_T=1500, n_rec=330, n_periods=2, seed=17, dead_fraction=0.1)
    params, kinds = wl.random_points(P, list(range(7)), seed=18)
    _check(rw, orc, inp, params, kinds, "gemm")


@pytest.mark.parametrize("mode", ["stream", "gemm"])
def test_config1_all_points(rw, orc, mode):
    inp = wl.make("cfg1_tiny_nsi")
    params, kinds = wl.scan_points("cfg1_tiny_nsi")
    _check(rw, orc, inp, params, kinds, mode)


@pytest.mark.parametrize("mode", ["stream", "gemm"])
def test_config2_all_points(rw, orc, mode):
    inp = wl.make("cfg2_mm_lowE")
    params, kinds = wl.scan_points("cfg2_mm_lowE")
    _check(rw, orc, inp, params, kinds, mode)
