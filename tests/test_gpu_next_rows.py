"""GPU parity of the SURVEY.md section 8(f) rows against the oracle, through the C ABI:
  f-1  RW_MODE_COLLAPSED (rank-K prefolded templates)     vs orc.eval_batch
  f-3  rw_eval_weights (dense fold on caller weights)     vs orc.eval_weights
Same bars as the main path: mu 1e-12 relative, -2lnL 1e-9 + 1e-12 * sum 2|term| (reading T)."""
import os

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 4


@pytest.fixture(scope="module")
def rw():
    import torch
    from paper_2607_00488_b200 import binding
    assert torch.cuda.is_available()
    binding.load_library()
    return binding


def _cuda(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _assert_parity(out, mu, ref, mu_ref, scale):
    rel = np.abs(mu - mu_ref) / np.abs(mu_ref)
    assert rel.max() <= 1e-12, "mu rel err %.3e" % rel.max()
    err = np.abs(out - ref)
    assert np.all(err <= 1e-9 + 1e-12 * scale), "-2lnL err %.3e at %.6e" % (err.max(), ref[err.argmax()])


# ------------------------------------------------------------------------------------- f-1 collapsed
@pytest.mark.parametrize("shape", [dict(n_E=31, n_T=77, n_rec=53, n_periods=2, P=37),
                                   dict(n_E=40, n_T=203, n_rec=1030, n_periods=3, P=300)])
def test_collapsed_mode_small_and_ragged(rw, orc, shape):
    """Odd n_rec (padded template rows), several 512-column strips with a ragged tail, several 64-point
    groups with a ragged tail, several periods, dead bins, all seven parameter kinds."""
    import torch
    P = shape.pop("P")
    inp = wl.make_custom(seed=11, dead_fraction=0.15, **shape)
    params, kinds = wl.random_points(P, list(range(7)), seed=12)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=P)
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="collapsed")
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    # literal Eq. 18 form through the collapsed path
    full = ctx.eval_batch(_cuda(params[:5]), kinds, full_eq18=True, mode="collapsed")
    ref_full = orc.eval_batch(inp, params[:5], kinds, full_eq18=True)
    torch.cuda.synchronize()
    assert np.all(np.abs(full.cpu().numpy() - ref_full) <= 1e-9 + 1e-12 * (scale[:5] + np.abs(ref_full)))
    ctx.close()


@pytest.mark.parametrize("name", ["cfg1_tiny_nsi", "cfg2_mm_lowE"])
def test_collapsed_mode_configs_1_2_all_points(rw, orc, name):
    import torch
    inp = wl.make(name)
    params, kinds = wl.scan_points(name)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=params.shape[0])
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="collapsed")
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    ctx.close()


def test_collapsed_templates_are_the_fold_of_the_prescaled_basis(rw):
    """G[d][b][k] = sum_i W^[d][b][i] R[d][i][k]: the stored templates against a float64 torch matmul of the
    stored pre-scaled basis (both device tables of the same context; property of the setup step)."""
    import torch
    inp = wl.make_custom(n_E=25, n_T=150, n_rec=61, n_periods=2, seed=13)
    ctx = rw.Reweighter(inp, max_batch=4)
    D, n_T, n_rec = inp["R"].shape
    What = ctx.table(rw.RW_TABLE_WHAT).reshape(D, 12, n_T)
    G = ctx.table(rw.RW_TABLE_G).reshape(D, 12, -1)              # one component: [D][1][12][ldG]
    R = _cuda(inp["R"])
    for d in range(D):
        ref = What[d, :11] @ R[d]
        got = G[d, :11, :n_rec]
        assert torch.all((got - ref).abs() <= 1e-13 * ref.abs().max())
        assert torch.all(G[d, :, n_rec:] == 0) and torch.all(G[d, 11] == 0)
    ctx.close()


def test_collapsed_mode_full_config3_sampled(rw, orc):
    """Config 3 at full size (10^4 points, 4096 x 2048) in one call; sampled points against the oracle and all
    points against the dense contraction of the same context."""
    import torch
    inp = wl.make("cfg3_nsi4")
    params, kinds = wl.scan_points("cfg3_nsi4")
    dev_inp = {k: _cuda(inp[k]) for k in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev_inp["f_tau"] = inp["f_tau"]
    ctx = rw.Reweighter(dev_inp, max_batch=10000)
    p_dev = _cuda(params)
    out_c = ctx.eval_batch(p_dev, kinds, mode="collapsed")
    out_g = ctx.eval_batch(p_dev, kinds, mode="gemm")
    torch.cuda.synchronize()
    out_c, out_g = out_c.cpu().numpy(), out_g.cpu().numpy()
    idx = np.unique(np.concatenate([[0, 63, 64, 9999], np.random.default_rng(33).integers(0, 10000, 20)]))
    ref, scale = orc.eval_batch(inp, params[idx], kinds, want_abs=True, nthreads=CORES)
    assert np.all(np.abs(out_c[idx] - ref) <= 1e-9 + 1e-12 * scale)
    assert np.all(np.abs(out_c - out_g) <= 2e-9 + 1e-11 * np.abs(out_g))
    ctx.close()


# ------------------------------------------------------------------------------------- f-3 weights
@pytest.mark.parametrize("mode,P", [("stream", 1), ("stream", 21), ("gemm", 37), ("gemm", 300), ("auto", 33)])
def test_eval_weights_ragged(rw, orc, mode, P):
    """Random (not low-rank) weights; n_T = 203 (partial 64-bin transpose tile and partial k-stage),
    n_rec = 330, 2 periods; ragged 16-point groups / 128-point tiles."""
    import torch
    inp = wl.make_custom(n_E=20, n_T=203, n_rec=330, n_periods=2, seed=21)
    w = np.random.default_rng(22).uniform(0.0, 3.0, size=(P, 203))
    w[0, :7] = 0.0
    ref, mu_ref, scale = orc.eval_weights(inp, w, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=max(P, 1))
    out, mu = ctx.eval_weights(_cuda(w), want_mu=True, mode=mode)
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    ctx.close()


def test_eval_weights_reproduces_eval_batch_and_sm_point(rw, orc):
    """Fed the oracle's spectrum-ratio weights, the weights path gives the oracle's eval_batch numbers;
    w == 1 gives the SM prediction; the Eq. 18 form and chunking (P > max_batch) work."""
    import torch
    inp = wl.make_custom(n_E=31, n_T=77, n_rec=53, n_periods=2, seed=5)
    params, kinds = wl.random_points(40, [wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU], seed=6)
    ref, mu_ref, scale = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    w = np.stack([orc.weights(inp, orc.theta_vector(params[p], kinds)) for p in range(40)])
    ctx = rw.Reweighter(inp, max_batch=16)
    for mode in ("stream", "gemm"):
        out, mu = ctx.eval_weights(_cuda(w), want_mu=True, mode=mode)
        torch.cuda.synchronize()
        # w itself is rounded to binary64 once: 1 ulp on every term
        rel = np.abs(mu.cpu().numpy() - mu_ref) / np.abs(mu_ref)
        assert rel.max() <= 1e-12
        assert np.all(np.abs(out.cpu().numpy() - ref) <= 1e-9 + 2e-12 * scale)
    _, mu1 = ctx.eval_weights(_cuda(np.ones((1, 77))), want_mu=True)
    torch.cuda.synchronize()
    for d in range(2):
        sm = inp["N_mc"][d] @ inp["R"][d] + inp["bkg"][d]
        assert np.all(np.abs(mu1.cpu().numpy()[0, d] / sm - 1) <= 1e-13)
    full = ctx.eval_weights(_cuda(w[:3]), full_eq18=True)
    ref_full = orc.eval_weights(inp, w[:3], full_eq18=True)
    torch.cuda.synchronize()
    assert np.all(np.abs(full.cpu().numpy() - ref_full) <= 1e-9 + 1e-12 * (scale[:3] + np.abs(ref_full)))
    with pytest.raises(rw.RwError):
        ctx.eval_weights(_cuda(w), mode="collapsed")
    ctx.close()


def test_eval_weights_config3_size_sampled(rw, orc):
    """Config-3-sized dense fold on random weights (4096 x 2048, 1000 points through the DMMA contraction,
    8 through the streaming fold); sampled rows against the oracle."""
    import torch
    inp = wl.make("cfg3_nsi4")
    rng = np.random.default_rng(44)
    P = 1000
    w = rng.uniform(0.5, 1.5, size=(P, 4096))
    ctx = rw.Reweighter(inp, max_batch=P)
    out = ctx.eval_weights(_cuda(w))
    out_s = ctx.eval_weights(_cuda(w[:8]), mode="stream")
    torch.cuda.synchronize()
    idx = np.array([0, 1, 7, 127, 128, 999, 500])
    ref, scale = orc.eval_weights(inp, w[idx], want_abs=True, nthreads=CORES)
    assert np.all(np.abs(out.cpu().numpy()[idx] - ref) <= 1e-9 + 1e-12 * scale)
    assert np.all(np.abs(out_s.cpu().numpy()[idx[:3]] - ref[:3]) <= 1e-9 + 1e-12 * scale[:3])
    ctx.close()


# ------------------------------------------------------------------------------------- f-2 profiled normalisation
def _profile_check(rw, orc, inp, params, kinds, mode, s0=1.0, sigma=0.0, max_batch=None):
    import torch
    ref, sc_ref, scale = orc.eval_profile(inp, params, kinds, s0=s0, sigma=sigma, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=max_batch or params.shape[0])
    out, sc = ctx.eval_profile(_cuda(params), kinds, s0=s0, sigma=sigma, mode=mode)
    torch.cuda.synchronize()
    out, sc = out.cpu().numpy(), sc.cpu().numpy()
    ctx.close()
    # the minimiser to 1e-10 relative (the value is flat there), the value to the usual bar (+ the pull term's rounding)
    assert np.all(np.abs(sc - sc_ref) <= 1e-10 * np.maximum(sc_ref, 1e-3)), np.abs(sc - sc_ref).max()
    err = np.abs(out - ref)
    assert np.all(err <= 1e-9 + 1e-12 * (scale + np.abs(ref))), "profiled -2lnL err %.3e" % err.max()
    return out, sc


@pytest.mark.parametrize("mode", ["stream", "gemm", "collapsed"])
def test_profile_ragged_with_and_without_pull(rw, orc, mode):
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=330, n_periods=2, seed=51, dead_fraction=0.1)
    params, kinds = wl.random_points(45, [wl.EPS_EE_L, wl.EPS_EE_R, wl.EPS_TT_L, wl.MU_NU], seed=52)
    out_free, sc_free = _profile_check(rw, orc, inp, params, kinds, mode)
    out_pull, sc_pull = _profile_check(rw, orc, inp, params, kinds, mode, s0=1.0, sigma=0.02, max_batch=16)
    assert np.all(out_pull >= out_free - 1e-9)                       # a constraint never lowers the minimum
    assert np.all(np.abs(sc_pull - 1.0) <= np.abs(sc_free - 1.0) + 1e-12)


def test_profile_asimov_recovery_and_boundary(rw, orc):
    """Asimov data built at (theta*, s* = 1.4) are recovered with value 0 and s^ = s*;
    data below the background give the boundary s^ = 0; the Eq. 18 form adds the saturated constant."""
    import torch
    inp = wl.make_custom(n_E=25, n_T=120, n_rec=90, n_periods=2, seed=53)
    params, kinds = wl.random_points(6, [wl.EPS_EE_L, wl.MU_NU], seed=54)
    _, mu = orc.eval_batch(inp, params, kinds, want_mu=True)
    asim = dict(inp)
    asim["counts"] = 1.4 * (mu[3] - inp["bkg"]) + inp["bkg"]
    out, sc = _profile_check(rw, orc, asim, params, kinds, "gemm")
    assert abs(sc[3] - 1.4) < 1e-10 and abs(out[3]) < 1e-9 and np.all(np.delete(out, 3) > 1e-6)
    low = dict(inp)
    low["counts"] = 0.5 * inp["bkg"]
    out, sc = _profile_check(rw, orc, low, params, kinds, "stream")
    assert np.all(sc == 0.0)
    ctx = rw.Reweighter(inp, max_batch=6)
    full, _ = ctx.eval_profile(_cuda(params), kinds, full_eq18=True)
    plain, _ = ctx.eval_profile(_cuda(params), kinds)
    torch.cuda.synchronize()
    ref_full = orc.eval_profile(inp, params, kinds, full_eq18=True)[0]
    assert np.all(np.abs(full.cpu().numpy() - ref_full) <= 1e-9 * np.abs(ref_full))
    const = (full - plain).cpu().numpy()
    assert np.all(np.abs(const - const[0]) <= 1e-9 * abs(const[0]))
    with pytest.raises(rw.RwError):
        ctx.eval_profile(_cuda(params), kinds, s0=float("nan"))
    ctx.close()


def test_profile_config2_all_points(rw, orc):
    """Config 2 (1000 mu_nu points, 867 dead recoil bins, exact zeros in R): dense and collapsed folds."""
    inp = wl.make("cfg2_mm_lowE")
    params, kinds = wl.scan_points("cfg2_mm_lowE")
    a, _ = _profile_check(rw, orc, inp, params, kinds, "auto")
    b, _ = _profile_check(rw, orc, inp, params, kinds, "collapsed", s0=1.0, sigma=0.1)
    assert np.all(b >= a - 1e-9)


# ------------------------------------------------------------------------------------- f-2 several signal components
@pytest.mark.parametrize("mode,P", [("stream", 3), ("stream", 21), ("gemm", 40), ("gemm", 300), ("auto", 9)])
def test_multi_component_rates(rw, orc, mode, P):
    """Three signal components (own flux tables and survival probabilities, concatenated recoil bins), rate scales of
    components 0 and 2 scanned together with couplings (Eq. 17) against orc.eval_components."""
    import torch
    inp = wl.make_components(n_comp=3, n_E=33, n_T=203, n_rec=330, n_periods=2, seed=71)
    kinds = np.array([wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU, 7, 9], np.int32)
    params, _ = wl.random_points(P, kinds, seed=72)
    ref, mu_ref, scale = orc.eval_components(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=max(P, 16))
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode=mode)
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    # the rank-K identity holds per component (11 n_comp templates, the rates applied to the template sums)
    out_c, mu_c = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="collapsed")
    torch.cuda.synchronize()
    _assert_parity(out_c.cpu().numpy(), mu_c.cpu().numpy(), ref, mu_ref, scale)
    with pytest.raises(rw.RwError):
        ctx.eval_batch(_cuda(params[:, :1]), [10])               # rate of a component that does not exist
    ctx.close()


def test_multi_component_device_tables_profile_and_fp32(rw, orc):
    """Device-resident multi-component tables; the profiled normalisation and the TF32 contraction on top."""
    import torch
    inp = wl.make_components(n_comp=2, n_E=29, n_T=160, n_rec=140, n_periods=1, seed=73)
    kinds = np.array([wl.EPS_EE_R, 8], np.int32)
    params, _ = wl.random_points(50, kinds, seed=74)
    ref, mu_ref, scale = orc.eval_components(inp, params, kinds, want_mu=True, want_abs=True, nthreads=CORES)
    dev = {k: _cuda(inp[k]) for k in ("E", "flux_w", "P_e", "T", "N_mc", "R", "bkg", "counts")}
    dev["comp_of_T"] = torch.from_numpy(inp["comp_of_T"]).cuda()
    dev["f_tau"] = 0.5
    ctx = rw.Reweighter(dev, max_batch=50, fp32=True)
    out, mu = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="gemm")
    out32, mu32 = ctx.eval_batch(_cuda(params), kinds, want_mu=True, mode="gemm", fp32=True)
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    assert (np.abs(mu32.cpu().numpy() - mu_ref) / mu_ref).max() <= 1e-5
    # profiling the overall normalisation on top of fixed relative rates: minimum over s of the oracle's objective
    prof, sc = ctx.eval_profile(_cuda(params[:6]), kinds)
    torch.cuda.synchronize()
    for p in range(6):
        s_ref, f_ref = orc.profile_scale((mu_ref[p] - inp["bkg"]).ravel(), inp["bkg"].ravel(), inp["counts"].ravel())
        assert abs(sc[p].item() - s_ref) <= 1e-10 * s_ref and abs(prof[p].item() - f_ref) <= 1e-9 + 1e-12 * scale[p]
    bad = dict(inp, comp_of_T=np.where(np.arange(160) == 7, 5, inp["comp_of_T"]).astype(np.int32))
    with pytest.raises(rw.RwError, match="comp_of_T"):
        rw.Reweighter(bad, max_batch=4)
    ctx.close()


# ------------------------------------------------------------------------------------- f-2 analytic gradient
def _grad_check(rw, orc, inp, params, kinds, mode, max_batch):
    import torch
    ref, gref = orc.eval_grad(inp, params, kinds, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=max_batch)
    out, grad = ctx.eval_grad(_cuda(params), kinds, mode=mode)
    torch.cuda.synchronize()
    out, grad = out.cpu().numpy(), grad.cpu().numpy()
    ctx.close()
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-11 * np.abs(ref))
    # the derivative rows come back as (d mu + bkg) - bkg: absolute rounding of the background scale per bin
    floor = 1e-11 * np.asarray(inp["bkg"]).sum()
    assert np.all(np.abs(grad - gref) <= 1e-10 * np.abs(gref) + floor), np.abs(grad - gref).max()
    return out, grad


@pytest.mark.parametrize("mode", ["stream", "gemm", "collapsed"])
def test_gradient_single_component(rw, orc, mode):
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=130, n_periods=2, seed=91, dead_fraction=0.1)
    kinds = np.array([0, 1, 4, 5, 6, 7], np.int32)                # couplings, mu_nu and the rate of the component
    params, _ = wl.random_points(23, kinds, seed=92)
    _grad_check(rw, orc, inp, params, kinds, mode, max_batch=64)


def test_gradient_multi_component_and_asimov_zero(rw, orc):
    import torch
    inp = wl.make_components(n_comp=3, n_E=27, n_T=120, n_rec=90, n_periods=1, seed=93)
    kinds = np.array([0, 2, 3, 6, 7, 8, 9], np.int32)
    params, _ = wl.random_points(40, kinds, seed=94)
    _grad_check(rw, orc, inp, params, kinds, "auto", max_batch=300)
    _grad_check(rw, orc, inp, params, kinds, "collapsed", max_batch=300)      # per-component templates, rate derivatives
    _, mu = orc.eval_components(inp, params[:1], kinds, want_mu=True)
    asim = dict(inp, counts=mu[0])
    ctx = rw.Reweighter(asim, max_batch=16)
    out, grad = ctx.eval_grad(_cuda(params[:1]), kinds)
    torch.cuda.synchronize()
    scale = np.abs(orc.eval_grad(inp, params[:1], kinds)[1])
    assert abs(out.item()) < 1e-9 and np.all(np.abs(grad.cpu().numpy()) <= 1e-9 * scale)
    ctx.close()


def test_gradient_through_the_sliced_contraction(rw, orc):
    """RW_SLICED on rw_eval_grad: a derivative row changes sign along the recoil bins, so it is folded as its positive
    and its negative part (1 + 2k rows per point) and k_grad takes the difference.  n_T = 2300 > 2048: seven slices;
    several passes of the row scratch; a last pass small enough for the FP64 streaming kernels (no split there)."""
    import torch
    inp = wl.make_custom(n_E=31, n_T=2300, n_rec=140, n_periods=2, seed=95, dead_fraction=0.1)
    kinds = np.array([0, 1, 2, 5, 6, 7], np.int32)
    params, _ = wl.random_points(43, kinds, seed=96)
    ref, gref = orc.eval_grad(inp, params, kinds, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=14 * 13, sliced=True)        # 14 points per pass (1 + 2*6 rows each); 43 = 3*14 + 1
    floor = 1e-11 * np.asarray(inp["bkg"]).sum()
    for sliced, rel in ((True, 1e-11), ("fast", 1e-5)):
        out, grad = ctx.eval_grad(_cuda(params), kinds, mode="auto", sliced=sliced)
        out_g, grad_g = ctx.eval_grad(_cuda(params), kinds, mode="gemm", sliced=sliced)
        torch.cuda.synchronize()
        for o, g in ((out, grad), (out_g, grad_g)):
            o, g = o.cpu().numpy(), g.cpu().numpy()
            tol_v = 1e-9 + 1e-11 * np.abs(ref) if sliced is True else 1e-4 * np.abs(ref) + 1.0
            assert np.all(np.abs(o - ref) <= tol_v), np.abs(o - ref).max()
            # each part carries the relative error of the contraction on ITS size; the gradient is their difference
            # summed over bins with weights 2 (1 - n/mu): compare on the scale of the whole gradient vector's row
            scale = np.abs(gref) + np.abs(gref).max(axis=1, keepdims=True) * 1e-3
            err = np.abs(g - gref) / scale
            print("grad sliced=%s: max rel err %.2e" % (sliced, err.max()))
            assert np.all(np.abs(g - gref) <= rel * scale + floor), err.max()
    with pytest.raises(rw.RwError, match="RW_SLICED_STRICT"):
        ctx.eval_grad(_cuda(params), kinds, sliced="strict")
    ctx.close()


# ------------------------------------------------------------------------------------- f-3 per-point survival probabilities
@pytest.mark.parametrize("mode,P", [("stream", 3), ("gemm", 45), ("auto", 150), ("auto", 12), ("auto", 40)])
def test_per_point_survival_probability(rw, orc, mode, P):
    """P_ee table per point: spectrum on the (E_nu x T) grid per point (n_E = 300: three staging chunks with a
    ragged tail; dead bins), then the dense fold; against orc.eval_pee."""
    import torch
    inp = wl.make_custom(n_E=300, n_T=203, n_rec=130, n_periods=2, seed=101, dead_fraction=0.15)
    params, kinds = wl.random_points(P, [wl.EPS_EE_L, wl.EPS_EE_R, wl.EPS_TT_L, wl.MU_NU], seed=102)
    rng = np.random.default_rng(103)
    Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.25, 0.25, size=(P, 300)), 0.0, 1.0)
    Pp[0] = inp["P_e"]
    ref, mu_ref, scale = orc.eval_pee(inp, params, kinds, Pp, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=max(P, 16))
    out, mu = ctx.eval_pee(_cuda(params), kinds, _cuda(Pp), want_mu=True, mode=mode)
    plain = ctx.eval_batch(_cuda(params[:1]), kinds)
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    assert abs(plain.item() - out[0].item()) <= 1e-9 + 1e-11 * abs(plain.item())     # nominal table = ordinary path
    with pytest.raises(rw.RwError):
        ctx.eval_pee(_cuda(params), kinds, _cuda(Pp), mode="collapsed")
    ctx.close()


def test_per_point_survival_probability_config3_size(rw, orc):
    """Config-3-sized grids (4096 flux entries x 4096 recoil bins x 2048 rec bins), 40 points with their own tables."""
    import torch
    inp = wl.make("cfg3_nsi4")
    params, kinds = wl.scan_points("cfg3_nsi4")
    params = params[:40]
    rng = np.random.default_rng(104)
    shift = rng.uniform(-0.1, 0.1, size=(40, 1))
    Pp = np.clip(inp["P_e"][None, :] + shift, 0.0, 1.0)
    ctx = rw.Reweighter(inp, max_batch=64)
    out = ctx.eval_pee(_cuda(params), kinds, _cuda(Pp))
    torch.cuda.synchronize()
    idx = np.array([0, 1, 17, 39])
    ref, scale = orc.eval_pee(inp, params[idx], kinds, Pp[idx], want_abs=True, nthreads=CORES)
    assert np.all(np.abs(out.cpu().numpy()[idx] - ref) <= 1e-9 + 1e-12 * scale)
    ctx.close()


def test_per_point_survival_probability_with_a_single_evaluation_context(rw, orc):
    """A context made for single evaluations (max_batch = 1) on a shape with n_T > n_rec: the weights of a pass
    live in the mu scratch, which must hold at least one row of n_T doubles."""
    import torch
    inp = wl.make_custom(n_E=60, n_T=600, n_rec=37, n_periods=1, seed=111)
    params, kinds = wl.random_points(3, [wl.EPS_EE_L, wl.MU_NU], seed=112)
    rng = np.random.default_rng(113)
    Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.2, 0.2, size=(3, 60)), 0.0, 1.0)
    ref, mu_ref, scale = orc.eval_pee(inp, params, kinds, Pp, want_mu=True, want_abs=True)
    for mb in (1, 2):
        ctx = rw.Reweighter(inp, max_batch=mb)
        out, mu = ctx.eval_pee(_cuda(params), kinds, _cuda(Pp), want_mu=True)      # 3 points => passes of mb
        torch.cuda.synchronize()
        _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
        ctx.close()


@pytest.mark.parametrize("explicit", [False, True])
def test_per_point_survival_probability_components_and_explicit_tables(rw, orc, explicit):
    """rw_eval_pee with three signal components (their own flux / survival tables, P_e_pts[P][3][n_E]) and, when
    `explicit`, nominal nu_mu / nu_tau tables whose mu : tau ratio every point keeps (reading R17); against
    orc.eval_pee_components.  The flux grid is NOT sorted (a line is appended last): the sorted-grid scan must not care."""
    import torch
    inp = wl.make_components(n_comp=3, n_E=150, n_T=240, n_rec=130, n_periods=2, seed=121)
    rng = np.random.default_rng(122)
    if explicit:
        frac = rng.uniform(0.2, 0.8, size=inp["P_e"].shape)
        inp["P_mu"] = (1.0 - inp["P_e"]) * frac
        inp["P_tau"] = (1.0 - inp["P_e"]) * (1.0 - frac)
    P = 37
    params, kinds = wl.random_points(P, [wl.EPS_EE_L, wl.EPS_MM_R, wl.EPS_TT_L, wl.MU_NU], seed=123)
    pts = np.clip(inp["P_e"][None] + rng.uniform(-0.25, 0.25, size=(P, 3, 150)), 0.0, 1.0)
    pts[0] = inp["P_e"]
    ref, mu_ref, scale = orc.eval_pee_components(inp, params, kinds, pts, want_mu=True, want_abs=True, nthreads=CORES)
    ctx = rw.Reweighter(inp, max_batch=64)
    out, mu = ctx.eval_pee(_cuda(params), kinds, _cuda(pts), want_mu=True)
    plain = ctx.eval_batch(_cuda(params[:1]), kinds)
    torch.cuda.synchronize()
    _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    assert abs(plain.item() - out[0].item()) <= 1e-9 + 1e-11 * abs(plain.item())     # nominal tables = ordinary path
    ctx.close()


def test_per_point_survival_probability_two_live_contexts_of_different_flux_grids(rw, orc):
    """k_pee_scan keeps its three suffix sums in dynamic shared memory: 3 (n_E + 1) doubles, 62 KB at n_E = 2600 -- more than
    the 48 KB a kernel gets without cudaFuncAttributeMaxDynamicSharedMemorySize.  That attribute belongs to the function,
    not to a context: a context created LATER with a small flux grid must not lower it under the first one."""
    import torch
    big = wl.make_custom(n_E=2600, n_T=90, n_rec=70, n_periods=1, seed=131)
    small = wl.make_custom(n_E=120, n_T=77, n_rec=53, n_periods=1, seed=132)
    kin = [wl.EPS_EE_L, wl.EPS_TT_R, wl.MU_NU]
    rng = np.random.default_rng(133)
    cases = []
    for inp, P, seed in ((big, 9, 134), (small, 7, 135)):
        params, kinds = wl.random_points(P, kin, seed=seed)
        Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.2, 0.2, size=(P, inp["E"].size)), 0.0, 1.0)
        cases.append((inp, params, kinds, Pp) + orc.eval_pee(inp, params, kinds, Pp, want_mu=True, want_abs=True, nthreads=CORES))
    ctx_big = rw.Reweighter(big, max_batch=16)
    ctx_small = rw.Reweighter(small, max_batch=16)          # created second: its rw_create sets the attribute last
    for _ in range(2):                                      # alternately, twice
        for ctx, (inp, params, kinds, Pp, ref, mu_ref, scale) in zip((ctx_big, ctx_small), cases):
            out, mu = ctx.eval_pee(_cuda(params), kinds, _cuda(Pp), want_mu=True)
            torch.cuda.synchronize()
            _assert_parity(out.cpu().numpy(), mu.cpu().numpy(), ref, mu_ref, scale)
    ctx_small.close()
    ctx_big.close()
