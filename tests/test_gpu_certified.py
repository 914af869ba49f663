"""The sliced (INT8 tensor-core) contraction made certifiable: rw_eval_certified returns a rigorous
per-point bound on max_k |mu~ - mu| / mu, and RW_SLICED_STRICT / RW_FP32 recompute every point whose bound exceeds the
bar of the mode in FP64.  Checked against the CPU oracle on inputs built to break a scale-relative fixed point:
columns whose large entries meet empty recoil bins, weights spanning > 1e6, near-identity responses, one-entry columns."""
import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu


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


def _mu_rel(mu, mu_ref):
    return np.abs(mu - mu_ref) / np.abs(mu_ref)


def _run_case(rw, orc, inp, params, kinds, label, expect_fallback=None):
    """(1) plain sliced + certificate: the measured error of every point is below its certified bound;
    (2) strict: every mu within 1e-12 of the oracle, -2lnL within the usual bar; (3) fast-strict / RW_FP32: 1e-5."""
    import torch
    P = params.shape[0]
    ref, mu_ref, ab = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True, nthreads=8)
    ctx = rw.Reweighter(inp, max_batch=max(P, 8), sliced=True)
    p = _cuda(params)
    for sliced, bar in ((True, 1e-12), ("fast", 1e-5)):
        out, bound = ctx.eval_certified(p, kinds, sliced=sliced, mode="gemm")
        _, mu = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced=sliced)
        torch.cuda.synchronize()
        bound, mu = bound.cpu().numpy(), mu.cpu().numpy()
        ok = np.isfinite(mu).all(axis=(1, 2))                       # rows the slicer refused come back NaN: bound = inf
        assert np.all(np.isinf(bound[~ok]))
        worst = _mu_rel(mu[ok], mu_ref[ok]).max(axis=(1, 2))
        # the certificate is a BOUND (2e-13: the oracle-vs-FP64 rounding of N' itself, common to every GPU path)
        assert np.all(worst <= bound[ok] + 2e-13), "%s %s: error %.3e above its certified bound %.3e" % (
            label, sliced, worst.max(), bound[ok][worst.argmax()])
        print("%s [%s]: measured max %.2e, certified max %.2e, points over the %.0e bar: %d of %d" % (
            label, sliced, worst.max() if ok.any() else np.nan, bound.max(), bar, int((bound > bar).sum()), P))
    before = ctx.strict_fallback_count()
    out_s, mu_s = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced="strict")
    out_s2 = ctx.eval_batch(p, kinds, mode="gemm", sliced="strict")             # without mu: per-point fallback path
    out_c, bound_c = ctx.eval_certified(p, kinds, sliced="strict", mode="gemm")
    torch.cuda.synchronize()
    fired = ctx.strict_fallback_count() - before
    assert _mu_rel(mu_s.cpu().numpy(), mu_ref).max() <= 1e-12, "%s strict: mu off by %.3e" % (label, _mu_rel(mu_s.cpu().numpy(), mu_ref).max())
    for o in (out_s, out_s2, out_c):
        assert np.all(np.abs(o.cpu().numpy() - ref) <= 1e-9 + 1e-12 * ab), label
    assert np.all(bound_c.cpu().numpy() <= 1e-12)                   # what is left either certified or recomputed (0)
    if expect_fallback is not None:
        assert (fired > 0) == expect_fallback, "%s: strict fallbacks fired = %d" % (label, fired)
    out_f, mu_f = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", fp32=True)  # RW_FP32 = fast + strict at 1e-5
    torch.cuda.synchronize()
    assert _mu_rel(mu_f.cpu().numpy(), mu_ref).max() <= 1e-5, label
    ctx.close()
    return fired


def test_baseline_shaped_input_certifies_without_fallback(rw, orc):
    """A smooth Gaussian response with a flat tail and NSI-sized weights: everything certifies, nothing is recomputed."""
    inp = wl.make_custom(n_E=24, n_T=2500, n_rec=300, n_periods=2, seed=301)
    params, kinds = wl.random_points(40, [0, 1, 4, 5], seed=302)
    _run_case(rw, orc, inp, params, kinds, "smooth", expect_fallback=False)


def test_column_whose_large_entries_meet_empty_recoil_bins(rw, orc):
    """Columns 5..9 of R are dominated (x 1e13) by recoil bins in which the MC spectrum is empty: their mu is made of
    the tiny entries, far below the column's fixed-point resolution, and there is no background to hide behind."""
    inp = wl.make_custom(n_E=24, n_T=2300, n_rec=140, n_periods=1, seed=311, tail=0.0)
    inp["N_mc"][0, 1800:] = 0.0                                     # empty recoil bins (N' = 0 there)
    inp["R"][0][:1800, 5:10] *= 1e-13                              # what the live bins send into these columns: tiny
    inp["R"][0][1800:, 5:10] = 0.4                                 # ... next to large entries that meet N' = 0
    inp["bkg"][0, 5:10] = 0.0
    inp["counts"][0, 5:10] = 0.0
    params, kinds = wl.random_points(24, [0, 1, 6], seed=312)
    _run_case(rw, orc, inp, params, kinds, "empty-bins", expect_fallback=True)


def test_weights_spanning_six_decades_with_seven_slices(rw, orc):
    """mu_nu up to 3e-8 mu_B on a logarithmic recoil grid from 10 eV to 18 MeV: the 1/T enhancement of Eq. (8) makes the
    weights span > 1e6 along a row (n_T = 4100 > 2048: seven slices), so the high-energy columns sit far below the
    row's fixed-point scale."""
    inp = wl.make_custom(n_E=20, n_T=4100, n_rec=200, n_periods=1, seed=321, tail=0.0)
    inp["T"] = np.logspace(-5.0, 1.25, 4100)                       # representative recoil energies, 10 eV .. 17.8 MeV
    inp["E"] = np.linspace(0.3, 21.0, 20)
    inp["bkg"][:] = 0.01
    params = np.zeros((12, 2))
    params[:, 0] = np.linspace(-0.3, 0.3, 12)
    params[:, 1] = np.logspace(-9, -7.5, 12)
    kinds = np.array([wl.EPS_EE_L, wl.MU_NU], np.int32)
    w = np.array([orc.weights(inp, orc.theta_vector(params[-1], kinds))])
    live = w[0][np.isfinite(w[0]) & (w[0] > 0)]
    assert live.max() / live.min() > 1e6, "the test wants weights spanning six decades, got %.1e" % (live.max() / live.min())
    _run_case(rw, orc, inp, params, kinds, "wide-weights")


def test_near_identity_response_and_single_entry_columns(rw, orc):
    """sigma -> 0: R is (efficiency x) a permutation-like band, every column has one or two entries; column 7 has exactly
    one.  mu_k is then a single product, and the certificate is as tight as it gets."""
    rng = np.random.default_rng(331)
    n_T = n_rec = 260
    inp = wl.make_custom(n_E=24, n_T=n_T, n_rec=n_rec, n_periods=1, seed=332)
    R = np.zeros((n_T, n_rec))
    idx = np.arange(n_T)
    R[idx, idx] = rng.uniform(0.5, 0.9, n_T)
    R[idx[:-1], idx[:-1] + 1] = rng.uniform(0.0, 0.1, n_T - 1)
    R[6, 7] = 0.0                                                   # column 7 keeps its diagonal entry only
    inp["R"] = R[None]
    params, kinds = wl.random_points(30, [0, 1, 2, 3, 4, 5, 6], seed=333)
    _run_case(rw, orc, inp, params, kinds, "near-identity")


def test_strict_weights_path_and_flag_errors(rw, orc):
    """rw_eval_weights with RW_SLICED_STRICT: a chunk with an uncertified point is recomputed as a whole in FP64.
    Flag misuse is an error, not a silent downgrade."""
    import torch
    inp = wl.make_custom(n_E=24, n_T=600, n_rec=130, n_periods=1, seed=341, tail=0.0)
    rng = np.random.default_rng(342)
    w = rng.uniform(0.5, 2.0, size=(70, 600))
    w[:, 300:] *= 1e-9                                              # half of every row nine decades down
    inp["bkg"][:] = 1e-9                                            # ... and no background to hide the columns they feed
    inp["counts"][:] = 0.0                                          # (n >> mu would only test log1p near -1, in every path)
    ref, mu_ref, ab = orc.eval_weights(inp, w, want_mu=True, want_abs=True)
    ctx = rw.Reweighter(inp, max_batch=128, sliced=True)
    before = ctx.strict_fallback_count()
    out, mu = ctx.eval_weights(_cuda(w), want_mu=True, mode="gemm", sliced="strict")
    torch.cuda.synchronize()
    assert _mu_rel(mu.cpu().numpy(), mu_ref).max() <= 1e-12
    assert np.all(np.abs(out.cpu().numpy() - ref) <= 1e-9 + 1e-12 * ab)
    fired = ctx.strict_fallback_count() - before
    print("weights path: strict fallbacks fired for %d of 70 points" % fired)
    assert fired > 0
    params, kinds = wl.random_points(8, [0], seed=343)
    with pytest.raises(rw.RwError, match="RW_SLICED_STRICT"):
        ctx._check(ctx._L.rw_eval_batch(ctx._ctx, _cuda(params).data_ptr(), 8, 1, (rw.C.c_int32 * 1)(0),
                                        torch.empty(8, dtype=torch.float64, device="cuda").data_ptr(), None,
                                        rw.RW_SLICED_STRICT, None), ctx._ctx)
    with pytest.raises(rw.RwError):
        ctx.eval_certified(_cuda(params), kinds, sliced=False)       # an FP64 path has no input-dependent bound
    plain = rw.Reweighter(inp, max_batch=16)
    with pytest.raises(rw.RwError, match="RW_CREATE_SLICED"):
        plain.eval_batch(_cuda(params), kinds, mode="gemm", sliced="strict")
    plain.close()
    ctx.close()


def test_entries_below_the_fixed_point_resolution_are_charged_to_the_bound(rw):
    """Columns 5..9: three large entries (0.4) in recoil bins where the MC spectrum is empty (N' = 0 there, so they add
    nothing to mu but set the column's fixed-point scale), and a floor of 2^-68 in all 2260 live bins -- below the
    resolution 2^-58 of the seven-slice fixed point even after the rescaling by 2^tau = 512, so every one of them is
    rounded to zero and the column's whole signal (~2e-15 on a background of 2e-4: ~1e-11 relative) is lost.  The bound
    must own up to that: measured error <= certified bound with NO slack, against the FP64 DMMA path (same N', so the
    oracle-vs-GPU rounding of N' does not enter), and the strict mode must recompute these points."""
    import torch
    inp = wl.make_custom(n_E=24, n_T=2300, n_rec=140, n_periods=1, seed=331, tail=0.0)
    inp["N_mc"][0, :2260] = 256.0
    inp["N_mc"][0, 2260:] = 0.0                                     # tau = 0 for the last bins (33-bin window all empty)
    inp["R"][0][:, 5:10] = 0.0
    inp["R"][0][:2260, 5:10] = 2.0 ** -68
    inp["R"][0][-3:, 5:10] = 0.4
    inp["bkg"][0, 5:10] = 2e-4
    inp["counts"][0, 5:10] = 0.0
    params, kinds = wl.random_points(24, [0, 1, 6], seed=332)
    ctx = rw.Reweighter(inp, max_batch=32, sliced=True)
    p = _cuda(params)
    _, mu64 = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm")
    _, mu8 = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced=True)
    _, bound = ctx.eval_certified(p, kinds, sliced=True, mode="gemm")
    torch.cuda.synchronize()
    mu64, mu8, bound = mu64.cpu().numpy(), mu8.cpu().numpy(), bound.cpu().numpy()
    worst = _mu_rel(mu8, mu64).max(axis=(1, 2))
    lost = _mu_rel(mu8[:, 0, 5:10], mu64[:, 0, 5:10]).max(axis=1)
    assert np.all(lost > 1e-12), "the construction must lose the floor: %.3e" % lost.min()
    assert np.all(worst <= bound), "error %.3e above its certified bound %.3e" % (worst.max(), bound[worst.argmax()])
    before = ctx.strict_fallback_count()
    _, mu_s = ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced="strict")
    torch.cuda.synchronize()
    assert ctx.strict_fallback_count() - before == 24               # every point holds such columns
    assert _mu_rel(mu_s.cpu().numpy(), mu64).max() <= 1e-14
    ctx.close()
