"""GPU edge cases and invariants through the C ABI (all compared with the oracle or with exact
properties): empty / single / sliced batches, n = 0 bins, mu = 0 < n, NaN parameters, the literal
Eq. (18) form, Asimov re-scans, host-buffer path, explicit flavour tables, constant overrides,
input validation."""
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


def _tol(scale):
    return 1e-9 + 1e-12 * scale


def _cuda(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def test_empty_single_and_sliced_batches(rw, orc):
    import torch
    inp = wl.make_custom(n_E=25, n_T=50, n_rec=34, n_periods=2, seed=21)
    params, kinds = wl.random_points(300, [0, 1, 6], seed=22)
    ref, scale = orc.eval_batch(inp, params, kinds, want_abs=True, nthreads=8)
    ctx = rw.Reweighter(inp, max_batch=64)          # 300 points => 4 slices of 64 + one of 44
    out = ctx.eval_batch(_cuda(params), kinds)
    torch.cuda.synchronize()
    assert np.all(np.abs(out.cpu().numpy() - ref) <= _tol(scale))
    out1 = ctx.eval_batch(_cuda(params[:1]), kinds)                 # single evaluation
    out1g = ctx.eval_batch(_cuda(params[:1]), kinds, mode="gemm")
    torch.cuda.synchronize()
    assert abs(out1.item() - ref[0]) <= _tol(scale[0]) and abs(out1g.item() - ref[0]) <= _tol(scale[0])
    empty = ctx.eval_batch(torch.empty((0, 3), dtype=torch.float64, device="cuda"), kinds)   # P = 0: no-op
    assert empty.numel() == 0
    # k = 0: every point is the SM point
    sm = ctx.eval_batch(torch.empty((5, 0), dtype=torch.float64, device="cuda"), [])
    torch.cuda.synchronize()
    ref0 = orc.eval_batch(inp, np.zeros((1, 1)), [0])
    assert np.all(np.abs(sm.cpu().numpy() - ref0[0]) <= 1e-9)
    ctx.close()


def test_sm_point_weights_are_one_and_mu_is_sm_prediction(rw, orc):
    import torch
    inp = wl.make_custom(n_E=25, n_T=96, n_rec=40, n_periods=1, seed=23, dead_fraction=0.3)
    ctx = rw.Reweighter(inp, max_batch=8)
    for mode in ("stream", "gemm"):
        _, mu = ctx.eval_batch(_cuda(np.zeros((1, 2))), [0, 6], want_mu=True, mode=mode)
        torch.cuda.synchronize()
        ref = inp["N_mc"][0] @ inp["R"][0] + inp["bkg"][0]
        assert np.all(np.abs(mu.cpu().numpy()[0, 0] / ref - 1) < 1e-14)
    S = ctx.table(rw.RW_TABLE_S_SM).cpu().numpy()
    S_ref = orc.spectrum(inp, np.zeros(7))
    assert np.array_equal(S == 0.0, S_ref == 0.0) and np.any(S == 0.0)      # same dead bins (same cut)
    live = S_ref > 0
    assert np.all(np.abs(S[live] / S_ref[live] - 1) < 1e-14)
    ctx.close()


def test_zero_count_bins_zero_mu_and_nan_parameters(rw, orc):
    import torch
    inp = wl.make_custom(n_E=25, n_T=48, n_rec=32, n_periods=1, seed=24)
    inp["counts"][0, :5] = 0.0                       # n = 0 => term = mu
    params, kinds = wl.random_points(20, [0, 4], seed=25)
    ref, scale = orc.eval_batch(inp, params, kinds, want_abs=True)
    ctx = rw.Reweighter(inp, max_batch=32)
    for mode in ("stream", "gemm"):
        out = ctx.eval_batch(_cuda(params), kinds, mode=mode)
        torch.cuda.synchronize()
        assert np.all(np.abs(out.cpu().numpy() - ref) <= _tol(scale))
    bad = params.copy()
    bad[3, 0] = np.nan
    bad[7, 1] = np.inf
    for mode in ("stream", "gemm"):
        out = ctx.eval_batch(_cuda(bad), kinds, mode=mode).cpu().numpy()
        assert np.isnan(out[3]) and not np.isfinite(out[7])
        ok = np.ones(20, bool)
        ok[[3, 7]] = False
        assert np.all(np.abs(out[ok] - ref[ok]) <= _tol(scale[ok]))          # only those points are affected
    ctx.close()
    # a reconstructed bin that nothing reaches and that has no background: mu = 0 with n > 0 => +inf
    dead = dict(inp, R=inp["R"].copy(), bkg=inp["bkg"].copy(), counts=inp["counts"].copy())
    dead["R"][0][:, 9] = 0.0
    dead["bkg"][0, 9] = 0.0
    dead["counts"][0, 9] = 3.0
    assert orc.eval_batch(dead, params[:2], kinds)[0] == np.inf
    ctx = rw.Reweighter(dead, max_batch=32)
    for mode in ("stream", "gemm"):
        out = ctx.eval_batch(_cuda(params[:2]), kinds, mode=mode).cpu().numpy()
        assert np.all(out == np.inf)
    dead["counts"][0, 9] = 0.0                       # mu = 0, n = 0 => contributes 0
    ctx.set_counts(dead["counts"])
    out = ctx.eval_batch(_cuda(params[:2]), kinds).cpu().numpy()
    assert np.all(np.abs(out - orc.eval_batch(dead, params[:2], kinds)) <= 1e-9)
    ctx.close()


def test_full_eq18_form_and_asimov_rescan(rw, orc):
    import torch
    inp = wl.make("cfg1_tiny_nsi")
    params, kinds = wl.scan_points("cfg1_tiny_nsi")
    ctx = rw.Reweighter(inp, max_batch=121)
    full = ctx.eval_batch(_cuda(params), kinds, full_eq18=True).cpu().numpy()
    ref_full = orc.eval_batch(inp, params, kinds, full_eq18=True, nthreads=4)
    assert np.all(np.abs(full - ref_full) <= 1e-9 + 1e-12 * np.abs(ref_full))
    # Asimov data at the injected point of PAPER.md:311 => minimum of the scan there, value 0
    inj = np.array([[0.05, 0.0]])
    _, mu = ctx.eval_batch(_cuda(inj), kinds, want_mu=True)
    ctx.set_counts(mu[0])                           # device tensor, non-integer counts
    scan = np.stack([np.linspace(-0.05, 0.15, 41), np.zeros(41)], axis=1)
    out = ctx.eval_batch(_cuda(scan), kinds).cpu().numpy()
    assert np.argmin(out) == 20 and abs(out[20]) < 1e-9 and np.all(np.delete(out, 20) > 1e-6)
    _, mu_o = orc.eval_batch(inp, inj, kinds, want_mu=True)
    ref = orc.eval_batch(dict(inp, counts=mu_o[0]), scan, kinds)
    assert np.all(np.abs(out - ref) <= 1e-9 + 1e-9 * np.abs(ref))
    ctx.close()


def test_host_buffer_path_matches_device_path(rw, orc):
    import torch
    inp = wl.make_custom(n_E=25, n_T=64, n_rec=48, n_periods=2, seed=26)
    params, kinds = wl.random_points(150, [1, 2, 6], seed=27)
    ctx = rw.Reweighter(inp, max_batch=150)
    dev = ctx.eval_batch(_cuda(params), kinds).cpu().numpy()
    host = ctx.eval_batch(params, kinds)            # numpy in, pinned CPU tensor out
    torch.cuda.synchronize()
    assert isinstance(host, torch.Tensor) and not host.is_cuda
    assert np.array_equal(host.numpy(), dev)
    ctx.close()


def test_device_tables_equal_host_tables_and_explicit_flavours(rw, orc):
    import torch
    inp = wl.make_custom(n_E=25, n_T=64, n_rec=48, n_periods=1, seed=28)      # even n_rec: R is borrowed
    rng = np.random.default_rng(29)
    P_mu = (1 - inp["P_e"]) * rng.uniform(0.2, 0.8, inp["E"].size)
    inp2 = dict(inp, P_mu=P_mu, P_tau=1 - inp["P_e"] - P_mu)
    params, kinds = wl.random_points(40, [2, 3, 4, 5], seed=30)
    ref, scale = orc.eval_batch(inp2, params, kinds, want_abs=True, nthreads=4)
    host_ctx = rw.Reweighter(inp2, max_batch=64)
    dev_inp = {k: _cuda(v) for k, v in inp2.items() if isinstance(v, np.ndarray) and k != "rec_edges" and k != "exposure"}
    dev_ctx = rw.Reweighter(dev_inp, max_batch=64)
    a = host_ctx.eval_batch(_cuda(params), kinds).cpu().numpy()
    b = dev_ctx.eval_batch(_cuda(params), kinds).cpu().numpy()
    assert np.array_equal(a, b)
    assert np.all(np.abs(a - ref) <= _tol(scale))
    host_ctx.close()
    dev_ctx.close()


def test_constant_overrides(rw, orc):
    inp = wl.make_custom(n_E=25, n_T=48, n_rec=32, n_periods=1, seed=31)
    params, kinds = wl.random_points(10, [0, 6], seed=32)
    c = orc.default_consts()
    c.sin2_theta_w, c.alpha_em = 0.2386, 1 / 128.0
    ref, scale = orc.eval_batch(inp, params, kinds, want_abs=True, consts=c)
    ctx = rw.Reweighter(inp, max_batch=16, consts={"sin2_theta_w": 0.2386, "alpha_em": 1 / 128.0})
    out = ctx.eval_batch(_cuda(params), kinds).cpu().numpy()
    assert np.all(np.abs(out - ref) <= _tol(scale))
    assert np.any(np.abs(out - orc.eval_batch(inp, params, kinds)) > 1e-6)     # the override matters
    ctx.close()


def test_invalid_inputs_are_reported_not_computed(rw):
    inp = wl.make_custom(n_E=25, n_T=48, n_rec=32, n_periods=1, seed=33)
    for key, val, msg in (("T", -1.0, "T_MeV"), ("R", -0.5, "R must"), ("counts", np.nan, "counts"),
                          ("E", 0.0, "E_MeV"), ("P_e", 1.5, "P_e")):
        bad = dict(inp)
        bad[key] = inp[key].copy()
        bad[key].reshape(-1)[3] = val
        with pytest.raises(rw.RwError, match=msg):
            rw.Reweighter(bad, max_batch=8)
        dev_bad = {k: _cuda(v) for k, v in bad.items() if isinstance(v, np.ndarray) and k not in ("rec_edges", "exposure")}
        with pytest.raises(rw.RwError, match=msg):
            rw.Reweighter(dev_bad, max_batch=8)
    ctx = rw.Reweighter(inp, max_batch=8)
    with pytest.raises(rw.RwError, match="duplicate"):
        ctx.eval_batch(_cuda(np.zeros((2, 2))), [0, 0])
    with pytest.raises(rw.RwError, match="out of range"):
        ctx.eval_batch(_cuda(np.zeros((2, 1))), [9])
    with pytest.raises(rw.RwError, match="counts"):
        ctx.set_counts(-np.ones((1, 32)))
    ctx.close()


def test_symmetries_hold_on_the_gpu(rw, orc):
    """Exact partner points: eps -> -2g - eps per flavour (chirality flip) and mu_nu -> -mu_nu."""
    inp = wl.make_custom(n_E=25, n_T=64, n_rec=48, n_periods=1, seed=34)
    gL, gR = orc.sm_couplings()
    a = np.array([[0.11, -0.23, 2e-11], [-2 * gL[0] - 0.11, -2 * gR[0] + 0.23, -2e-11]])
    ctx = rw.Reweighter(inp, max_batch=8)
    for mode in ("stream", "gemm"):
        out = ctx.eval_batch(_cuda(a), [0, 1, 6], mode=mode).cpu().numpy()
        assert abs(out[0] - out[1]) <= 1e-9 + 1e-12 * abs(out[0])
    ctx.close()


def test_eval_batch_is_cuda_graph_capturable(rw, orc):
    """rw_eval_batch only enqueues work (no allocation, no synchronisation): a minimiser loop can capture it in a
    CUDA graph and replay it with new parameters written into the same device buffer."""
    import torch
    inp = wl.make("cfg1_tiny_nsi")
    params, kinds = wl.scan_points("cfg1_tiny_nsi")
    ref = orc.eval_batch(inp, params, kinds, nthreads=4)
    ctx = rw.Reweighter(inp, max_batch=121, sliced=True)
    for P, mode in ((1, "auto"), (121, "auto"), (121, "collapsed"), (121, "sliced")):
        buf = _cuda(params[:P].copy())
        out = torch.empty(P, dtype=torch.float64, device="cuda")
        kw = dict(mode="gemm", sliced=True) if mode == "sliced" else dict(mode=mode)
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            ctx.eval_batch(buf, kinds, out=out, **kw)               # warm-up outside capture
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            ctx.eval_batch(buf, kinds, out=out, **kw)
        for lo in (0, 60):                                           # replay with other points in the same buffer
            sel = np.arange(lo, lo + P) % 121
            buf.copy_(_cuda(params[sel]))
            g.replay()
            torch.cuda.synchronize()
            assert np.all(np.abs(out.cpu().numpy() - ref[sel]) <= 1e-9), (P, mode)
    ctx.close()


def test_every_regime_is_bit_reproducible_run_to_run(rw):
    """The design has no floating-point atomics: reductions across tiles, k-ranges, row ranges and periods run in a
    fixed order (tickets only decide WHO sums).  The same call twice must therefore give the same bits, in every
    regime: streaming (1, 4 and 16 points per launch), DMMA contraction with and without split-K, collapsed, TF32 x 3,
    sliced, fast sliced, profile, gradient."""
    import torch
    inp = wl.make_custom(n_E=31, n_T=1500, n_rec=700, n_periods=2, seed=141, dead_fraction=0.05)
    params, kinds = wl.random_points(700, [wl.EPS_EE_L, wl.EPS_EE_R, wl.EPS_TT_L, wl.MU_NU], seed=142)
    ctx = rw.Reweighter(inp, max_batch=512, fp32=True, sliced=True)
    p = _cuda(params)

    def twice(fn):
        a = fn()
        torch.cuda.synchronize()
        a = [t.clone() for t in (a if isinstance(a, tuple) else (a,))]
        b = fn()
        torch.cuda.synchronize()
        b = b if isinstance(b, tuple) else (b,)
        for x, y in zip(a, b):
            assert torch.equal(x, y)

    for n, mode in ((1, "stream"), (4, "stream"), (16, "stream"), (16, "gemm"), (40, "gemm"), (300, "gemm"),
                    (700, "gemm"), (700, "collapsed")):
        twice(lambda: ctx.eval_batch(p[:n], kinds, want_mu=True, mode=mode))
    twice(lambda: ctx.eval_batch(p, kinds, mode="gemm", fp32=True))
    twice(lambda: ctx.eval_batch(p, kinds, want_mu=True, mode="gemm", sliced=True))
    twice(lambda: ctx.eval_batch(p, kinds, mode="gemm", sliced="fast"))
    twice(lambda: ctx.eval_profile(p[:200], kinds, s0=1.0, sigma=0.1))
    twice(lambda: ctx.eval_grad(p[:100], kinds))
    ctx.close()


def test_rejected_device_counts_leave_the_context_unchanged(rw, orc):
    """rw_set_counts validates a device array before it touches the context: after RW_ERR_INVALID the old counts
    and the old saturated constant (literal Eq. 18) are still in force."""
    import torch
    inp = wl.make_custom(n_E=25, n_T=48, n_rec=32, n_periods=1, seed=24)
    params, kinds = wl.random_points(6, [0, 4], seed=25)
    ctx = rw.Reweighter(inp, max_batch=8)
    before = ctx.eval_batch(_cuda(params), kinds, full_eq18=True).cpu().numpy()
    bad = torch.full((1, 32), 3.0, dtype=torch.float64, device="cuda")
    bad[0, 5] = -1.0
    with pytest.raises(rw.RwError):
        ctx.set_counts(bad)
    bad[0, 5] = float("nan")
    with pytest.raises(rw.RwError):
        ctx.set_counts(bad)
    after = ctx.eval_batch(_cuda(params), kinds, full_eq18=True).cpu().numpy()
    assert np.array_equal(before, after)
    ref = orc.eval_batch(inp, params, kinds, full_eq18=True)
    assert np.all(np.abs(after - ref) <= 1e-9 + 1e-12 * np.abs(ref))
    ctx.close()


@pytest.mark.parametrize("world", [2, 3])
def test_a_scan_split_with_shard_range_reassembles_to_the_single_call(rw, orc, world):
    """Strong scaling on one GPU: the shards that `bench.py --scaling strong` hands to the ranks (sharding.shard_range),
    each through its own context, concatenated in rank order, against the one-call scan and the oracle.  The shards
    start new rows of tiles, so the tiled contraction may split its k-ranges differently: equal to rounding, not to
    the bit."""
    import torch
    from paper_2607_00488_b200 import sharding
    inp = wl.make_custom(n_E=31, n_T=700, n_rec=390, n_periods=2, seed=171)
    params, kinds = wl.random_points(301, [0, 1, 4, 6], seed=172)
    ref, scale = orc.eval_batch(inp, params, kinds, want_abs=True, nthreads=8)
    whole_ctx = rw.Reweighter(inp, max_batch=301)
    whole = whole_ctx.eval_batch(_cuda(params), kinds).cpu().numpy()
    whole_ctx.close()
    parts, seen = [], 0
    for rank in range(world):
        lo, hi = sharding.shard_range(301, rank, world)
        assert lo == seen
        seen = hi
        ctx = rw.Reweighter(inp, max_batch=hi - lo)                   # a rank's own context, sized for its shard
        parts.append(ctx.eval_batch(_cuda(params[lo:hi]), kinds).cpu().numpy())
        ctx.close()
    torch.cuda.synchronize()
    assert seen == 301
    cat = np.concatenate(parts)
    assert np.all(np.abs(cat - whole) <= 1e-12 * np.abs(whole))
    assert np.all(np.abs(cat - ref) <= 1e-9 + 1e-12 * scale)


def test_host_buffers_can_return_mu(rw, orc):
    """rw_eval_batch with RW_PARAM_HOST | RW_OUT_HOST and out_mu: mu is staged through the workspace slice by slice (the
    context is sized for 128 points, the call has 300: slices of 128, 128 and 44) and copied D2H on the stream; bit-equal
    to the device-resident call, and within the bars of the oracle on sampled points around the slice edges."""
    import torch
    inp = wl.make_custom(n_E=31, n_T=203, n_rec=130, n_periods=2, seed=181)
    params, kinds = wl.random_points(300, [0, 1, 4, 6], seed=182)
    ctx = rw.Reweighter(inp, max_batch=128)
    out_d, mu_d = ctx.eval_batch(torch.from_numpy(params).cuda(), kinds, want_mu=True)
    out_h, mu_h = ctx.eval_batch(torch.from_numpy(params).pin_memory(), kinds, want_mu=True)
    torch.cuda.synchronize()
    assert not out_h.is_cuda and not mu_h.is_cuda
    assert np.array_equal(out_h.numpy(), out_d.cpu().numpy())
    assert np.array_equal(mu_h.numpy(), mu_d.cpu().numpy())
    idx = np.array([0, 127, 128, 255, 256, 299])
    ref, mu_ref, scale = orc.eval_batch(inp, params[idx], kinds, want_mu=True, want_abs=True, nthreads=4)
    assert np.all(np.abs(mu_h.numpy()[idx] - mu_ref) <= 1e-12 * np.abs(mu_ref))
    assert np.all(np.abs(out_h.numpy()[idx] - ref) <= 1e-9 + 1e-12 * scale)
    ctx.close()
