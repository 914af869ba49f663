"""rw_fold_weights_static: the entry point for callers that cannot allocate device memory.

Every other call of the library runs on a workspace the caller got from cudaMalloc.  A likelihood that lives as a plugin
inside an application whose own pool already owns the GPU, or a fit that must not trigger the device-wide
synchronisation cudaMalloc / cudaFree bring, has no such workspace to give.  rw_fold_weights_static needs none: its
scratch is a fixed 4 MiB array compiled into librw.so (hence the limit n_rec <= RW_STATIC_MAX_N_REC = 8192), shared by
all calls on a GPU and never cleared between them.

What is checked: its -2lnL and mu equal those of the existing path (rw_eval_weights, one point, streaming fold, which
works on a caller workspace) within the bars every parity test here uses (mu 1e-12 relative, -2lnL 1e-9 + 1e-12 x its
size), and the oracle's -- on two calls in a row with different weights, then on a smaller problem right after a
larger one, so that anything a call leaves behind in the shared array would show.  The file is named to be collected
last: `pytest -x` stops at the first failure and a failure here must not hide the other tests."""
import ctypes

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

MU_RTOL = 1e-12


def m2lnl_tol(scale):
    return 1e-9 + 1e-12 * np.abs(scale)


def _device_tables(inp):
    """The period-0 tables of a workload as CUDA tensors; R on an even row pitch (the entry point's requirement)."""
    import torch
    R = np.ascontiguousarray(inp["R"][0])
    n_T, n_rec = R.shape
    pitch = n_rec + (n_rec & 1)
    Rp = torch.zeros((n_T, pitch), dtype=torch.float64, device="cuda")
    Rp[:, :n_rec] = torch.from_numpy(R).cuda()
    cu = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()   # noqa: E731
    return cu(inp["N_mc"][0]), Rp[:, :n_rec], cu(inp["bkg"][0]), cu(inp["counts"][0])


def _compare(rw, orc, inp, w_rows):
    """Each row of w_rows: one static call, compared with the workspace path and with the oracle."""
    import torch
    N_mc, R, bkg, counts = _device_tables(inp)
    n_rec = R.shape[1]
    ctx = rw.Reweighter(inp, max_batch=1)
    out = torch.empty(1, dtype=torch.float64, device="cuda")          # caller-owned outputs: the call allocates nothing
    mu = torch.empty(n_rec, dtype=torch.float64, device="cuda")
    for w in w_rows:
        w_dev = torch.from_numpy(w).cuda()
        out.fill_(-1.0)
        mu.fill_(-1.0)
        rw.fold_weights_static(w_dev, N_mc, R, bkg, counts, out=out, out_mu=mu)
        ref, mu_ref = ctx.eval_weights(w_dev[None], want_mu=True, mode="stream")
        torch.cuda.synchronize()
        got, got_mu = out.cpu().numpy()[0], mu.cpu().numpy()
        ref, mu_ref = ref.cpu().numpy()[0], mu_ref.cpu().numpy()[0, 0]
        assert np.all(np.abs(got_mu - mu_ref) <= MU_RTOL * np.abs(mu_ref)), np.abs(got_mu / mu_ref - 1).max()
        assert abs(got - ref) <= m2lnl_tol(ref), (got, ref)
        o_ref, o_mu, o_scale = orc.eval_weights(inp, w[None], want_mu=True, want_abs=True, nthreads=4)
        assert np.all(np.abs(got_mu - o_mu[0, 0]) <= MU_RTOL * np.abs(o_mu[0, 0]))
        assert abs(got - o_ref[0]) <= m2lnl_tol(o_scale[0]), (got, o_ref[0])
    ctx.close()


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path_on_consecutive_calls(orc):
    import torch
    from paper_2607_00488_b200 import binding as rw
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rng = np.random.default_rng(77)
    # three column strips with a ragged tail (odd n_rec), 13 row ranges of 64 with a ragged last one
    big = wl.make_custom(n_E=24, n_T=777, n_rec=1031, n_periods=1, seed=71, dead_fraction=0.1)
    w1 = rng.uniform(0.0, 3.0, size=777)
    w2 = rng.uniform(0.5, 1.5, size=777)
    w2[:9] = 0.0
    _compare(rw, orc, big, [w1, w2, w1])
    # a smaller problem next: fewer strips and row ranges than the scratch still holds from the calls above
    small = wl.make_custom(n_E=20, n_T=203, n_rec=330, n_periods=1, seed=21)
    _compare(rw, orc, small, [rng.uniform(0.0, 3.0, size=203), np.ones(203)])
    # and the large one again
    _compare(rw, orc, big, [w2])


@pytest.mark.gpu
def test_static_scratch_degenerate_sizes():
    """No recoil bins: mu is the background.  Counts of zero and a dead column: values, not errors."""
    import torch
    from paper_2607_00488_b200 import binding as rw
    bkg = torch.tensor([2.0, 0.5, 0.0, 3.0], dtype=torch.float64, device="cuda")
    counts = torch.tensor([2.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")
    empty = torch.empty(0, dtype=torch.float64, device="cuda")
    out, mu = rw.fold_weights_static(empty, empty, torch.empty((0, 4), dtype=torch.float64, device="cuda"), bkg, counts,
                                     want_mu=True)
    torch.cuda.synchronize()
    assert np.array_equal(mu.cpu().numpy(), bkg.cpu().numpy())
    expect = 2.0 * ((0.5 - 1.0 + np.log(1.0 / 0.5)) + 3.0)
    assert abs(out.item() - expect) <= 1e-14
    counts[2] = 1.0                                              # mu = 0 < n: +inf, as rw_eval_batch documents
    out = rw.fold_weights_static(empty, empty, torch.empty((0, 4), dtype=torch.float64, device="cuda"), bkg, counts)
    torch.cuda.synchronize()
    assert np.isposinf(out.item())


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    """Runs without a GPU: the size check comes before any CUDA call and names the limit."""
    from paper_2607_00488_b200 import binding as rw
    L = rw.load_library()
    assert rw.RW_STATIC_MAX_N_REC == 8192
    rc = L.rw_fold_weights_static(None, None, None, 8194, 10, rw.RW_STATIC_MAX_N_REC + 1, None, None, None, None, None)
    assert rc == -1
    msg = L.rw_last_error(None).decode()
    assert "RW_STATIC_MAX_N_REC" in msg and "8193" in msg, msg
    assert L.rw_fold_weights_static(None, None, None, 0, -1, 4, None, None, None, None, None) == -1
    out = ctypes.c_double(0.0)
    # pointers are checked before anything is launched
    assert L.rw_fold_weights_static(None, None, None, 4, 10, 4, None, None, ctypes.byref(out), None, None) == -1
