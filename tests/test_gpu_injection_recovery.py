"""End-to-end injection-recovery on the GPU path (Sec. VI B): Asimov data are built at an injected
parameter value, the parameter is scanned with the overall rate normalisation profiled at every scan point, and the
profile -2 Delta lnL must have its minimum (= 0) at the injected value -- eps_ee^L = 0.05 and mu_nu = 3e-11 mu_B are
the paper's two examples (tests/golden/paper_values.txt).  A gradient-based fit through rw_eval_grad started away
from the truth must converge to it as well.  The Asimov data come from the oracle, the scans from the C ABI."""
import os

import numpy as np
import pytest

from paper_2607_00488_b200 import workloads as wl

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 4


def _golden(name):
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")
    for line in open(path):
        f = line.split()
        if f and f[0] == name:
            return float(f[1])
    raise KeyError(name)


def _cuda(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("kind,name,lo,hi", [(wl.EPS_EE_L, "inject_eps_ee_L", -0.05, 0.15),
                                             (wl.MU_NU, "inject_mu_nu", 0.0, 8e-11)])
def test_profile_scan_recovers_the_injected_value(orc, kind, name, lo, hi):
    import torch
    from paper_2607_00488_b200 import binding
    inj = _golden(name)
    inp = wl.make("cfg2_mm_lowE" if kind == wl.MU_NU else "cfg1_tiny_nsi")
    _, mu = orc.eval_batch(inp, np.array([[inj]]), [kind], want_mu=True, nthreads=CORES)
    asimov = dict(inp, counts=mu[0])                                  # non-integer counts
    scan = np.unique(np.concatenate([np.linspace(lo, hi, 301), [inj]]))
    ctx = binding.Reweighter(asimov, max_batch=scan.size)
    prof, scale = ctx.eval_profile(_cuda(scan[:, None]), [kind])
    plain = ctx.eval_batch(_cuda(scan[:, None]), [kind])
    torch.cuda.synchronize()
    prof, scale, plain = prof.cpu().numpy(), scale.cpu().numpy(), plain.cpu().numpy()
    i_inj = int(np.argmin(np.abs(scan - inj)))
    assert int(np.argmin(prof)) == i_inj and abs(prof[i_inj]) < 1e-8 and abs(scale[i_inj] - 1.0) < 1e-9
    assert np.all(prof <= plain + 1e-8)                               # profiling can only lower the curve
    # the profile rises on both sides of the injected value (its width only reflects the Asimov statistics of the
    # synthetic data set); mu_nu >= 0 leaves the lower side open
    assert prof[-1] > 0.5 and (prof[0] > 0.5 or kind == wl.MU_NU)
    assert np.all(np.diff(prof[i_inj:]) > -1e-9) and np.all(np.diff(prof[:i_inj + 1]) < 1e-9)   # one minimum
    ctx.close()


def test_gradient_fit_converges_to_the_injected_point(orc):
    """Two couplings and the rate fitted together from a displaced start with scipy's BFGS fed by rw_eval_grad."""
    import torch
    from scipy.optimize import minimize
    from paper_2607_00488_b200 import binding
    inp = wl.make("cfg1_tiny_nsi")
    kinds = np.array([wl.EPS_EE_L, wl.EPS_EE_R, 7], np.int32)
    truth = np.array([_golden("inject_eps_ee_L"), -0.03, 1.1])
    _, mu = orc.eval_components(dict(inp, comp_of_T=np.zeros(inp["T"].size, np.int32)), truth[None, :], kinds, want_mu=True)
    ctx = binding.Reweighter(dict(inp, counts=mu[0]), max_batch=16)
    calls = [0]

    def fun(x):
        calls[0] += 1
        f, g = ctx.eval_grad(_cuda(np.asarray(x)[None, :]), kinds)
        torch.cuda.synchronize()
        return f.item(), g.cpu().numpy()[0]

    res = minimize(fun, truth + np.array([0.08, -0.06, -0.2]), jac=True, method="BFGS", options={"gtol": 1e-6})
    assert np.all(np.abs(res.x - truth) < 1e-6) and res.fun < 1e-8, (res.x, res.fun, calls[0])
    assert calls[0] < 200                                              # "a few hundred evaluations" per scan at most
    ctx.close()
