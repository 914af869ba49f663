"""Closure of the reweighting method against a continuum reference (Sec. VI A).

The paper's validation problem, rebuilt from its description: a monoenergetic 7Be line (E_nu = 0.862 MeV),
a light yield of 500 pe/MeV with a quenching non-linearity that suppresses the low-energy yield, and a Gaussian
photo-electron resolution with variance = mean.  The "direct" prediction folds the modified recoil spectrum
through P(N_p | T) on a fine grid; the "reweighting" prediction bins the SM spectrum in n_T recoil bins, applies ONE
weight per bin (evaluated at the bin's representative energy) and folds through the response matrix assembled from
the same P(N_p | T) (weighted by the SM spectrum inside each bin, as an SM Monte-Carlo histogram would be, Eq. 15).
What the paper prints and this file checks:
  * the integral deviation over 50 < N_p < 400 falls as n_T^-2 (Fig. 5)         -> fitted slope
  * the magnetic-moment deviation is several times the NSI one at fixed binning (~7x)
  * 25 bins close to better than 0.01 %; 2000 bins to < 1e-6 integral and < 1e-5 per bin
  * at theta = 0 the two predictions coincide by construction
The quenching law is not given in the paper (the chosen one is below), so its absolute 0.0013 % / 0.0097 % are
checked to order of magnitude only; the slope and the by-construction identity do not depend on that choice.
The oracle supplies the spectra, weights and fold; the GPU test runs the same inputs through the C ABI.
"""
import numpy as np
import pytest
from scipy.special import ndtr

E_LINE = 0.862
LIGHT_YIELD = 500.0      # pe / MeV
N_FINE = 48000           # continuum grid (divisible by every n_T used)
NP_EDGES = np.arange(0.0, 401.0)     # 1-pe bins; region of interest 50 < N_p < 400
ROI = slice(50, 400)
NSI = {0: 0.1, 1: 0.1}   # eps_ee^L = eps_ee^R = 0.1
MM = {6: 2.8e-11}        # mu_nu = 2.8e-11 mu_B


def _mean_pe(T):
    """<N_p>(T): 500 pe/MeV with a smooth quenching that suppresses the low-energy yield (chosen)."""
    return LIGHT_YIELD * T * (1.0 - 0.12 * np.exp(-T / 0.15))


def _theta(d):
    th = np.zeros(7)
    for k, v in d.items():
        th[k] = v
    return th


@pytest.fixture(scope="module")
def continuum(orc):
    """Fine-grid spectra and the conditional density P(N_p bin | T) on the fine grid."""
    t_max = orc.tmax(E_LINE)
    edges = np.linspace(0.0, t_max, N_FINE + 1)
    Tf = 0.5 * (edges[:-1] + edges[1:])
    dT = np.diff(edges)
    line = dict(E=np.array([E_LINE]), flux_w=np.array([1.0e24]), P_e=np.array([0.54]), f_tau=0.5, T=Tf)
    m = _mean_pe(Tf)
    cdf = ndtr((NP_EDGES[None, :] - m[:, None]) / np.sqrt(m)[:, None])
    Pk = np.diff(cdf, axis=1)                                     # [N_FINE][400]
    S = {name: orc.spectrum(line, _theta(d)) * dT for name, d in (("sm", {}), ("nsi", NSI), ("mm", MM))}
    direct = {name: S[name] @ Pk for name in S}
    return dict(t_max=t_max, line=line, S=S, Pk=Pk, direct=direct)


def _reweighting_inputs(orc, c, n_T):
    """N_mc[n_T], R[n_T][400], representative energies T[n_T] for a uniform recoil binning."""
    M = N_FINE // n_T
    S_sm = c["S"]["sm"]
    N_mc = S_sm.reshape(n_T, M).sum(1)
    R = (S_sm[:, None] * c["Pk"]).reshape(n_T, M, -1).sum(1) / N_mc[:, None]
    edges = np.linspace(0.0, c["t_max"], n_T + 1)
    T = 0.5 * (edges[:-1] + edges[1:])
    return N_mc, R, T


def _reweighted(orc, c, n_T, theta):
    N_mc, R, T = _reweighting_inputs(orc, c, n_T)
    inp = dict(c["line"], T=T)
    w = orc.weights(inp, theta)
    return orc.fold(w, N_mc, R, np.zeros(R.shape[1]))


def _integral_deviation(mu, ref):
    return abs(mu[ROI].sum() - ref[ROI].sum()) / ref[ROI].sum()


def test_sm_point_closes_exactly(orc, continuum):
    for n_T in (25, 400):
        mu = _reweighted(orc, continuum, n_T, np.zeros(7))
        assert np.all(np.abs(mu[ROI] / continuum["direct"]["sm"][ROI] - 1) < 1e-13)


def test_closure_scaling_and_magnitudes(orc, continuum):
    grid = [25, 50, 100, 200, 400, 800]
    dev = {}
    for name, d in (("nsi", NSI), ("mm", MM)):
        dev[name] = np.array([_integral_deviation(_reweighted(orc, continuum, n, _theta(d)), continuum["direct"][name])
                              for n in grid])
        slope = np.polyfit(np.log(grid), np.log(dev[name]), 1)[0]
        assert abs(slope + 2.0) < 0.1, (name, slope, dev[name])             # falls as n_T^-2
    ratio = dev["mm"] / dev["nsi"]
    assert np.all((ratio > 2.0) & (ratio < 25.0)), ratio                      # "about seven times"
    # 25 bins: "closes to better than 0.01 %" -- 0.0013 % (NSI), 0.0097 % (MM) with the paper's own quenching law
    assert 1e-6 < dev["nsi"][0] < 1e-4 and 1e-5 < dev["mm"][0] < 1e-3, (dev["nsi"][0], dev["mm"][0])


def test_closure_at_the_default_2000_bins(orc, continuum):
    """integral deviation below 1e-6 and bin-by-bin residual below 1e-5 at 2000 recoil bins."""
    for name, d in (("nsi", NSI), ("mm", MM)):
        mu = _reweighted(orc, continuum, 2000, _theta(d))
        ref = continuum["direct"][name]
        assert _integral_deviation(mu, ref) < 1e-6
        assert np.max(np.abs(mu[ROI] / ref[ROI] - 1)) < 1e-5


@pytest.mark.gpu
def test_closure_through_the_gpu_path(orc, continuum):
    """The same construction through the C ABI (collapsed, streaming and DMMA folds): the GPU prediction closes
    on the continuum reference exactly as the oracle's does."""
    import torch
    from paper_2607_00488_b200 import binding
    n_T = 2000
    N_mc, R, T = _reweighting_inputs(orc, continuum, n_T)
    inp = dict(continuum["line"], T=T, N_mc=N_mc[None], R=R[None], bkg=np.zeros((1, 400)), counts=np.ones((1, 400)))
    params = np.array([[0.1, 0.1, 0.0], [0.0, 0.0, 2.8e-11], [0.0, 0.0, 0.0]])
    kinds = [0, 1, 6]
    ctx = binding.Reweighter(inp, max_batch=64)
    p_dev = torch.from_numpy(params).cuda()
    for mode in ("stream", "gemm", "collapsed"):
        _, mu = ctx.eval_batch(p_dev, kinds, want_mu=True, mode=mode)
        torch.cuda.synchronize()
        mu = mu.cpu().numpy()[:, 0, :]
        for row, name in enumerate(("nsi", "mm", "sm")):
            ref = continuum["direct"][name]
            assert _integral_deviation(mu[row], ref) < 1e-6, (mode, name)
            assert np.max(np.abs(mu[row][ROI] / ref[ROI] - 1)) < 1e-5, (mode, name)
            orc_mu = _reweighted(orc, continuum, n_T, _theta({0: params[row, 0], 1: params[row, 1], 6: params[row, 2]}))
            assert np.max(np.abs(mu[row][ROI] / orc_mu[ROI] - 1)) < 1e-12, (mode, name)
    ctx.close()
