"""Pins of the CPU oracle against things other than itself: closed forms, textbook numbers,
library routines, invariants and brute force (prompt section (3); SURVEY.md 8(c) "What pins
each part").  All CPU, all `-m "not gpu"`."""
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, stats

from paper_2607_00488_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _table(fn):
    rows = {}
    for line in open(os.path.join(GOLD, fn)):
        line = line.split("#")[0].strip()
        if line:
            f = line.split()
            rows[f[0]] = f[1:]
    return rows


TEXT = _table("textbook_values.txt")
PAPER = _table("paper_values.txt")
HBARC2 = float(TEXT["hbarc2_cm2_MeV2"][0])


def _txt(name):
    return float(TEXT[name][0]), float(TEXT[name][1])


def test_long_double_is_extended(orc):
    assert orc.long_double_mant_dig() >= 64


# ----------------------------------------------------------------------------- T_max
def test_tmax_closed_form_and_textbook_edges(orc):
    c = orc.default_consts()
    mp.mp.dps = 40
    for E in (0.05, 0.42, 0.862, 1.44, 3.0, 16.0):
        ref = 2 * mp.mpf(E) ** 2 / (mp.mpf(c.m_e) + 2 * mp.mpf(E))
        assert abs(orc.tmax(E) - float(ref)) <= 2 * np.spacing(float(ref))
    v, tol = _txt("be7_compton_edge_MeV")
    assert abs(orc.tmax(float(PAPER["be7_line_MeV"][0])) / v - 1) < tol
    v, tol = _txt("pp_endpoint_edge_MeV")
    assert abs(orc.tmax(0.42) / v - 1) < tol
    # E >> m_e: E - T_max -> m_e/2 (backward scattering leaves m_e/2 to the neutrino)
    assert abs((1e4 - orc.tmax(1e4)) - c.m_e / 2) < 1e-4


# ----------------------------------------------------------------------------- couplings
def test_sm_couplings_eq2_eq3(orc):
    c = orc.default_consts()
    gL, gR = orc.sm_couplings()
    rows = _table("sm_couplings.txt")
    for a, fl in enumerate(("e", "mu", "tau")):
        assert gL[a] == float(rows[fl][0]) + c.sin2_theta_w
        assert gR[a] == float(rows[fl][1]) + c.sin2_theta_w


# ----------------------------------------------------------------------------- Eq. (4)
def _weak_antiderivative(c, E, T, gL, gR):
    """F(T) with dF/dT = Eq.(4): C0 [gL^2 T - gR^2 (E/3)(1-T/E)^3 - gL gR m_e T^2/(2E^2)]."""
    C0 = 2 * c.G_F ** 2 * c.m_e / np.pi
    return C0 * (gL ** 2 * T - gR ** 2 * (E / 3.0) * (1 - T / E) ** 3 - gL * gR * c.m_e * T ** 2 / (2 * E * E))


@pytest.mark.parametrize("E,gL,gR", [(0.862, 0.73121, 0.23121), (0.3, -0.26879, 0.23121),
                                     (10.0, 0.9, -0.4), (2.0, -0.1, 0.7)])
def test_dsigma_weak_integrates_to_closed_form(orc, E, gL, gR):
    c = orc.default_consts()
    T1, T2 = 0.02 * E, orc.tmax(E)
    num, err = integrate.quad(lambda t: orc.dsigma_weak(E, t, gL, gR), T1, T2, epsabs=0, epsrel=1e-13)
    ref = _weak_antiderivative(c, E, T2, gL, gR) - _weak_antiderivative(c, E, T1, gL, gR)
    assert abs(num / ref - 1) < 1e-11


def test_dsigma_weak_textbook_cross_sections(orc):
    c = orc.default_consts()
    gL, gR = orc.sm_couplings()
    v, tol = _txt("sigma0_cm2")
    # T = 0, gR = 0, gL = 1: dsigma/dT = 2 G_F^2 m_e / pi  ->  times m_e = sigma_0
    assert abs(orc.dsigma_weak(1.0, 0.0, 1.0, 0.0) * c.m_e * HBARC2 / v - 1) < tol
    for a, name in ((0, "sigma_nue_e_10MeV_cm2"), (1, "sigma_numu_e_10MeV_cm2")):
        E = 10.0
        sig, _ = integrate.quad(lambda t: orc.dsigma_weak(E, t, gL[a], gR[a]), 0.0, orc.tmax(E),
                                epsabs=0, epsrel=1e-12)
        v, tol = _txt(name)
        assert abs(sig * HBARC2 / v - 1) < tol


def test_dsigma_weak_term_structure(orc):
    """Each bracket term of Eq.(4) in isolation: gL^2; gR^2 (1-T/E)^2; -gL gR m_e T/E^2."""
    c = orc.default_consts()
    C0 = 2 * c.G_F ** 2 * c.m_e / np.pi
    E, T = 1.7, 0.6
    assert abs(orc.dsigma_weak(E, T, 0.8, 0.0) / (C0 * 0.64) - 1) < 1e-15
    assert abs(orc.dsigma_weak(E, T, 0.0, 0.5) / (C0 * 0.25 * (1 - T / E) ** 2) - 1) < 1e-15
    cross = orc.dsigma_weak(E, T, 0.8, 0.5) - orc.dsigma_weak(E, T, 0.8, 0.0) - orc.dsigma_weak(E, T, 0.0, 0.5)
    assert abs(cross / (-C0 * 0.4 * c.m_e * T / E ** 2) - 1) < 1e-13
    assert cross < 0


# ----------------------------------------------------------------------------- Eq. (8)
def test_dsigma_mm_closed_forms(orc):
    c = orc.default_consts()
    v, tol = _txt("pi_re2_cm2")
    # E >> T: T dsigma/dT -> pi alpha^2/m_e^2 mu^2 = pi r_e^2 (mu_nu/mu_B)^2
    assert abs(orc.dsigma_mm(1e12, 1.0, 1.0) * HBARC2 / v - 1) < tol
    assert orc.dsigma_mm(0.7, 0.7, 1.0) == 0.0          # bracket 1/T - 1/E vanishes at T = E
    assert orc.dsigma_mm(0.862, 0.3, 2e-11) == orc.dsigma_mm(0.862, 0.3, -2e-11)   # even in mu_nu
    assert abs(orc.dsigma_mm(0.862, 0.3, 4e-11) / orc.dsigma_mm(0.862, 0.3, 2e-11) - 4) < 1e-15
    E, T1, T2, mu = 0.862, 0.01, orc.tmax(0.862), 2.8e-11
    num, _ = integrate.quad(lambda t: orc.dsigma_mm(E, t, mu), T1, T2, epsabs=0, epsrel=1e-13)
    Cmm = np.pi * c.alpha_em ** 2 / c.m_e ** 2
    ref = Cmm * mu ** 2 * (np.log(T2 / T1) - (T2 - T1) / E)
    assert abs(num / ref - 1) < 1e-11


# ----------------------------------------------------------------------------- Eq. (12)
def _tiny_inputs(seed=5, n_E=6, n_T=9):
    rng = np.random.default_rng(seed)
    E = np.sort(rng.uniform(0.3, 3.0, n_E))
    return dict(E=E, flux_w=rng.uniform(0.5, 2.0, n_E), P_e=rng.uniform(0.3, 0.6, n_E), f_tau=0.37,
                T=np.sort(rng.uniform(0.02, 2.5, n_T)))


def test_spectrum_single_line_reduces_to_dsigma(orc):
    gL, gR = orc.sm_couplings()
    E0, fw, Pe = 0.862, 3.7, 0.52
    T = np.array([0.05, 0.3, 0.66, 0.6649, 0.67, 0.9])
    inp = dict(E=np.array([E0]), flux_w=np.array([fw]), P_e=np.array([Pe]), f_tau=0.25, T=T)
    th = orc.theta_vector([0.1, -0.2, 0.05, 0.3, -0.15, 0.02, 2.8e-11], range(7))
    S = orc.spectrum(inp, th)
    Pmu, Ptau = (1 - Pe) * 0.75, (1 - Pe) * 0.25
    for i, t in enumerate(T):
        if t <= orc.tmax(E0):
            ref = fw * (Pe * orc.dsigma_weak(E0, t, gL[0] + 0.1, gR[0] - 0.2)
                        + Pmu * orc.dsigma_weak(E0, t, gL[1] + 0.05, gR[1] + 0.3)
                        + Ptau * orc.dsigma_weak(E0, t, gL[2] - 0.15, gR[2] + 0.02)
                        + orc.dsigma_mm(E0, t, 2.8e-11))
            assert abs(S[i] / ref - 1) < 1e-15
        else:
            assert S[i] == 0.0            # kinematic cut: nothing above the Compton edge
    assert S[4] == 0.0 and S[3] > 0.0     # 0.67 > T_max(0.862) = 0.66492 > 0.6649


def test_spectrum_mpmath_brute_force(orc):
    """Independent-precision brute force on a tiny grid (40 digits)."""
    mp.mp.dps = 40
    c = orc.default_consts()
    inp = _tiny_inputs()
    th = orc.theta_vector([0.21, -0.13, 0.4, 1.7e-11], [orc.EPS_EE_L, orc.EPS_TT_R, orc.EPS_MM_L, orc.MU_NU])
    S = orc.spectrum(inp, th)
    s2, me, GF, al = (mp.mpf(x) for x in (c.sin2_theta_w, c.m_e, c.G_F, c.alpha_em))
    g = {"e": (mp.mpf(1) / 2 + s2 + mp.mpf(0.21), s2), "m": (-mp.mpf(1) / 2 + s2 + mp.mpf(0.4), s2),
         "t": (-mp.mpf(1) / 2 + s2, s2 + mp.mpf(-0.13))}
    C0, Cmm = 2 * GF ** 2 * me / mp.pi, mp.pi * al ** 2 / me ** 2
    for i, Ti in enumerate(inp["T"]):
        acc = mp.mpf(0)
        for j, Ej in enumerate(inp["E"]):
            Ej_, Ti_ = mp.mpf(Ej), mp.mpf(Ti)
            if Ti_ > 2 * Ej_ ** 2 / (me + 2 * Ej_):
                continue
            Pe = mp.mpf(inp["P_e"][j])
            P = {"e": Pe, "m": (1 - Pe) * (1 - mp.mpf(0.37)), "t": (1 - Pe) * mp.mpf(0.37)}
            term = mp.mpf(0)
            for a in "emt":
                gL, gR = g[a]
                term += P[a] * C0 * (gL ** 2 + gR ** 2 * (1 - Ti_ / Ej_) ** 2 - gL * gR * me * Ti_ / Ej_ ** 2)
            term += Cmm * mp.mpf(1.7e-11) ** 2 * (1 / Ti_ - 1 / Ej_)
            acc += mp.mpf(inp["flux_w"][j]) * term
        if acc == 0:
            assert S[i] == 0.0
        else:
            assert abs(S[i] / float(acc) - 1) < 4e-16


def test_spectrum_continuum_limit_matches_integrated_cross_section(orc):
    """sum_i S(T_i) dT -> sum_j flux_w[j] * int_{T_lo}^{T_max(E_j)} dsigma/dT dT (closed forms).
    A missing kinematic cut, flux weight or flavour factor breaks this at O(1)."""
    c = orc.default_consts()
    gL, gR = orc.sm_couplings()
    rng = np.random.default_rng(11)
    E = np.array([0.5, 0.862, 1.3, 2.2, 4.0])
    fw = rng.uniform(0.5, 2.0, E.size)
    Pe = rng.uniform(0.3, 0.6, E.size)
    T_lo, T_hi, n_T = 0.05, 4.0, 40000
    edges = np.linspace(T_lo, T_hi, n_T + 1)
    T = 0.5 * (edges[1:] + edges[:-1])
    eps = [0.1, -0.05, 0.2, 0.1, -0.3, 0.15]
    mu = 5e-11
    S = orc.spectrum(dict(E=E, flux_w=fw, P_e=Pe, f_tau=0.5, T=T), orc.theta_vector(eps + [mu], range(7)))
    lhs = S.sum() * (T_hi - T_lo) / n_T
    Cmm = np.pi * c.alpha_em ** 2 / c.m_e ** 2
    rhs = 0.0
    for j in range(E.size):
        Tm = orc.tmax(E[j])
        P = (Pe[j], (1 - Pe[j]) * 0.5, (1 - Pe[j]) * 0.5)
        for a in range(3):
            l, r = gL[a] + eps[2 * a], gR[a] + eps[2 * a + 1]
            rhs += fw[j] * P[a] * (_weak_antiderivative(c, E[j], Tm, l, r) - _weak_antiderivative(c, E[j], T_lo, l, r))
        rhs += fw[j] * Cmm * mu ** 2 * (np.log(Tm / T_lo) - (Tm - T_lo) / E[j])
    assert abs(lhs / rhs - 1) < 2e-4      # midpoint rule + all-or-nothing edge bins: O(dT)


def test_spectrum_is_quadratic_in_eps_and_linear_in_mu2(orc):
    inp = _tiny_inputs(seed=8, n_E=12, n_T=15)
    for kind in range(6):
        S = [orc.spectrum(inp, orc.theta_vector([e, 0.07], [kind, (kind + 1) % 6])) for e in (-0.3, -0.1, 0.1, 0.3)]
        d3 = S[3] - 3 * S[2] + 3 * S[1] - S[0]
        assert np.all(np.abs(d3) <= 1e-14 * np.abs(S[3]))
        d2 = S[2] - 2 * S[1] + S[0]
        assert np.any(np.abs(d2) > 1e-3 * np.abs(S[1]))   # genuinely quadratic, not linear
    S0 = orc.spectrum(inp, orc.theta_vector([0.2], [orc.EPS_EE_R]))
    S1 = orc.spectrum(inp, orc.theta_vector([0.2, 3e-11], [orc.EPS_EE_R, orc.MU_NU]))
    S2 = orc.spectrum(inp, orc.theta_vector([0.2, 6e-11], [orc.EPS_EE_R, orc.MU_NU]))
    live = S0 > 0
    assert np.all(np.abs((S2 - S0)[live] / (S1 - S0)[live] - 4) < 1e-11)


def test_spectrum_chirality_sign_flip_symmetry(orc):
    """(gL,gR) -> (-gL,-gR) leaves Eq.(4) unchanged: eps -> -2g - eps is an exact partner point."""
    inp = _tiny_inputs(seed=9, n_E=10, n_T=11)
    gL, gR = orc.sm_couplings()
    a = orc.theta_vector([0.11, -0.23], [orc.EPS_EE_L, orc.EPS_EE_R])
    b = orc.theta_vector([-2 * gL[0] - 0.11, -2 * gR[0] + 0.23], [orc.EPS_EE_L, orc.EPS_EE_R])
    Sa, Sb = orc.spectrum(inp, a), orc.spectrum(inp, b)
    assert np.all(np.abs(Sa - Sb) <= 4e-16 * np.abs(Sa))


def test_spectrum_flavour_routing(orc):
    """P_e = 1: only eps_ee matters.  P_e = 0, f_tau = 0: only eps_mumu.  f_tau = 1: only eps_tautau."""
    base = _tiny_inputs(seed=10)
    for P_e, f_tau, live in ((1.0, 0.5, (0, 1)), (0.0, 0.0, (2, 3)), (0.0, 1.0, (4, 5))):
        inp = dict(base, P_e=np.full_like(base["E"], P_e), f_tau=f_tau)
        S0 = orc.spectrum(inp, np.zeros(7))
        for kind in range(6):
            S = orc.spectrum(inp, orc.theta_vector([0.2], [kind]))
            if kind in live:
                assert np.any(S != S0)
            else:
                assert np.array_equal(S, S0)


# ----------------------------------------------------------------------------- weights
def test_weights_are_one_at_sm_point_and_in_dead_bins(orc):
    inp = _tiny_inputs(seed=12, n_E=8, n_T=30)
    inp["T"] = np.linspace(0.05, 6.0, 30)          # bins above every T_max are dead
    w = orc.weights(inp, np.zeros(7))
    assert np.all(w == 1.0)
    S0 = orc.spectrum(inp, np.zeros(7))
    assert np.any(S0 == 0.0) and np.any(S0 > 0.0)
    th = orc.theta_vector([0.3, 4e-11], [orc.EPS_EE_L, orc.MU_NU])
    w = orc.weights(inp, th)
    assert np.all(w[S0 == 0.0] == 1.0)
    live = S0 > 0
    assert np.all(np.abs(w[live] / (orc.spectrum(inp, th)[live] / S0[live]) - 1) < 4e-16)


# ----------------------------------------------------------------------------- fold
def test_fold_special_responses_and_library_matmul(orc):
    rng = np.random.default_rng(3)
    n_T, n_rec = 37, 23
    w, N, bkg = rng.uniform(0.5, 1.5, n_T), rng.uniform(1, 100, n_T), rng.uniform(0, 5, n_rec)
    R = rng.uniform(0, 1, (n_T, n_rec))
    mu = orc.fold(w, N, R, bkg)
    ref = (w * N) @ R + bkg                       # library routine on a non-square operand
    assert np.all(np.abs(mu / ref - 1) < 1e-15)
    # identity response: mu = N' + B
    mu_id = orc.fold(w, N, np.eye(n_T), np.arange(n_T, dtype=float))
    assert np.all(np.abs(mu_id - (w * N + np.arange(n_T))) <= 1e-13)
    # rank-1 response eff_i * q_k
    eff, q = rng.uniform(0.8, 1, n_T), rng.dirichlet(np.ones(n_rec))
    mu_r1 = orc.fold(w, N, np.outer(eff, q), np.zeros(n_rec))
    assert np.all(np.abs(mu_r1 / (q * np.sum(w * N * eff)) - 1) < 1e-15)
    # folded total = sum_i w_i N_i * (row efficiency)   (north_star invariant)
    assert abs((mu - bkg).sum() / np.sum(w * N * R.sum(axis=1)) - 1) < 1e-15


# ----------------------------------------------------------------------------- likelihood
def test_deviance_and_eq18_against_scipy_poisson(orc):
    rng = np.random.default_rng(4)
    mu = rng.uniform(0.5, 300.0, 64)
    n = rng.poisson(mu).astype(float)
    n[:3] = 0.0
    full = -2.0 * stats.poisson.logpmf(n, mu).sum()
    sat = -2.0 * stats.poisson.logpmf(n, np.where(n > 0, n, 1e-300)).sum()
    assert abs(orc.eq18(mu, n) / full - 1) < 1e-13
    assert abs(orc.deviance(mu, n) - (full - sat)) < 1e-10 * abs(full)
    assert orc.deviance(n[3:], n[3:]) == 0.0                       # counts == mu  =>  0
    assert orc.deviance(np.array([2.5, 0.0]), np.array([0.0, 0.0])) == 5.0   # n = 0 => 2 mu
    assert orc.deviance(np.array([0.0]), np.array([1.0])) == np.inf
    # small-d expansion 2[d - n log1p(d/n)] = d^2/n - (2/3) d^3/n^2 + ...
    nn, d = 1000.0, 1e-3
    assert abs(orc.deviance(np.array([nn + d]), np.array([nn])) / (d * d / nn - (2.0 / 3) * d ** 3 / nn ** 2) - 1) < 1e-9
    # non-integer (Asimov) counts are accepted: PAPER.md:309
    assert orc.deviance(np.array([10.25]), np.array([10.25])) == 0.0


# ----------------------------------------------------------------------------- whole path
def _small_problem(D=2):
    return wl.make_custom(n_E=19, n_T=41, n_rec=29, n_periods=D, seed=77)


def test_eval_batch_is_the_composition_of_its_steps(orc):
    inp = _small_problem()
    params, kinds = wl.random_points(5, [orc.EPS_TT_L, orc.MU_NU, orc.EPS_EE_R], seed=2)
    out, mu, ab = orc.eval_batch(inp, params, kinds, want_mu=True, want_abs=True)
    for p in range(5):
        th = orc.theta_vector(params[p], kinds)
        w = orc.weights(inp, th)
        tot = 0.0
        for d in range(2):
            m = orc.fold(w, inp["N_mc"][d], inp["R"][d], inp["bkg"][d])
            assert np.all(np.abs(mu[p, d] / m - 1) < 1e-15)
            tot += orc.deviance(m, inp["counts"][d])
        assert abs(out[p] / tot - 1) < 1e-13
        assert ab[p] >= out[p] > 0
    # kind order is irrelevant; absent kinds are zero; threads do not change results
    perm = [2, 0, 1]
    out2 = orc.eval_batch(inp, params[:, perm], kinds[perm], nthreads=2)
    assert np.array_equal(out, out2)
    full = orc.eval_batch(inp, params, kinds, full_eq18=True)
    sat_const = full - out
    assert np.all(np.abs(sat_const - sat_const[0]) < 1e-9 * abs(sat_const[0]))   # theta independent
    with pytest.raises(ValueError):
        orc.eval_batch(inp, params, [0, 0, 1])


def test_rank_K_prefold_identity(orc):
    """SURVEY finding 0.2: mu - B is linear in the spectrum, so folding basis spectra first gives
    the same prediction.  Checked with spectra at 3 points of a 1-D quadratic (exact Lagrange)."""
    inp = _small_problem(D=1)
    e = np.array([-0.4, 0.0, 0.4])
    x = 0.17
    lag = np.array([(x - e[1]) * (x - e[2]) / ((e[0] - e[1]) * (e[0] - e[2])),
                    (x - e[0]) * (x - e[2]) / ((e[1] - e[0]) * (e[1] - e[2])),
                    (x - e[0]) * (x - e[1]) / ((e[2] - e[0]) * (e[2] - e[1]))])
    _, mu_nodes = orc.eval_batch(inp, e[:, None], [orc.EPS_EE_L], want_mu=True)
    _, mu_x = orc.eval_batch(inp, np.array([[x]]), [orc.EPS_EE_L], want_mu=True)
    B = inp["bkg"][0]
    pred = np.tensordot(lag, mu_nodes[:, 0, :] - B, axes=1) + B
    assert np.all(np.abs(pred / mu_x[0, 0] - 1) < 1e-13)


def test_eval_weights_pins(orc):
    """Caller-supplied weights (Eq. 1 with an arbitrary diag(r)): (i) fed the spectrum-ratio weights
    it reproduces eval_batch; (ii) on random weights mu = (w*N_mc) @ R + bkg by numpy and the
    likelihood is -2 sum logpmf by scipy; (iii) w == 1 is the SM prediction; (iv) a transposed or
    period-swapped operand fails (ii)."""
    from scipy.stats import poisson
    inp = _small_problem(D=2)
    params, kinds = wl.random_points(4, [orc.EPS_EE_L, orc.MU_NU], seed=9)
    ref, mu_ref = orc.eval_batch(inp, params, kinds, want_mu=True)
    w = np.stack([orc.weights(inp, orc.theta_vector(params[p], kinds)) for p in range(4)])
    out, mu = orc.eval_weights(inp, w, want_mu=True, nthreads=2)
    assert np.all(np.abs(mu / mu_ref - 1) < 1e-15) and np.all(np.abs(out / ref - 1) < 1e-13)
    rng = np.random.default_rng(10)
    w = rng.uniform(0.2, 3.0, size=(3, inp["T"].size))
    out, mu, ab = orc.eval_weights(inp, w, want_mu=True, want_abs=True)
    full = orc.eval_weights(inp, w, full_eq18=True)
    for p in range(3):
        tot = 0.0
        for d in range(2):
            m = (w[p] * inp["N_mc"][d]) @ inp["R"][d] + inp["bkg"][d]
            assert np.all(np.abs(mu[p, d] / m - 1) < 1e-14)
            tot += -2.0 * poisson.logpmf(inp["counts"][d], m).sum()
        assert abs(full[p] / tot - 1) < 1e-12
        assert ab[p] >= out[p] > 0
    _, mu1 = orc.eval_weights(inp, np.ones((1, inp["T"].size)), want_mu=True)
    for d in range(2):
        assert np.all(np.abs(mu1[0, d] / (inp["N_mc"][d] @ inp["R"][d] + inp["bkg"][d]) - 1) < 1e-15)


def test_profile_scale_pins(orc):
    """Profiled rate normalisation (rate_k of Eq. 17, pull of Eq. 18):
    (i) no background, no pull: Poisson MLE of a scale, s^ = sum n / sum S (closed form);
    (ii) Asimov data n = s* S + B: s^ = s*, value 0;  (iii) scipy minimize_scalar on a numpy objective,
    with and without pull;  (iv) sigma -> 0 pins s^ to s0, huge sigma = no pull;  (v) boundary s^ = 0;
    (vi) the Eq. 18 form has the same minimiser and differs by the saturated constant."""
    from scipy.optimize import minimize_scalar
    from scipy.special import gammaln, xlogy
    rng = np.random.default_rng(3)
    S = rng.uniform(1.0, 300.0, 57)
    B = rng.uniform(0.5, 20.0, 57)
    n = rng.poisson(1.3 * S + B).astype(float)
    s, f = orc.profile_scale(S, np.zeros(57), n)
    assert abs(s / (n.sum() / S.sum()) - 1) < 1e-15
    s, f = orc.profile_scale(S, B, 0.83 * S + B)
    assert abs(s - 0.83) < 1e-15 and abs(f) < 1e-12

    def obj(x, s0=1.0, sig=0.0):
        mu = x * S + B
        v = 2.0 * np.sum(mu - n + xlogy(n, n) - xlogy(n, mu))
        return v + ((x - s0) / sig) ** 2 if sig > 0 else v
    for s0, sig in ((1.0, 0.0), (1.0, 0.05), (0.7, 0.01)):
        s, f = orc.profile_scale(S, B, n, s0=s0, sigma=sig)
        r = minimize_scalar(lambda x: obj(x, s0, sig), bounds=(0.0, 5.0), method="bounded", options={"xatol": 1e-12})
        assert abs(s - r.x) < 1e-6 and abs(f - r.fun) < 1e-8 * max(1.0, abs(r.fun))
        assert abs(f - obj(s, s0, sig)) < 1e-9 * max(1.0, abs(f))
        assert f <= obj(1.0, s0, sig) + 1e-9                      # profiling never raises the value
    s_tight, _ = orc.profile_scale(S, B, n, s0=0.9, sigma=1e-9)
    assert abs(s_tight - 0.9) < 1e-9
    s_free, f_free = orc.profile_scale(S, B, n)
    s_loose, f_loose = orc.profile_scale(S, B, n, s0=0.9, sigma=1e9)
    assert abs(s_loose - s_free) < 1e-9 and abs(f_loose - f_free) < 1e-9
    # boundary: data below the background everywhere => no signal wanted
    s0_, f0_ = orc.profile_scale(S, B, 0.5 * B)
    assert s0_ == 0.0 and abs(f0_ - orc.deviance(B, 0.5 * B)) < 1e-12
    sf, ff = orc.profile_scale(S, B, n, full_eq18=True)
    const = 2.0 * np.sum(gammaln(n + 1) - xlogy(n, n) + n)
    assert abs(sf - s_free) < 1e-15 and abs(ff - f_free - const) < 1e-9 * abs(ff)


def test_eval_profile_composition_and_asimov(orc):
    """eval_profile = (fold without background) -> profile_scale over the bins of all periods; Asimov data made
    at (theta*, s*) are recovered with value 0 at theta* (PAPER.md:309-311); value <= the unprofiled one."""
    inp = _small_problem(D=2)
    params, kinds = wl.random_points(4, [orc.EPS_EE_L, orc.MU_NU], seed=31)
    out, sc, ab = orc.eval_profile(inp, params, kinds, want_abs=True, nthreads=2)
    plain, mu = orc.eval_batch(inp, params, kinds, want_mu=True)
    for p in range(4):
        S = (mu[p] - inp["bkg"]).ravel()
        s, f = orc.profile_scale(S, inp["bkg"].ravel(), inp["counts"].ravel())
        assert abs(s / sc[p] - 1) < 1e-12 and abs(f - out[p]) < 1e-9 * max(1.0, f)
        assert out[p] <= plain[p] + 1e-9 and ab[p] >= out[p]
    asim = dict(inp)
    asim["counts"] = 1.7 * (mu[2] - inp["bkg"]) + inp["bkg"]
    out, sc = orc.eval_profile(asim, params, kinds)
    assert abs(sc[2] - 1.7) < 1e-12 and abs(out[2]) < 1e-9 and np.all(out[[0, 1, 3]] > 1e-3)
    pulled, scp = orc.eval_profile(asim, params, kinds, s0=1.0, sigma=0.1)
    assert pulled[2] > out[2] and 1.0 < scp[2] < 1.7


def test_eval_components_pins(orc):
    """Multi-component path (Eq. 17): (i) one component = eval_batch; (ii) two components with the same
    tables = eval_batch on the concatenated bins; (iii) mu - bkg is linear in the rates, with the single-component
    predictions as coefficients; (iv) a component's bins are weighted with its own flux table."""
    one = _small_problem(D=2)
    params, kinds = wl.random_points(4, [orc.EPS_EE_L, orc.EPS_TT_R, orc.MU_NU], seed=41)
    ref, mu_ref = orc.eval_batch(one, params, kinds, want_mu=True)
    as1 = dict(one, comp_of_T=np.zeros(one["T"].size, np.int32))
    out, mu = orc.eval_components(as1, params, kinds, want_mu=True)
    assert np.array_equal(out, ref) and np.array_equal(mu, mu_ref)
    split = dict(one, flux_w=np.stack([one["flux_w"]] * 2), P_e=np.stack([one["P_e"]] * 2),
                 comp_of_T=(np.arange(one["T"].size) % 2).astype(np.int32))
    out, mu = orc.eval_components(split, params, kinds, want_mu=True, nthreads=2)
    assert np.array_equal(out, ref) and np.array_equal(mu, mu_ref)

    mc = wl.make_components(n_comp=3, n_E=30, n_T=60, n_rec=31, n_periods=2, seed=42)
    kinds3 = np.array([orc.EPS_EE_L, orc.MU_NU, orc.RATE_0, orc.RATE_0 + 2], np.int32)
    p3, _ = wl.random_points(3, kinds3, seed=43)
    out, mu = orc.eval_components(mc, p3, kinds3, want_mu=True)
    for p in range(3):
        pred = np.zeros_like(mu[p])
        rates = [p3[p, 2], 1.0, p3[p, 3]]
        for c in range(3):
            only = dict(mc, N_mc=np.where(mc["comp_of_T"] == c, mc["N_mc"], 0.0))
            _, mu_c = orc.eval_components(only, p3[p:p + 1, :2], kinds3[:2], want_mu=True)
            pred += rates[c] * (mu_c[0] - mc["bkg"])
            # (iv) component c alone = a single-component problem with its own table on its own bins
            sel = mc["comp_of_T"] == c
            single = dict(E=mc["E"], flux_w=mc["flux_w"][c], P_e=mc["P_e"][c], f_tau=0.5, T=mc["T"][sel],
                          N_mc=mc["N_mc"][:, sel], R=mc["R"][:, sel, :], bkg=mc["bkg"], counts=mc["counts"])
            _, mu_s = orc.eval_batch(single, p3[p:p + 1, :2], kinds3[:2], want_mu=True)
            assert np.all(np.abs(mu_s[0] / mu_c[0] - 1) < 1e-15)
        assert np.all(np.abs((pred + mc["bkg"]) / mu[p] - 1) < 1e-14)
    with pytest.raises(ValueError):
        orc.eval_components(mc, p3, [0, 6, 7, 10])          # rate kind of a component that does not exist


def test_eval_grad_pins(orc):
    """Analytic gradient against Richardson-extrapolated central differences of eval_components in every kind
    (all six couplings, mu_nu, two rates); the value output is eval_components'; at an Asimov point the
    gradient vanishes (the injected point is the minimum)."""
    mc = wl.make_components(n_comp=2, n_E=26, n_T=50, n_rec=37, n_periods=2, seed=81)
    kinds = np.array([0, 1, 2, 3, 4, 5, 6, 7, 8], np.int32)
    params, _ = wl.random_points(3, kinds, seed=82)
    params[:, 6] = [2e-11, 5e-11, 8e-11]
    out, grad = orc.eval_grad(mc, params, kinds, nthreads=2)
    ref = orc.eval_components(mc, params, kinds)
    assert np.array_equal(out, ref)
    for a in range(kinds.size):
        h = 1e-12 if kinds[a] == 6 else 1e-3

        def diff(step):
            up, dn = params.copy(), params.copy()
            up[:, a] += step
            dn[:, a] -= step
            return (orc.eval_components(mc, up, kinds) - orc.eval_components(mc, dn, kinds)) / (2 * step)
        fd = (4.0 * diff(h / 2) - diff(h)) / 3.0
        assert np.all(np.abs(fd - grad[:, a]) <= 1e-7 * np.abs(grad[:, a]) + 1e-9 * np.abs(ref) / h * 1e-3), (a, fd, grad[:, a])
    _, mu = orc.eval_components(mc, params[:1], kinds, want_mu=True)
    asim = dict(mc, counts=mu[0])
    out0, g0 = orc.eval_grad(asim, params[:1], kinds)
    scale = np.abs(orc.eval_grad(mc, params[:1], kinds)[1])
    assert abs(out0[0]) < 1e-9 and np.all(np.abs(g0) <= 1e-10 * scale)


def test_eval_pee_pins(orc):
    """Per-point survival probabilities: (i) the nominal table for every point = eval_batch; (ii) = eval_weights fed
    spectrum(point's table, theta) / spectrum(nominal table, 0), both from orc.spectrum; (iii) on a single line,
    P_ee = 1 and P_ee = 0 give the pure nu_e and nu_mu,tau cross sections of Eq. (4) over the nominal mixture."""
    inp = _small_problem(D=2)
    params, kinds = wl.random_points(4, [orc.EPS_EE_L, orc.EPS_TT_R, orc.MU_NU], seed=51)
    n_E = inp["E"].size
    ref, mu_ref = orc.eval_batch(inp, params, kinds, want_mu=True)
    out, mu = orc.eval_pee(inp, params, kinds, np.tile(inp["P_e"], (4, 1)), want_mu=True)
    assert np.array_equal(out, ref) and np.array_equal(mu, mu_ref)
    rng = np.random.default_rng(52)
    Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.2, 0.2, size=(4, n_E)), 0.0, 1.0)
    out, mu = orc.eval_pee(inp, params, kinds, Pp, want_mu=True, nthreads=2)
    S0 = orc.spectrum(inp, np.zeros(7))
    live = S0 > 0                                                    # dead bins keep w = 1 (reading R9)
    w = np.stack([np.where(live, orc.spectrum(dict(inp, P_e=Pp[p]), orc.theta_vector(params[p], kinds)) /
                           np.where(live, S0, 1.0), 1.0) for p in range(4)])
    out_w, mu_w = orc.eval_weights(inp, w, want_mu=True)
    assert np.all(np.abs(mu / mu_w - 1) < 1e-14) and np.all(np.abs(out / out_w - 1) < 1e-12)
    assert not np.allclose(out, ref, rtol=1e-6)                      # the tables do matter
    # (iii) a single line, one recoil bin below the Compton edge
    E0, T0, pe0 = 0.862, 0.3, 0.54
    gL, gR = orc.sm_couplings()
    line = dict(E=np.array([E0]), flux_w=np.array([2.0]), P_e=np.array([pe0]), f_tau=0.5, T=np.array([T0]),
                N_mc=np.array([[100.0]]), R=np.array([[[0.9]]]), bkg=np.array([[1.0]]), counts=np.array([[50.0]]))
    se, sm = orc.dsigma_weak(E0, T0, gL[0], gR[0]), orc.dsigma_weak(E0, T0, gL[1], gR[1])
    nominal = pe0 * se + (1 - pe0) * sm
    _, mu1 = orc.eval_pee(line, np.zeros((2, 1)), [0], np.array([[1.0], [0.0]]), want_mu=True)
    assert abs(mu1[0, 0, 0] - (1.0 + 0.9 * 100.0 * se / nominal)) < 1e-12 * mu1[0, 0, 0]
    assert abs(mu1[1, 0, 0] - (1.0 + 0.9 * 100.0 * sm / nominal)) < 1e-12 * mu1[1, 0, 0]


def test_eval_pee_components_pins(orc):
    """Per-point survival probabilities with components / explicit nominal nu_mu, nu_tau tables (reading R17):
    (i) one component, no explicit tables = orc_eval_pee; (ii) the nominal P_e for every point = orc_eval_components,
    with explicit tables too (the rho split then returns exactly P_mu, P_tau); (iii) = eval_weights fed spectrum
    ratios built with orc.spectrum from hand-split tables P_mu^p = (1 - P_e^p) P_mu / (P_mu + P_tau);
    (iv) changing the table of component 1 leaves the bins of component 0 untouched; (v) a single line with
    explicit tables in ratio 3 : 1: P_e^p = 0 gives the 3/4 nu_mu + 1/4 nu_tau cross-section mixture."""
    inp = _small_problem(D=2)
    params, kinds = wl.random_points(3, [orc.EPS_EE_L, orc.EPS_MM_R, orc.EPS_TT_L, orc.MU_NU], seed=61)
    n_E = inp["E"].size
    rng = np.random.default_rng(62)
    Pp = np.clip(inp["P_e"][None, :] + rng.uniform(-0.2, 0.2, size=(3, n_E)), 0.0, 1.0)
    a, mu_a = orc.eval_pee(inp, params, kinds, Pp, want_mu=True)
    b, mu_b = orc.eval_pee_components(inp, params, kinds, Pp, want_mu=True)
    assert np.array_equal(a, b) and np.array_equal(mu_a, mu_b)                                   # (i)
    mc = wl.make_components(n_comp=2, n_E=21, n_T=30, n_rec=17, n_periods=1, seed=63)
    frac = rng.uniform(0.2, 0.8, size=mc["P_e"].shape)
    mc["P_mu"] = (1.0 - mc["P_e"]) * frac
    mc["P_tau"] = (1.0 - mc["P_e"]) * (1.0 - frac)
    ref, mu_ref = orc.eval_components(mc, params, kinds, want_mu=True)
    nom = np.tile(mc["P_e"][None], (3, 1, 1))
    out, mu = orc.eval_pee_components(mc, params, kinds, nom, want_mu=True)
    assert np.all(np.abs(mu / mu_ref - 1) < 1e-14) and np.all(np.abs(out - ref) <= 1e-11 * np.abs(ref))   # (ii)
    pts = np.clip(nom + rng.uniform(-0.2, 0.2, size=nom.shape), 0.0, 1.0)
    out, mu = orc.eval_pee_components(mc, params, kinds, pts, want_mu=True, nthreads=2)
    comp = mc["comp_of_T"]
    w = np.ones((3, mc["T"].size))
    for q in range(2):
        one = dict(mc, flux_w=mc["flux_w"][q], P_e=mc["P_e"][q], P_mu=mc["P_mu"][q], P_tau=mc["P_tau"][q])
        S0 = orc.spectrum(one, np.zeros(7))
        for p in range(3):
            share = mc["P_mu"][q] / (mc["P_mu"][q] + mc["P_tau"][q])
            tab = dict(one, P_e=pts[p, q], P_mu=(1 - pts[p, q]) * share, P_tau=(1 - pts[p, q]) * (1 - share))
            S = orc.spectrum(tab, orc.theta_vector(params[p], kinds))
            sel = (comp == q) & (S0 > 0)
            w[p, sel] = S[sel] / S0[sel]
    out_w, mu_w = orc.eval_weights(mc, w, want_mu=True)
    assert np.all(np.abs(mu / mu_w - 1) < 1e-14) and np.all(np.abs(out / out_w - 1) < 1e-12)              # (iii)
    pts2 = pts.copy()
    pts2[:, 1] = np.clip(pts[:, 1] + 0.1, 0.0, 1.0)
    # a response that keeps the components apart in the observable: identity-like rows
    iso = dict(mc, R=np.eye(mc["T"].size)[None], bkg=np.ones((1, mc["T"].size)), counts=np.ones((1, mc["T"].size)))
    _, m1 = orc.eval_pee_components(iso, params, kinds, pts, want_mu=True)
    _, m2 = orc.eval_pee_components(iso, params, kinds, pts2, want_mu=True)
    assert np.array_equal(m1[:, 0, comp == 0], m2[:, 0, comp == 0]) and not np.allclose(m1[:, 0, comp == 1], m2[:, 0, comp == 1])  # (iv)
    E0, T0, pe0 = 0.862, 0.3, 0.54
    gL, gR = orc.sm_couplings()
    line = dict(E=np.array([E0]), flux_w=np.array([2.0]), P_e=np.array([pe0]), P_mu=np.array([0.75 * (1 - pe0)]),
                P_tau=np.array([0.25 * (1 - pe0)]), T=np.array([T0]), N_mc=np.array([[100.0]]), R=np.array([[[0.9]]]),
                bkg=np.array([[1.0]]), counts=np.array([[50.0]]))
    eps_tt = 0.2                                                     # makes nu_tau differ from nu_mu
    se = orc.dsigma_weak(E0, T0, gL[0], gR[0])
    sm = orc.dsigma_weak(E0, T0, gL[1], gR[1])
    st = orc.dsigma_weak(E0, T0, gL[2] + eps_tt, gR[2])
    nominal = pe0 * se + (1 - pe0) * (0.75 * sm + 0.25 * orc.dsigma_weak(E0, T0, gL[2], gR[2]))
    _, mu1 = orc.eval_pee_components(line, np.full((1, 1), eps_tt), [orc.EPS_TT_L], np.array([[0.0]]), want_mu=True)
    assert abs(mu1[0, 0, 0] - (1.0 + 0.9 * 100.0 * (0.75 * sm + 0.25 * st) / nominal)) < 1e-12 * mu1[0, 0, 0]       # (v)


def test_sm_point_gives_sm_prediction(orc):
    inp = _small_problem(D=2)
    _, mu = orc.eval_batch(inp, np.zeros((1, 1)), [orc.EPS_EE_L], want_mu=True)
    for d in range(2):
        ref = inp["N_mc"][d] @ inp["R"][d] + inp["bkg"][d]
        assert np.all(np.abs(mu[0, d] / ref - 1) < 1e-15)


@pytest.mark.parametrize("kind,name", [(0, "inject_eps_ee_L"), (6, "inject_mu_nu")])
def test_asimov_injection_recovery(orc, kind, name):
    """Asimov data at the injected value => the scan minimum sits there (and is 0)."""
    inj = float(PAPER[name][0])
    inp = wl.make("cfg1_tiny_nsi") if kind == 0 else _small_problem(D=1)
    _, mu = orc.eval_batch(inp, np.array([[inj]]), [kind], want_mu=True)
    asimov = dict(inp, counts=mu[0])
    scan = inj * np.linspace(0.0, 2.0, 41)
    out = orc.eval_batch(asimov, scan[:, None], [kind])
    assert np.argmin(out) == 20 and abs(out[20]) < 1e-12
    assert np.all(np.delete(out, 20) > 1e-9)


# ----------------------------------------------------------------------------- workloads
def test_config1_recipe_and_stored_derived_inputs(orc):
    """BASELINE config 1: the 0.862 MeV line holds 30 % of SM events; the stored S_hat / counts are
    what the oracle produces today (they are written by oracle/write_derived_inputs.py only)."""
    inp = wl.make("cfg1_tiny_nsi")
    zero = np.zeros(7)
    S = orc.spectrum(inp, zero)
    line = dict(inp, E=inp["E"][-1:], flux_w=inp["flux_w"][-1:], P_e=inp["P_e"][-1:])
    assert abs(orc.spectrum(line, zero).sum() / S.sum() - 0.30) < 1e-12
    assert np.all(np.abs(inp["N_mc"][0] - 1e4 * S / S.sum()) <= 1e-12 * inp["N_mc"][0].max())
    assert abs(inp["N_mc"].sum() - 1e4) < 1e-8
    mu_sm = orc.fold(np.ones(100), inp["N_mc"][0], inp["R"][0], inp["bkg"][0])
    assert np.array_equal(np.random.default_rng(0).poisson(mu_sm), inp["counts"][0])
    # Gaussian response with efficiency 0.9 (interior rows), flat background 5
    assert abs(inp["R"][0][50].sum() - 0.9) < 1e-12 and np.all(inp["bkg"] == 5.0)
    p, kinds = wl.scan_points("cfg1_tiny_nsi")
    assert p.shape == (121, 2) and list(kinds) == [0, 1] and p.min() == -0.5 and p.max() == 0.5


def test_config2_stored_derived_inputs(orc):
    inp = wl.make("cfg2_mm_lowE")
    S = orc.spectrum(inp, np.zeros(7))
    assert np.sum(S == 0.0) > 800          # bins above the 665 keV edge are dead (reading R9)
    assert np.all(np.abs(inp["N_mc"][0] - 1e5 * S / S.sum()) <= 1e-12 * inp["N_mc"][0].max())
    p, kinds = wl.scan_points("cfg2_mm_lowE")
    assert p.shape == (1000, 1) and list(kinds) == [6]
    assert abs(p[0, 0] / 1e-12 - 1) < 1e-12 and abs(p[-1, 0] / 1e-10 - 1) < 1e-12


def test_tolerance_scale_equals_the_deviance_two_sided(orc):
    """`abs_out` = sum_k 2|term_k| sets every -2lnL tolerance of the GPU tests (1e-9 + 1e-12 x scale, reading T), so an
    inflated scale would loosen every parity bar unnoticed.  Every deviance term of Eq. (18) is >= 0,
    hence in deviance mode the scale must EQUAL the value to rounding -- in every oracle entry point that returns one;
    for the profiled value it equals the value minus the Gaussian pull at the minimiser."""
    tol = 4e-16
    inp = _small_problem(D=2)
    params, kinds = wl.random_points(6, [orc.EPS_EE_L, orc.EPS_TT_R, orc.MU_NU], seed=91)
    out, ab = orc.eval_batch(inp, params, kinds, want_abs=True)
    assert np.all(out > 0) and np.all(np.abs(ab - out) <= tol * out)
    w = np.random.default_rng(92).uniform(0.1, 3.0, size=(4, inp["T"].size))
    out, ab = orc.eval_weights(inp, w, want_abs=True)
    assert np.all(out > 0) and np.all(np.abs(ab - out) <= tol * out)
    mc = wl.make_components(n_comp=3, n_E=30, n_T=60, n_rec=31, n_periods=2, seed=42)
    kinds3 = np.array([orc.EPS_EE_L, orc.MU_NU, orc.RATE_0, orc.RATE_0 + 2], np.int32)
    p3, _ = wl.random_points(3, kinds3, seed=93)
    out, ab = orc.eval_components(mc, p3, kinds3, want_abs=True)
    assert np.all(out > 0) and np.all(np.abs(ab - out) <= tol * out)
    Pp = np.clip(inp["P_e"][None, :] + np.random.default_rng(94).uniform(-0.2, 0.2, size=(6, inp["E"].size)), 0.0, 1.0)
    out, ab = orc.eval_pee(inp, params, kinds, Pp, want_abs=True)
    assert np.all(out > 0) and np.all(np.abs(ab - out) <= tol * out)
    # profiled: no pull -> the scale is the value; with a pull -> the value minus ((s^ - s0)/sigma)^2
    out, sc, ab = orc.eval_profile(inp, params, kinds, want_abs=True)
    assert np.all(out > 0) and np.all(np.abs(ab - out) <= tol * out)
    s0, sigma = 1.0, 0.05
    out, sc, ab = orc.eval_profile(inp, params, kinds, s0=s0, sigma=sigma, want_abs=True)
    pull = ((sc - s0) / sigma) ** 2
    assert np.all(pull > 0) and np.all(np.abs(ab + pull - out) <= 4 * tol * out)
