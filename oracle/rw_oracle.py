"""ctypes loader for the CPU oracle (oracle/rw_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, ``__graft_entry__.smoke()`` and
bench.py's ``cpu_baseline`` / ``--impl reference`` legs may import this module.
It imports nothing from ``paper_2607_00488_b200`` and the package never imports it.

Every function is a thin marshalling layer over the C routine of the same name;
see rw_oracle.c for the PAPER.md passage each one restates.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rw_oracle.c")
_LIB = os.path.join(_HERE, "librw_oracle.so")

# param kinds (DESIGN.md "param_kind" table)
EPS_EE_L, EPS_EE_R, EPS_MM_L, EPS_MM_R, EPS_TT_L, EPS_TT_R, MU_NU = range(7)
N_KINDS = 7
RATE_0 = 7          # kind 7 + c: rate scale of signal component c (eval_components only)


def build(force=False):
    """Compile rw_oracle.c with gcc (plain C99, no FMA contraction, OpenMP over points)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-Wall", "-ffp-contract=off", "-fopenmp", "-shared",
           "-fPIC", _SRC, "-o", _LIB, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


class Consts(C.Structure):
    _fields_ = [("sin2_theta_w", C.c_double), ("m_e", C.c_double),
                ("G_F", C.c_double), ("alpha_em", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_tmax.restype = C.c_double
        L.orc_tmax.argtypes = [C.c_double, C.c_double]
        L.orc_dsigma_weak.restype = C.c_double
        L.orc_dsigma_weak.argtypes = [C.POINTER(Consts)] + [C.c_double] * 4
        L.orc_dsigma_mm.restype = C.c_double
        L.orc_dsigma_mm.argtypes = [C.POINTER(Consts)] + [C.c_double] * 3
        L.orc_deviance.restype = C.c_double
        L.orc_eq18.restype = C.c_double
        L.orc_eval_batch.restype = C.c_int
        _lib = L
    return _lib


def default_consts():
    c = Consts()
    lib().orc_default_consts(C.byref(c))
    return c


def _a(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _p(x):
    return x.ctypes.data_as(_dp)


def long_double_mant_dig():
    return lib().orc_long_double_mant_dig()


def max_threads():
    return lib().orc_max_threads()


def tmax(E, m_e=None):
    m_e = default_consts().m_e if m_e is None else m_e
    return lib().orc_tmax(float(E), float(m_e))


def sm_couplings(consts=None):
    c = consts or default_consts()
    gL = (C.c_double * 3)()
    gR = (C.c_double * 3)()
    lib().orc_sm_couplings(C.byref(c), gL, gR)
    return np.array(gL[:]), np.array(gR[:])


def dsigma_weak(E, T, gL, gR, consts=None):
    c = consts or default_consts()
    return lib().orc_dsigma_weak(C.byref(c), float(E), float(T), float(gL), float(gR))


def dsigma_mm(E, T, mu_nu, consts=None):
    c = consts or default_consts()
    return lib().orc_dsigma_mm(C.byref(c), float(E), float(T), float(mu_nu))


def theta_vector(params, kinds):
    th = np.zeros(N_KINDS)
    for v, k in zip(params, kinds):
        th[int(k)] = v
    return th


def _flavour_probs(inp):
    """P_e, P_mu, P_tau; default split of 1-P_e by f_tau (reading R3)."""
    P_e = _a(inp["P_e"])
    if inp.get("P_mu") is not None and inp.get("P_tau") is not None:
        return P_e, _a(inp["P_mu"]), _a(inp["P_tau"])
    f_tau = inp.get("f_tau", 0.5)
    return P_e, _a((1.0 - P_e) * (1.0 - f_tau)), _a((1.0 - P_e) * f_tau)


def spectrum(inp, theta, consts=None):
    """S_theta(T_i), Eq. (12) with the cut; ``theta`` is the 7-vector indexed by kind."""
    c = consts or default_consts()
    E, fw, T = _a(inp["E"]), _a(inp["flux_w"]), _a(inp["T"])
    P_e, P_mu, P_tau = _flavour_probs(inp)
    th = _a(theta)
    out = np.empty(T.size)
    lib().orc_spectrum(C.byref(c), C.c_int(E.size), _p(E), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
                       C.c_int(T.size), _p(T), _p(th), _p(out))
    return out


def weights(inp, theta, consts=None):
    c = consts or default_consts()
    E, fw, T = _a(inp["E"]), _a(inp["flux_w"]), _a(inp["T"])
    P_e, P_mu, P_tau = _flavour_probs(inp)
    th = _a(theta)
    out = np.empty(T.size)
    lib().orc_weights(C.byref(c), C.c_int(E.size), _p(E), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
                      C.c_int(T.size), _p(T), _p(th), _p(out))
    return out


def fold(w, N_mc, R, bkg):
    w, N_mc, R, bkg = _a(w), _a(N_mc), _a(R), _a(bkg)
    n_T, n_rec = R.shape
    assert w.size == n_T and N_mc.size == n_T and bkg.size == n_rec
    out = np.empty(n_rec)
    lib().orc_fold(C.c_int(n_T), C.c_int(n_rec), _p(w), _p(N_mc), _p(R), _p(bkg), _p(out))
    return out


def deviance(mu, n):
    mu, n = _a(mu), _a(n)
    assert mu.size == n.size
    return lib().orc_deviance(C.c_int(mu.size), _p(mu), _p(n))


def eq18(mu, n):
    mu, n = _a(mu), _a(n)
    assert mu.size == n.size
    return lib().orc_eq18(C.c_int(mu.size), _p(mu), _p(n))


def eval_batch(inp, params, kinds, want_mu=False, want_abs=False, full_eq18=False,
               nthreads=1, consts=None):
    """Whole path for params[P][k].  ``inp`` holds E, flux_w, P_e[, P_mu, P_tau | f_tau], T,
    N_mc[D][n_T], R[D][n_T][n_rec], bkg[D][n_rec], counts[D][n_rec].
    Returns out[P] (and mu[P][D][n_rec], abs[P] when asked)."""
    c = consts or default_consts()
    E, fw, T = _a(inp["E"]), _a(inp["flux_w"]), _a(inp["T"])
    P_e, P_mu, P_tau = _flavour_probs(inp)
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    assert T.size == n_T
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    assert kinds.size == k
    out = np.empty(P)
    mu = np.empty((P, D, n_rec)) if want_mu else None
    ab = np.empty(P) if want_abs else None
    rc = lib().orc_eval_batch(
        C.byref(c), C.c_int(E.size), _p(E), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
        C.c_int(n_T), _p(T), C.c_int(n_rec), C.c_int(D), _p(N_mc), _p(R), _p(bkg), _p(counts),
        C.c_int64(P), C.c_int(k), kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params),
        _p(out), _p(mu) if want_mu else None, _p(ab) if want_abs else None,
        C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_batch: invalid param kinds")
    res = [out]
    if want_mu:
        res.append(mu)
    if want_abs:
        res.append(ab)
    return res[0] if len(res) == 1 else tuple(res)


def eval_weights(inp, w, want_mu=False, want_abs=False, full_eq18=False, nthreads=1):
    """Fold + likelihood for caller-supplied weights w[P][n_T] (Eq. 1 with an arbitrary diag(r))."""
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    w = _a(w)
    if w.ndim == 1:
        w = w[None]
    P = w.shape[0]
    assert w.shape[1] == n_T
    out = np.empty(P)
    mu = np.empty((P, D, n_rec)) if want_mu else None
    ab = np.empty(P) if want_abs else None
    L = lib()
    L.orc_eval_weights.restype = C.c_int
    L.orc_eval_weights(C.c_int(n_T), C.c_int(n_rec), C.c_int(D), _p(N_mc), _p(R), _p(bkg), _p(counts),
                       C.c_int64(P), _p(w), _p(out), _p(mu) if want_mu else None,
                       _p(ab) if want_abs else None, C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    res = [out]
    if want_mu:
        res.append(mu)
    if want_abs:
        res.append(ab)
    return res[0] if len(res) == 1 else tuple(res)


def profile_scale(S, B, n, s0=1.0, sigma=0.0, full_eq18=False):
    """(s_hat, f_min) of f(s) = deviance(s S + B, n) + ((s - s0)/sigma)^2 over s >= 0 (pull iff sigma > 0)."""
    S, B, n = _a(S).ravel(), _a(B).ravel(), _a(n).ravel()
    assert S.size == B.size == n.size
    L = lib()
    L.orc_profile_scale.restype = C.c_double
    f = C.c_double(0.0)
    s = L.orc_profile_scale(C.c_int(S.size), _p(S), _p(B), _p(n), C.c_double(s0), C.c_double(sigma),
                            C.c_int(1 if full_eq18 else 0), C.byref(f))
    return s, f.value


def eval_profile(inp, params, kinds, s0=1.0, sigma=0.0, want_abs=False, full_eq18=False, nthreads=1, consts=None):
    """Whole path with the overall rate normalisation profiled per point. Returns (out[P], s_hat[P][, abs[P]])."""
    c = consts or default_consts()
    E, fw, T = _a(inp["E"]), _a(inp["flux_w"]), _a(inp["T"])
    P_e, P_mu, P_tau = _flavour_probs(inp)
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    out, sc = np.empty(P), np.empty(P)
    ab = np.empty(P) if want_abs else None
    L = lib()
    L.orc_eval_profile.restype = C.c_int
    rc = L.orc_eval_profile(
        C.byref(c), C.c_int(E.size), _p(E), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
        C.c_int(n_T), _p(T), C.c_int(n_rec), C.c_int(D), _p(N_mc), _p(R), _p(bkg), _p(counts),
        C.c_int64(P), C.c_int(k), kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params),
        C.c_double(s0), C.c_double(sigma), _p(out), _p(sc), _p(ab) if want_abs else None,
        C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_profile: invalid param kinds")
    return (out, sc, ab) if want_abs else (out, sc)


def eval_components(inp, params, kinds, want_mu=False, want_abs=False, full_eq18=False, nthreads=1, consts=None):
    """Multi-component path (Eq. 17).  ``inp`` as for eval_batch, but flux_w, P_e (and P_mu, P_tau if given) are
    [n_comp][n_E] and ``comp_of_T`` [n_T] assigns every recoil bin to a component; kinds 7 + c are rate scales."""
    c = consts or default_consts()
    E, T = _a(inp["E"]), _a(inp["T"])
    fw = np.atleast_2d(_a(inp["flux_w"]))
    n_comp, n_E = fw.shape
    P_e = np.atleast_2d(_a(inp["P_e"]))
    if inp.get("P_mu") is not None and inp.get("P_tau") is not None:
        P_mu, P_tau = np.atleast_2d(_a(inp["P_mu"])), np.atleast_2d(_a(inp["P_tau"]))
    else:
        f_tau = inp.get("f_tau", 0.5)
        P_mu, P_tau = _a((1.0 - P_e) * (1.0 - f_tau)), _a((1.0 - P_e) * f_tau)
    comp = np.ascontiguousarray(inp.get("comp_of_T", np.zeros(T.size)), dtype=np.int32)
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    out = np.empty(P)
    mu = np.empty((P, D, n_rec)) if want_mu else None
    ab = np.empty(P) if want_abs else None
    L = lib()
    L.orc_eval_components.restype = C.c_int
    rc = L.orc_eval_components(
        C.byref(c), C.c_int(n_E), _p(E), C.c_int(n_comp), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
        C.c_int(n_T), _p(T), comp.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int(n_rec), C.c_int(D),
        _p(N_mc), _p(R), _p(bkg), _p(counts), C.c_int64(P), C.c_int(k),
        kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params), _p(out), _p(mu) if want_mu else None,
        _p(ab) if want_abs else None, C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_components: invalid kinds / component indices")
    res = [out]
    if want_mu:
        res.append(mu)
    if want_abs:
        res.append(ab)
    return res[0] if len(res) == 1 else tuple(res)


def eval_grad(inp, params, kinds, nthreads=1, consts=None):
    """(-2lnL[P], d(-2lnL)/dtheta [P][k]) for the (multi-)component path; inputs as eval_components
    (a single component may pass 1-D flux_w / P_e and no comp_of_T)."""
    c = consts or default_consts()
    E, T = _a(inp["E"]), _a(inp["T"])
    fw = np.atleast_2d(_a(inp["flux_w"]))
    n_comp, n_E = fw.shape
    P_e = np.atleast_2d(_a(inp["P_e"]))
    if inp.get("P_mu") is not None and inp.get("P_tau") is not None:
        P_mu, P_tau = np.atleast_2d(_a(inp["P_mu"])), np.atleast_2d(_a(inp["P_tau"]))
    else:
        f_tau = inp.get("f_tau", 0.5)
        P_mu, P_tau = _a((1.0 - P_e) * (1.0 - f_tau)), _a((1.0 - P_e) * f_tau)
    comp = np.ascontiguousarray(inp.get("comp_of_T", np.zeros(T.size)), dtype=np.int32)
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    out, grad = np.empty(P), np.empty((P, k))
    L = lib()
    L.orc_eval_grad.restype = C.c_int
    rc = L.orc_eval_grad(
        C.byref(c), C.c_int(n_E), _p(E), C.c_int(n_comp), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
        C.c_int(n_T), _p(T), comp.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int(n_rec), C.c_int(D),
        _p(N_mc), _p(R), _p(bkg), _p(counts), C.c_int64(P), C.c_int(k),
        kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params), _p(out), _p(grad), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_grad: invalid kinds / component indices")
    return out, grad


def eval_pee(inp, params, kinds, P_e_pts, want_mu=False, want_abs=False, full_eq18=False, nthreads=1, consts=None):
    """Whole path with a survival-probability table per point, P_e_pts[P][n_E]; the SM reference keeps inp["P_e"]."""
    c = consts or default_consts()
    E, fw, T, P_e = _a(inp["E"]), _a(inp["flux_w"]), _a(inp["T"]), _a(inp["P_e"])
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    Pp = _a(P_e_pts)
    assert Pp.shape == (P, E.size)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    out = np.empty(P)
    mu = np.empty((P, D, n_rec)) if want_mu else None
    ab = np.empty(P) if want_abs else None
    L = lib()
    L.orc_eval_pee.restype = C.c_int
    rc = L.orc_eval_pee(
        C.byref(c), C.c_int(E.size), _p(E), _p(fw), _p(P_e), C.c_double(inp.get("f_tau", 0.5)),
        C.c_int(n_T), _p(T), C.c_int(n_rec), C.c_int(D), _p(N_mc), _p(R), _p(bkg), _p(counts),
        C.c_int64(P), C.c_int(k), kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params), _p(Pp),
        _p(out), _p(mu) if want_mu else None, _p(ab) if want_abs else None,
        C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_pee: invalid param kinds")
    res = [out]
    if want_mu:
        res.append(mu)
    if want_abs:
        res.append(ab)
    return res[0] if len(res) == 1 else tuple(res)


def eval_pee_components(inp, params, kinds, P_e_pts, want_mu=False, want_abs=False, full_eq18=False, nthreads=1,
                        consts=None):
    """Per-point survival probabilities with several components and / or explicit nominal P_mu, P_tau tables
    (reading R17).  ``inp`` as for eval_components; P_e_pts is [P][n_comp][n_E] ([P][n_E] for one)."""
    c = consts or default_consts()
    E, T = _a(inp["E"]), _a(inp["T"])
    fw = np.atleast_2d(_a(inp["flux_w"]))
    n_comp, n_E = fw.shape
    P_e = np.atleast_2d(_a(inp["P_e"]))
    have = inp.get("P_mu") is not None and inp.get("P_tau") is not None
    f_tau = float(inp.get("f_tau", 0.5))
    if have:
        P_mu, P_tau = np.atleast_2d(_a(inp["P_mu"])), np.atleast_2d(_a(inp["P_tau"]))
    else:
        P_mu, P_tau = _a((1.0 - P_e) * (1.0 - f_tau)), _a((1.0 - P_e) * f_tau)
    comp = np.ascontiguousarray(inp.get("comp_of_T", np.zeros(T.size)), dtype=np.int32)
    R = _a(inp["R"])
    if R.ndim == 2:
        R = R[None]
    D, n_T, n_rec = R.shape
    N_mc = _a(inp["N_mc"]).reshape(D, n_T)
    bkg = _a(inp["bkg"]).reshape(D, n_rec)
    counts = _a(inp["counts"]).reshape(D, n_rec)
    params = _a(params)
    if params.ndim == 1:
        params = params[:, None]
    P, k = params.shape
    pts = _a(P_e_pts).reshape(P, n_comp, n_E)
    kinds = np.ascontiguousarray(kinds, dtype=np.int32)
    out = np.empty(P)
    mu = np.empty((P, D, n_rec)) if want_mu else None
    ab = np.empty(P) if want_abs else None
    L = lib()
    L.orc_eval_pee_components.restype = C.c_int
    rc = L.orc_eval_pee_components(
        C.byref(c), C.c_int(n_E), _p(E), C.c_int(n_comp), _p(fw), _p(P_e), _p(P_mu), _p(P_tau),
        C.c_int(1 if have else 0), C.c_double(f_tau), C.c_int(n_T), _p(T), comp.ctypes.data_as(C.POINTER(C.c_int32)),
        C.c_int(n_rec), C.c_int(D), _p(N_mc), _p(R), _p(bkg), _p(counts), C.c_int64(P), C.c_int(k),
        kinds.ctypes.data_as(C.POINTER(C.c_int32)), _p(params), _p(pts), _p(out), _p(mu) if want_mu else None,
        _p(ab) if want_abs else None, C.c_int(1 if full_eq18 else 0), C.c_int(int(nthreads)))
    if rc != 0:
        raise ValueError("orc_eval_pee_components: invalid kinds / component indices")
    res = [out]
    if want_mu:
        res.append(mu)
    if want_abs:
        res.append(ab)
    return res[0] if len(res) == 1 else tuple(res)
