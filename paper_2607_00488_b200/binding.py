"""Thin ctypes binding of include/rw.h -- argument marshalling only.

Every step of the likelihood path runs in the CUDA kernels of librw.so; PyTorch is used here
for device memory (the workspace, parameter and output tensors) and the CUDA stream, nothing
else.  There is no CPU fallback: if librw.so is missing or the device is not sm_100 the calls
raise.  Names mirror the C ABI: rw_workspace_bytes / rw_create / rw_set_counts /
rw_eval_batch / rw_get_table / rw_destroy.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librw.so")

# param kinds (include/rw.h)
RW_EPS_EE_L, RW_EPS_EE_R, RW_EPS_MM_L, RW_EPS_MM_R, RW_EPS_TT_L, RW_EPS_TT_R, RW_MU_NU = range(7)
RW_RATE_0 = 7        # RW_RATE_0 + c: rate scale of signal component c
RW_MEM_HOST, RW_MEM_DEVICE = 0, 1
RW_FULL_EQ18 = 1 << 0
RW_MODE_AUTO, RW_MODE_STREAM, RW_MODE_GEMM, RW_MODE_COLLAPSED, RW_MODE_RIDGE = 0, 1 << 4, 2 << 4, 3 << 4, 4 << 4
RW_PARAM_HOST, RW_OUT_HOST, RW_FP32, RW_SLICED, RW_SLICED_FAST, RW_SLICED_STRICT = 1 << 8, 1 << 9, 1 << 10, 1 << 11, 1 << 12, 1 << 13
RW_CREATE_FP32, RW_CREATE_SLICED = 1, 2
RW_TABLE_S_SM, RW_TABLE_BASIS, RW_TABLE_WHAT, RW_TABLE_G = 0, 1, 2, 3
RW_STATIC_MAX_N_REC = 8192
_MODES = {"auto": RW_MODE_AUTO, "stream": RW_MODE_STREAM, "gemm": RW_MODE_GEMM, "collapsed": RW_MODE_COLLAPSED,
          "ridge": RW_MODE_RIDGE}

EXPORTS = ("rw_workspace_bytes", "rw_create", "rw_set_counts", "rw_eval_batch", "rw_eval_certified", "rw_strict_fallback_count", "rw_eval_weights", "rw_eval_profile", "rw_eval_grad", "rw_eval_pee", "rw_get_table",
           "rw_launch_count", "rw_profile_begin", "rw_profile_end", "rw_destroy", "rw_strerror",
           "rw_last_error", "rw_fold_weights_static")

_dp = C.POINTER(C.c_double)


class rw_constants(C.Structure):
    _fields_ = [("sin2_theta_w", C.c_double), ("m_e_MeV", C.c_double), ("G_F_MeV2", C.c_double),
                ("alpha_em", C.c_double)]


class rw_inputs(C.Structure):
    _fields_ = [("n_E", C.c_int32), ("E_MeV", C.c_void_p), ("flux_w", C.c_void_p), ("P_e", C.c_void_p),
                ("P_mu", C.c_void_p), ("P_tau", C.c_void_p), ("f_tau", C.c_double),
                ("n_T", C.c_int32), ("T_MeV", C.c_void_p), ("n_rec", C.c_int32), ("n_periods", C.c_int32),
                ("N_mc", C.c_void_p), ("R", C.c_void_p), ("bkg", C.c_void_p), ("counts", C.c_void_p),
                ("consts", rw_constants), ("mem_kind", C.c_int32), ("create_flags", C.c_uint32),
                ("n_comp", C.c_int32), ("comp_of_T", C.c_void_p)]


def _sliced_flag(sliced):
    """sliced = False | True (FP64-grade, RW_SLICED) | "fast" (top four slices, FP32-grade, RW_SLICED_FAST) |
    "strict" / "fast-strict" (the same with RW_SLICED_STRICT: uncertified points are recomputed in FP64)."""
    if sliced in ("fast", "fast-strict"):
        return RW_SLICED_FAST | (RW_SLICED_STRICT if sliced == "fast-strict" else 0)
    if sliced == "strict":
        return RW_SLICED | RW_SLICED_STRICT
    return RW_SLICED if sliced else 0


class RwError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("rw status %d: %s" % (status, msg))
        self.status = status


_lib = None


def load_library():
    """dlopen librw.so and declare the prototypes.  Fails loudly when the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("%s not found: build it with `python -m paper_2607_00488_b200.build` "
                           "(there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    L.rw_workspace_bytes.argtypes = [C.POINTER(rw_inputs), C.c_int64, C.POINTER(C.c_size_t)]
    L.rw_create.argtypes = [C.POINTER(rw_inputs), C.c_int64, C.c_void_p, C.c_size_t, C.c_void_p,
                            C.POINTER(C.c_void_p)]
    L.rw_set_counts.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
    L.rw_eval_batch.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int32),
                                C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_certified.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int32),
                                    C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_certified.restype = C.c_int
    L.rw_strict_fallback_count.argtypes = [C.c_void_p]
    L.rw_strict_fallback_count.restype = C.c_int64
    L.rw_eval_weights.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_weights.restype = C.c_int
    L.rw_eval_profile.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int32), C.c_double,
                                  C.c_double, C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_profile.restype = C.c_int
    L.rw_eval_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int32), C.c_void_p,
                               C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_grad.restype = C.c_int
    L.rw_eval_pee.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.POINTER(C.c_int32), C.c_void_p,
                              C.c_void_p, C.c_void_p, C.c_uint32, C.c_void_p]
    L.rw_eval_pee.restype = C.c_int
    L.rw_get_table.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_int64)]
    L.rw_launch_count.argtypes = [C.c_void_p]
    L.rw_launch_count.restype = C.c_int64
    L.rw_destroy.argtypes = [C.c_void_p]
    L.rw_profile_begin.argtypes = [C.c_void_p]
    L.rw_profile_end.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
    L.rw_strerror.argtypes = [C.c_int]
    L.rw_strerror.restype = C.c_char_p
    L.rw_last_error.argtypes = [C.c_void_p]
    L.rw_last_error.restype = C.c_char_p
    L.rw_fold_weights_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.rw_fold_weights_static.restype = C.c_int
    for f in ("rw_workspace_bytes", "rw_create", "rw_set_counts", "rw_eval_batch", "rw_get_table",
              "rw_destroy", "rw_profile_begin", "rw_profile_end"):
        getattr(L, f).restype = C.c_int
    _lib = L
    return L


def _stream_ptr():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class _DevicePointer:
    """A float64 device array owned by the library, exposed through __cuda_array_interface__."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f8", "data": (int(ptr), False),
                                         "version": 3, "strides": None}


def fold_weights_static(w, N_mc, R, bkg, counts, out=None, out_mu=None, want_mu=False):
    """rw_fold_weights_static: -2lnL (and mu) of one point and one period for caller weights w[n_T], without a
    Reweighter and without any workspace -- for users who cannot allocate device memory (a plugin inside an
    application whose memory pool owns the GPU, a fit that must not trigger the device-wide synchronisation of
    cudaMalloc).  The library's built-in 4 MiB scratch serves all calls, so n_rec <= RW_STATIC_MAX_N_REC, and calls
    on one GPU must not overlap (keep them on one stream).  All arguments are CUDA float64 tensors; R is
    [n_T][n_rec] (a row pitch is taken from R.stride(0); it must be even).  Pass `out` (1 element) and `out_mu`
    ([n_rec]) to keep this wrapper allocation-free as well; they are created with torch.empty otherwise.
    Asynchronous on the current stream."""
    L = load_library()
    for name, t in (("w", w), ("N_mc", N_mc), ("R", R), ("bkg", bkg), ("counts", counts)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64):
            raise RwError(-1, "fold_weights_static: %s must be a CUDA float64 tensor" % name)
    n_T, n_rec = (int(x) for x in R.shape)
    if R.stride(1) != 1 and n_rec > 1:
        raise RwError(-1, "fold_weights_static: the reconstructed index of R must be contiguous")
    ldR = int(R.stride(0)) if n_T > 1 else max(n_rec + (n_rec & 1), int(R.stride(0)))
    assert w.numel() == n_T and N_mc.numel() == n_T and bkg.numel() == n_rec and counts.numel() == n_rec
    for t in (w, N_mc, bkg, counts):
        assert t.is_contiguous()
    if out is None:
        out = torch.empty(1, dtype=torch.float64, device=R.device)
    if want_mu and out_mu is None:
        out_mu = torch.empty(n_rec, dtype=torch.float64, device=R.device)
    with torch.cuda.device(R.device):
        rc = L.rw_fold_weights_static(C.c_void_p(w.data_ptr()), C.c_void_p(N_mc.data_ptr()), C.c_void_p(R.data_ptr()),
                                      ldR, n_T, n_rec, C.c_void_p(bkg.data_ptr()), C.c_void_p(counts.data_ptr()),
                                      C.c_void_p(out.data_ptr()),
                                      C.c_void_p(out_mu.data_ptr()) if out_mu is not None else None, _stream_ptr())
    if rc != 0:
        raise RwError(rc, L.rw_last_error(None).decode() or L.rw_strerror(rc).decode())
    return (out, out_mu) if (want_mu or out_mu is not None) else out


class Reweighter:
    """One rw_ctx: device-resident tables of one analysis + its workspace (a torch uint8 tensor).

    `inputs` is a dict with E, flux_w, P_e, [P_mu, P_tau | f_tau], T, N_mc[D][n_T], R[D][n_T][n_rec],
    bkg[D][n_rec], counts[D][n_rec] as numpy arrays (host: copied at create) or CUDA float64 torch tensors
    (R is borrowed, the rest copied).  Several signal components (Eq. 17): flux_w, P_e[, P_mu, P_tau] as
    [n_comp][n_E] plus comp_of_T[n_T]; parameter kinds RW_RATE_0 + c then scale component c."""

    def __init__(self, inputs, max_batch, device="cuda:0", consts=None, fp32=False, sliced=False):
        self._L = load_library()
        self._ctx = C.c_void_p(None)
        self.device = torch.device(device)
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2607_00488_b200 needs a CUDA device (sm_100a); no CPU fallback exists")
        torch.cuda.set_device(self.device)
        on_device = isinstance(inputs["R"], torch.Tensor)
        keep = {}

        def arr(name, required=True):
            v = inputs.get(name)
            if v is None:
                if required:
                    raise KeyError(name)
                return None
            if on_device:
                t = v.to(device=self.device, dtype=torch.float64).contiguous()
                keep[name] = t
                return C.c_void_p(t.data_ptr())
            a = np.ascontiguousarray(v, dtype=np.float64)
            keep[name] = a
            return C.c_void_p(a.ctypes.data)

        R = inputs["R"]
        if R.ndim == 2:
            R = R[None]
            inputs = dict(inputs, R=R)
        D, n_T, n_rec = (int(x) for x in R.shape)
        inp = rw_inputs()
        inp.n_E = int(np.prod(inputs["E"].shape))
        inp.E_MeV, inp.flux_w, inp.P_e = arr("E"), arr("flux_w"), arr("P_e")
        inp.P_mu, inp.P_tau = arr("P_mu", False), arr("P_tau", False)
        inp.f_tau = float(inputs.get("f_tau", 0.5))
        inp.n_T, inp.T_MeV = n_T, arr("T")
        inp.n_rec, inp.n_periods = n_rec, D
        inp.N_mc, inp.R, inp.bkg, inp.counts = arr("N_mc"), arr("R"), arr("bkg"), arr("counts")
        if consts:
            inp.consts = rw_constants(*[float(consts.get(k, 0.0)) for k in
                                        ("sin2_theta_w", "m_e_MeV", "G_F_MeV2", "alpha_em")])
        inp.mem_kind = RW_MEM_DEVICE if on_device else RW_MEM_HOST
        inp.create_flags = (RW_CREATE_FP32 if fp32 else 0) | (RW_CREATE_SLICED if sliced else 0)
        fw = inputs["flux_w"]
        inp.n_comp = int(fw.shape[0]) if fw.ndim == 2 else 1
        if inp.n_comp > 1:
            comp = inputs["comp_of_T"]
            if on_device:
                t = torch.as_tensor(comp).to(device=self.device, dtype=torch.int32).contiguous()
                keep["comp_of_T"] = t
                inp.comp_of_T = C.c_void_p(t.data_ptr())
            else:
                a = np.ascontiguousarray(comp.cpu().numpy() if isinstance(comp, torch.Tensor) else comp, dtype=np.int32)
                keep["comp_of_T"] = a
                inp.comp_of_T = C.c_void_p(a.ctypes.data)
        self.n_comp = inp.n_comp
        self.n_E, self.n_T, self.n_rec, self.n_periods = inp.n_E, n_T, n_rec, D
        self.max_batch = int(max_batch)
        nbytes = C.c_size_t(0)
        self._check(self._L.rw_workspace_bytes(C.byref(inp), self.max_batch, C.byref(nbytes)), None)
        self.workspace = torch.empty(nbytes.value + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) & ~255
        self._keep = keep            # borrowed device R must outlive the context
        ctx = C.c_void_p(None)
        self._check(self._L.rw_create(C.byref(inp), self.max_batch, C.c_void_p(base), nbytes.value,
                                      _stream_ptr(), C.byref(ctx)), None)
        self._ctx = ctx
        if not on_device:
            self._keep = {}

    # ------------------------------------------------------------------------------------------
    def _check(self, rc, ctx):
        if rc != 0:
            msg = self._L.rw_last_error(ctx).decode() or self._L.rw_strerror(rc).decode()
            raise RwError(rc, msg)

    def eval_batch(self, param, kinds, out=None, out_mu=None, want_mu=False, full_eq18=False, mode="auto", fp32=False,
                   sliced=False):
        """-2lnL[P] for param[P][k] (CUDA float64 tensor, or numpy/pinned CPU tensor => host path).

        Device params: asynchronous on the current stream, returns a CUDA tensor.
        Host params: H2D + kernels + D2H are enqueued on the current stream; returns a CPU tensor
        (pinned), valid after the stream is synchronised."""
        kinds_arr = (C.c_int32 * max(1, len(kinds)))(*[int(x) for x in kinds])
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | (RW_FP32 if fp32 else 0) | \
            _sliced_flag(sliced)
        host = not (isinstance(param, torch.Tensor) and param.is_cuda)
        if host:
            if isinstance(param, np.ndarray):
                param = torch.from_numpy(np.ascontiguousarray(param, dtype=np.float64))
            param = param.to(torch.float64).contiguous()
            if param.ndim == 1:
                param = param[:, None]
            P, k = param.shape
            if out is None:
                out = torch.empty(P, dtype=torch.float64, pin_memory=True)
            flags |= RW_PARAM_HOST | RW_OUT_HOST
            if want_mu and out_mu is None:
                out_mu = torch.empty((P, self.n_periods, self.n_rec), dtype=torch.float64, pin_memory=True)
        else:
            param = param.to(torch.float64).contiguous()
            if param.ndim == 1:
                param = param[:, None]
            P, k = param.shape
            if out is None:
                out = torch.empty(P, dtype=torch.float64, device=self.device)
            if want_mu and out_mu is None:
                out_mu = torch.empty((P, self.n_periods, self.n_rec), dtype=torch.float64, device=self.device)
        assert k == len(kinds), "param has %d columns but %d kinds were given" % (k, len(kinds))
        rc = self._L.rw_eval_batch(self._ctx, C.c_void_p(param.data_ptr()), P, k, kinds_arr,
                                   C.c_void_p(out.data_ptr()),
                                   C.c_void_p(out_mu.data_ptr()) if out_mu is not None else None,
                                   flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = param          # keep alive until the stream has consumed it
        return (out, out_mu) if (want_mu or out_mu is not None) else out

    def eval_certified(self, param, kinds, sliced=True, full_eq18=False, mode="auto", fp32=False):
        """(-2lnL[P], bound[P]) through a sliced contraction (rw_eval_certified): bound[p] is the certified
        max over bins of |mu~ - mu| / mu (0 where an FP64 path ran).  CUDA param[P][k] only."""
        if not (isinstance(param, torch.Tensor) and param.is_cuda):
            raise RwError(-4, "eval_certified needs a CUDA tensor param[P][k]")
        param = param.to(torch.float64).contiguous()
        if param.ndim == 1:
            param = param[:, None]
        P, k = param.shape
        assert k == len(kinds)
        kinds_arr = (C.c_int32 * max(1, len(kinds)))(*[int(x) for x in kinds])
        out = torch.empty(P, dtype=torch.float64, device=self.device)
        bound = torch.empty(P, dtype=torch.float64, device=self.device)
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | (RW_FP32 if fp32 else _sliced_flag(sliced))
        rc = self._L.rw_eval_certified(self._ctx, C.c_void_p(param.data_ptr()), P, k, kinds_arr,
                                       C.c_void_p(out.data_ptr()), C.c_void_p(bound.data_ptr()), flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = param
        return out, bound

    def strict_fallback_count(self):
        return int(self._L.rw_strict_fallback_count(self._ctx))

    def eval_profile(self, param, kinds, s0=1.0, sigma=0.0, full_eq18=False, mode="auto", sliced=False):
        """(-2lnL[P] with the overall signal normalisation profiled out, s_hat[P]) for CUDA param[P][k]
        (rw_eval_profile); sigma > 0 adds the Gaussian pull ((s - s0)/sigma)^2."""
        if not (isinstance(param, torch.Tensor) and param.is_cuda):
            raise RwError(-4, "eval_profile needs a CUDA tensor param[P][k]")
        param = param.to(torch.float64).contiguous()
        if param.ndim == 1:
            param = param[:, None]
        P, k = param.shape
        assert k == len(kinds)
        kinds_arr = (C.c_int32 * max(1, len(kinds)))(*[int(x) for x in kinds])
        out = torch.empty(P, dtype=torch.float64, device=self.device)
        scale = torch.empty(P, dtype=torch.float64, device=self.device)
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | _sliced_flag(sliced)
        rc = self._L.rw_eval_profile(self._ctx, C.c_void_p(param.data_ptr()), P, k, kinds_arr, float(s0), float(sigma),
                                     C.c_void_p(out.data_ptr()), C.c_void_p(scale.data_ptr()), flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = param
        return out, scale

    def eval_pee(self, param, kinds, P_e_pts, want_mu=False, full_eq18=False, mode="auto", sliced=False):
        """-2lnL[P] (and mu) with a survival-probability table per point, P_e_pts[P][n_E] (CUDA tensors; rw_eval_pee)."""
        if not (isinstance(param, torch.Tensor) and param.is_cuda and isinstance(P_e_pts, torch.Tensor) and P_e_pts.is_cuda):
            raise RwError(-4, "eval_pee needs CUDA tensors param[P][k] and P_e_pts[P][n_E]")
        param = param.to(torch.float64).contiguous()
        if param.ndim == 1:
            param = param[:, None]
        P, k = param.shape
        pts = P_e_pts.to(torch.float64).contiguous()
        assert pts.numel() == P * self.n_comp * self.n_E and k == len(kinds), "P_e_pts must be [P][n_comp][n_E]"
        kinds_arr = (C.c_int32 * max(1, len(kinds)))(*[int(x) for x in kinds])
        out = torch.empty(P, dtype=torch.float64, device=self.device)
        mu = torch.empty((P, self.n_periods, self.n_rec), dtype=torch.float64, device=self.device) if want_mu else None
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | _sliced_flag(sliced)
        rc = self._L.rw_eval_pee(self._ctx, C.c_void_p(param.data_ptr()), P, k, kinds_arr, C.c_void_p(pts.data_ptr()),
                                 C.c_void_p(out.data_ptr()), C.c_void_p(mu.data_ptr()) if want_mu else None,
                                 flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = (param, pts)
        return (out, mu) if want_mu else out

    def eval_grad(self, param, kinds, full_eq18=False, mode="auto", sliced=False):
        """(-2lnL[P], gradient[P][k]) for CUDA param[P][k] (rw_eval_grad).  sliced = True | "fast": the rows go through
        the INT8 contraction, every derivative row as its positive and its negative part."""
        if not (isinstance(param, torch.Tensor) and param.is_cuda):
            raise RwError(-4, "eval_grad needs a CUDA tensor param[P][k]")
        param = param.to(torch.float64).contiguous()
        if param.ndim == 1:
            param = param[:, None]
        P, k = param.shape
        assert k == len(kinds)
        kinds_arr = (C.c_int32 * max(1, len(kinds)))(*[int(x) for x in kinds])
        out = torch.empty(P, dtype=torch.float64, device=self.device)
        grad = torch.empty((P, k), dtype=torch.float64, device=self.device)
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | _sliced_flag(sliced)
        rc = self._L.rw_eval_grad(self._ctx, C.c_void_p(param.data_ptr()), P, k, kinds_arr,
                                  C.c_void_p(out.data_ptr()), C.c_void_p(grad.data_ptr()), flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = param
        return out, grad

    def eval_weights(self, w, out=None, out_mu=None, want_mu=False, full_eq18=False, mode="auto", sliced=False):
        """-2lnL[P] for caller-supplied weights w[P][n_T] (CUDA float64 tensor): the dense fold on arbitrary
        weights (rw_eval_weights).  Asynchronous on the current stream."""
        if not (isinstance(w, torch.Tensor) and w.is_cuda):
            raise RwError(-4, "eval_weights needs a CUDA tensor w[P][n_T]")
        w = w.to(torch.float64).contiguous()
        if w.ndim == 1:
            w = w[None]
        P, n_T = w.shape
        assert n_T == self.n_T, "w has %d columns, the recoil grid has %d bins" % (n_T, self.n_T)
        if out is None:
            out = torch.empty(P, dtype=torch.float64, device=self.device)
        if want_mu and out_mu is None:
            out_mu = torch.empty((P, self.n_periods, self.n_rec), dtype=torch.float64, device=self.device)
        flags = _MODES[mode] | (RW_FULL_EQ18 if full_eq18 else 0) | _sliced_flag(sliced)
        rc = self._L.rw_eval_weights(self._ctx, C.c_void_p(w.data_ptr()), P, C.c_void_p(out.data_ptr()),
                                     C.c_void_p(out_mu.data_ptr()) if out_mu is not None else None,
                                     flags, _stream_ptr())
        self._check(rc, self._ctx)
        self._last_param = w
        return (out, out_mu) if (want_mu or out_mu is not None) else out

    def set_counts(self, counts):
        if isinstance(counts, torch.Tensor) and counts.is_cuda:
            c = counts.to(torch.float64).contiguous()
            rc = self._L.rw_set_counts(self._ctx, C.c_void_p(c.data_ptr()), RW_MEM_DEVICE, _stream_ptr())
        else:
            c = np.ascontiguousarray(counts.cpu().numpy() if isinstance(counts, torch.Tensor) else counts,
                                     dtype=np.float64)
            rc = self._L.rw_set_counts(self._ctx, C.c_void_p(c.ctypes.data), RW_MEM_HOST, _stream_ptr())
        self._check(rc, self._ctx)

    def table(self, which):
        """Copy of a setup table as a CUDA tensor (RW_TABLE_S_SM / _BASIS / _WHAT)."""
        ptr, n = C.c_void_p(None), C.c_int64(0)
        self._check(self._L.rw_get_table(self._ctx, int(which), C.byref(ptr), C.byref(n)), self._ctx)
        view = _DevicePointer(ptr.value, n.value)
        return torch.as_tensor(view, device=self.device).clone()

    def profile_begin(self):
        self._check(self._L.rw_profile_begin(self._ctx), self._ctx)

    def profile_end(self):
        """(summed fold-kernel ms, launches timed) since profile_begin; synchronises."""
        ms, n = C.c_double(0.0), C.c_int64(0)
        self._check(self._L.rw_profile_end(self._ctx, C.byref(ms), C.byref(n)), self._ctx)
        return ms.value, n.value

    def launch_count(self):
        return int(self._L.rw_launch_count(self._ctx))

    def close(self):
        if self._ctx:
            torch.cuda.synchronize(self.device)
            self._L.rw_destroy(self._ctx)
            self._ctx = C.c_void_p(None)
            self.workspace = None
            self._keep = {}

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
