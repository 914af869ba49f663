"""ctypes binding of include/rw_probe.h (librw_probe.so): the FP64 issue-rate probes bench.py uses as roofline
denominators.  Measurement helper only -- the product library librw.so does not contain it."""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librw_probe.so")
EXPORTS = ("rw_probe_scratch_bytes", "rw_probe_fp64_peak")

_lib = None


def load_library():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s not found: build it with `python -m paper_2607_00488_b200.build`" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        L.rw_probe_scratch_bytes.restype = C.c_size_t
        L.rw_probe_fp64_peak.argtypes = [C.c_int32, C.c_int32, C.c_void_p, C.c_size_t, C.POINTER(C.c_double), C.c_void_p]
        L.rw_probe_fp64_peak.restype = C.c_int
        _lib = L
    return _lib


def fp64_peak(kind, iters=20000):
    """TFLOP/s of the register-resident FP64 probe on the current device (0 = DFMA, 1 = DMMA m8n8k4)."""
    L = load_library()
    nbytes = int(L.rw_probe_scratch_bytes())
    if nbytes == 0:
        raise RuntimeError("rw_probe_scratch_bytes: no CUDA device")
    scratch = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    out = C.c_double(0.0)
    rc = L.rw_probe_fp64_peak(int(kind), int(iters), C.c_void_p(scratch.data_ptr()), nbytes, C.byref(out),
                              C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise RuntimeError("rw_probe_fp64_peak failed with status %d" % rc)
    return out.value
