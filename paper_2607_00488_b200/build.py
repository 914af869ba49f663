"""Builds librw.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

Run:  python -m paper_2607_00488_b200.build   (or __graft_entry__.build()).
The .so is git-ignored but travels to the GPU box with the gpurun snapshot."""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librw.so")
SOURCES = ["rw_api.cu", "rw_setup.cu", "rw_coef.cu", "rw_fold_stream.cu", "rw_fold_gemm.cu", "rw_fold_ridge.cu", "rw_fold_i8.cu", "rw_collapsed.cu", "rw_profile.cu", "rw_grad.cu", "rw_pee.cu", "rw_noalloc.cu"]
PROBE_LIB = os.path.join(HERE, "librw_probe.so")      # bench-only FP64 peak probe (include/rw_probe.h)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _newer(target, deps):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def build_probe(force=False):
    src = os.path.join(CSRC, "rw_probe.cu")
    hdr = os.path.join(HERE, "..", "include", "rw_probe.h")
    if not force and _newer(PROBE_LIB, [src, hdr]):
        return PROBE_LIB
    p = subprocess.run(["nvcc"] + [f for f in NVCC_FLAGS if f not in ("-Xptxas", "-v")] + ["-shared", src, "-o", PROBE_LIB],
                       capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, p.stdout, p.stderr))
    return PROBE_LIB


def build(force=False, verbose=False):
    hdrs = [os.path.join(CSRC, "rw_internal.h"), os.path.join(HERE, "..", "include", "rw.h")]
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    build_probe(force)
    if not force and _newer(LIB, srcs + hdrs):
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(objdir, os.path.basename(src).replace(".cu", ".o"))
        if not force and _newer(obj, [src] + hdrs):
            return obj, ""
        p = subprocess.run(["nvcc"] + NVCC_FLAGS + ["-c", src, "-o", obj], capture_output=True, text=True)
        if p.returncode != 0:
            raise RuntimeError("nvcc failed for %s:\n%s\n%s" % (src, p.stdout, p.stderr))
        return obj, p.stderr

    with ThreadPoolExecutor(max_workers=len(srcs)) as ex:
        res = list(ex.map(compile_one, srcs))
    if verbose:
        for _, log in res:
            sys.stderr.write(log)
    objs = [o for o, _ in res]
    p = subprocess.run(["nvcc", "-shared", "-o", LIB] + objs + ["-gencode", "arch=compute_100a,code=sm_100a"],
                       capture_output=True, text=True)
    if p.returncode != 0:
        raise RuntimeError("link failed:\n%s\n%s" % (p.stdout, p.stderr))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
