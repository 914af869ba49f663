"""CPU-only checks of the host side: the C-ABI library loads and exports every symbol that
include/rw.h declares (no compute without a GPU), the workload tables have the BASELINE shapes,
and the N>1 plumbing works under gloo with world_size 2."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2607_00488_b200 import sharding, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions(header="rw.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rw_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2607_00488_b200 import build
    lib_path = build.build()
    lib = ctypes.CDLL(lib_path)
    names = _declared_functions()
    assert {"rw_create", "rw_eval_batch", "rw_destroy", "rw_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "librw.so does not export %s" % n
    from paper_2607_00488_b200 import binding
    assert set(binding.EXPORTS) == set(names)
    # the bench-only probe library (include/rw_probe.h) is separate: librw.so must not carry it
    from paper_2607_00488_b200 import probe
    plib = ctypes.CDLL(build.build_probe())
    pnames = _declared_functions("rw_probe.h")
    assert set(probe.EXPORTS) == set(pnames) and pnames
    for n in pnames:
        assert hasattr(plib, n), "librw_probe.so does not export %s" % n
        assert not hasattr(lib, n), "librw.so exports the measurement helper %s" % n


def test_binding_constants_match_the_header():
    """Every RW_* enumerator of include/rw.h that the binding also defines has the same value there (the binding
    retypes them; a drift would send the wrong flag or parameter kind through the ABI)."""
    from paper_2607_00488_b200 import binding
    text = open(os.path.join(ROOT, "include", "rw.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    header = {}
    for body in re.findall(r"enum\s*\w*\s*\{(.*?)\}", text, flags=re.S):
        nxt = 0
        for item in body.split(","):
            item = item.strip()
            if not item:
                continue
            m = re.match(r"(RW_[A-Z0-9_]+)\s*(?:=\s*(.+))?$", item, flags=re.S)
            assert m, item
            if m.group(2) is not None:
                expr = re.sub(r"(\d+)u\b", r"\1", m.group(2))
                expr = re.sub(r"RW_[A-Z0-9_]+", lambda mm: str(header[mm.group(0)]), expr)
                nxt = int(eval(expr, {"__builtins__": {}}))            # noqa: S307 (header arithmetic only)
            header[m.group(1)] = nxt
            nxt += 1
    assert header["RW_SLICED"] == 1 << 11 and header["RW_MU_NU"] == 6 and header["RW_N_KINDS"] == 11
    checked = 0
    for name, value in header.items():
        if hasattr(binding, name):
            assert getattr(binding, name) == value, "%s: header %d, binding %d" % (name, value, getattr(binding, name))
            checked += 1
    assert checked >= 12, checked


def test_abi_argument_errors_without_a_gpu():
    """Pure host-side validation paths return statuses, never crash (no kernel is launched)."""
    from paper_2607_00488_b200 import binding
    L = binding.load_library()
    nbytes = ctypes.c_size_t(0)
    inp = binding.rw_inputs()
    assert L.rw_workspace_bytes(ctypes.byref(inp), 16, ctypes.byref(nbytes)) == -1      # zero sizes
    inp.n_E, inp.n_T, inp.n_rec, inp.n_periods = 201, 100, 60, 1
    assert L.rw_workspace_bytes(ctypes.byref(inp), 0, ctypes.byref(nbytes)) == -1       # max_batch <= 0
    assert L.rw_workspace_bytes(ctypes.byref(inp), 121, ctypes.byref(nbytes)) == 0
    assert nbytes.value > 100 * 60 * 8 and nbytes.value % 256 == 0
    small = nbytes.value
    inp.n_T, inp.n_rec = 16384, 8192
    inp.mem_kind = binding.RW_MEM_DEVICE
    assert L.rw_workspace_bytes(ctypes.byref(inp), 65536, ctypes.byref(nbytes)) == 0
    assert small < nbytes.value < 5 << 30          # borrowed R: no copy; scratch = one <= 4 GiB chunk of N' + partials
    ctx = ctypes.c_void_p(None)
    assert L.rw_create(ctypes.byref(inp), 65536, None, 0, None, ctypes.byref(ctx)) in (-1, -2)
    assert ctx.value is None
    assert L.rw_eval_batch(None, None, 1, 0, None, None, None, 0, None) == -1
    assert L.rw_destroy(None) == 0
    assert b"invalid" in L.rw_strerror(-1)
    assert L.rw_last_error(None)                   # the failed rw_create left a message


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2607_00488_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.load_library()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00488_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "rw_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f


def test_baseline_config_shapes():
    shapes = {"cfg1_tiny_nsi": (201, 100, 60, 1, 121, 2), "cfg2_mm_lowE": (513, 1000, 500, 1, 1000, 1),
              "cfg3_nsi4": (4096, 4096, 2048, 1, 10000, 4)}
    for name, (n_E, n_T, n_rec, D, P, k) in shapes.items():
        inp = wl.make(name)
        assert inp["E"].size == n_E and inp["R"].shape == (D, n_T, n_rec)
        assert inp["N_mc"].shape == (D, n_T) and inp["counts"].shape == (D, n_rec)
        assert np.all(inp["R"] >= 0) and np.all(inp["R"].sum(axis=2) <= 1 + 1e-12)
        p, kinds = wl.scan_points(name)
        assert p.shape == (P, k) and len(kinds) == k
    p4, k4 = wl.scan_points("cfg4_dense")
    assert p4.shape == (65536, 7) and np.all(p4[:, 6] >= 1e-12) and np.all(p4[:, 6] <= 1e-10)
    p5, k5 = wl.scan_points("cfg5_joint6")
    assert p5.shape == (1000000, 6) and list(k5) == [0, 1, 4, 5, 2, 6]
    # Latin hypercube: every one of the 1e6 strata of every dimension holds exactly one point
    assert np.unique(np.floor((p5[:, 0] + 0.5) * 1e6).astype(np.int64)).size == 1000000
    assert 1000000 == 61 * 16384 + 576


def test_shard_range_partitions_every_point_once():
    for P, world in ((65536, 8), (1000003, 8), (5, 8), (121, 2)):
        seen = np.zeros(P, int)
        for r in range(world):
            lo, hi = sharding.shard_range(P, r, world)
            seen[lo:hi] += 1
        assert np.all(seen == 1)


_WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_2607_00488_b200 import sharding
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
p, kinds = sharding.rank_points("cfg1_tiny_nsi", rank)
assert p.shape == (121, 2)
# ranks fold different points of the same shape
g = [torch.zeros(121, 2, dtype=torch.float64) for _ in range(world)]
dist.all_gather(g, torch.from_numpy(p))
assert not torch.equal(g[0], g[1])
ms = sharding.max_over_ranks(10.0 + 5.0 * rank, "cpu", world)
assert ms == 15.0, ms
v = sharding.whole_job_value(world, 121, 4, ms)
assert abs(v - 2 * 121 * 4 / 0.015) < 1e-9
# strong scaling: one scan split into contiguous shards (61 + 60 points), every rank evaluates its own (here with the CPU
# oracle -- there is no GPU on this box), the shards are gathered into out[P] in scan order on every rank
import numpy as np
from oracle import rw_oracle as orc
from paper_2607_00488_b200 import workloads as wl
orc.build()
inp = wl.make("cfg1_tiny_nsi")
params, kinds = wl.scan_points("cfg1_tiny_nsi")
P = params.shape[0]
lo, hi = sharding.shard_range(P, rank, world)
assert (lo, hi) == ((0, 61) if rank == 0 else (61, 121))
mine = torch.from_numpy(np.asarray(orc.eval_batch(inp, params[lo:hi], kinds)))
pad = torch.zeros(sharding.shard_pad(P, world), dtype=torch.float64)
gathered = torch.empty(world * pad.numel(), dtype=torch.float64)
whole = sharding.gather_shards(mine, pad, gathered, P, world)
ref = torch.from_numpy(np.asarray(orc.eval_batch(inp, params, kinds)))
assert whole.shape == (P,) and torch.equal(whole, ref), (whole - ref).abs().max()
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank" + str(rank) + "-ok\n")
sys.stdout.flush()
"""


def test_two_rank_gloo_plumbing(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29641", str(script)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    p = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert p.returncode == 0, p.stdout + p.stderr
    assert "rank0-ok" in p.stdout and "rank1-ok" in p.stdout


def test_reference_arm_non_zero_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       capture_output=True, text=True, timeout=120, env=env)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the CPU oracle arm) prints one JSON line with the contract's keys."""
    import json
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config",
                        "cfg1_tiny_nsi", "--steps", "1", "--warmup", "3"], capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr
    line = json.loads(p.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                "scaling", "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["config"]["workload"] == "cfg1_tiny_nsi"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
