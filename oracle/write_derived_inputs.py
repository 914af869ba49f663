"""Writes paper_2607_00488_b200/workload_data/derived_inputs.npz -- the two inputs of the
BASELINE configs that are *defined through the SM prediction*:

  S_hat[i]   normalised SM recoil shape  S_SM(T_i)/sum S_SM   ("N_MC = SM spectrum x N events")
  counts[d][k]  seeded Poisson draw of the SM prediction  mu_SM = fold(w=1) + bkg
  line_ratio (config 1 only) line flux_w / sum(continuum flux_w) such that the 0.862 MeV
             line holds 30 % of the SM events on the recoil grid

This script calls ONLY oracle/ (plus the arithmetic-free table generators in
paper_2607_00488_b200/workloads.py); nothing here ever comes from the CUDA path.
Run from the repo root:  python oracle/write_derived_inputs.py
"""
import hashlib
import os
import sys
import time

import numpy as np

_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, _ROOT)

from oracle import rw_oracle as orc  # noqa: E402
from paper_2607_00488_b200 import workloads as wl  # noqa: E402

COUNT_SEEDS = {"cfg1_tiny_nsi": [0], "cfg2_mm_lowE": [21], "cfg3_nsi4": [31], "cfg4_dense": [41],
               "cfg5_joint6": [70 + d for d in range(8)]}


def derive(name):
    zero = np.zeros(orc.N_KINDS)
    out = {}
    line_ratio = None
    if name == "cfg1_tiny_nsi":
        raw1 = wl.raw_tables(name, line_ratio=1.0)
        cont = dict(raw1)
        cont["E"], cont["flux_w"], cont["P_e"] = raw1["E"][:-1], raw1["flux_w"][:-1], raw1["P_e"][:-1]
        line = dict(raw1)
        line["E"], line["flux_w"], line["P_e"] = raw1["E"][-1:], raw1["flux_w"][-1:], raw1["P_e"][-1:]
        Cc = orc.spectrum(cont, zero).sum()
        Ll = orc.spectrum(line, zero).sum()
        line_ratio = 0.3 * Cc / (0.7 * Ll)
        out["line_ratio"] = np.float64(line_ratio)
    raw = wl.raw_tables(name, line_ratio=line_ratio)
    S = orc.spectrum(raw, zero)
    S_hat = S / S.sum()
    out["S_hat"] = S_hat
    D, n_T, n_rec = raw["R"].shape
    counts = np.empty((D, n_rec), np.int32)
    ones = np.ones(n_T)
    for d in range(D):
        N_mc = raw["exposure"][d] * raw["N_tot"] * S_hat
        mu_sm = orc.fold(ones, N_mc, raw["R"][d], raw["bkg"][d])
        counts[d] = np.random.default_rng(COUNT_SEEDS[name][d]).poisson(mu_sm)
    out["counts"] = counts
    return out


def main():
    store = {}
    for name in wl.CONFIG_NAMES:
        t0 = time.time()
        d = derive(name)
        for k, v in d.items():
            store[name + "/" + k] = v
        print("%-14s S_hat[%d] counts%s sum=%d %s  (%.1f s)" % (
            name, d["S_hat"].size, d["counts"].shape, int(d["counts"].sum()),
            "line_ratio=%.15g" % d["line_ratio"] if "line_ratio" in d else "", time.time() - t0))
    path = os.path.join(_ROOT, "paper_2607_00488_b200", "workload_data", "derived_inputs.npz")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    np.savez_compressed(path, **store)
    h = hashlib.sha256(open(path, "rb").read()).hexdigest()
    print("wrote", path, os.path.getsize(path), "bytes sha256", h)


if __name__ == "__main__":
    main()
