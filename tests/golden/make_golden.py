#!/usr/bin/env python
"""Writes tests/golden/oracle_regression.txt -- values computed by the FP64 oracle ONLY (oracle/ + the seeded
input generators of workloads.py; nothing here touches the CUDA path).  They freeze the oracle's arithmetic:
tests/test_golden.py re-runs the oracle against them, so a later change to the oracle's formulas shows up as a
diff of this file and has to name the PAPER.md passage / DESIGN.md reading that justifies it.

    python tests/golden/make_golden.py

Contents: (1) the isolated-node state after 2 s without noise (G = 0) for b_e = 0, 60, 120 pA -- the rates the
paper's Eqs. (1)-(3) settle to under the readings of DESIGN.md section 3; (2) the state of three
regions of the cfg-1 sweep (BASELINE.json configs[0]) at step 1,000, noise off and noise on (Philox seed 1).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402
from oracle import oracle as orc  # noqa: E402

NAMES = ("E", "I", "C_ee", "C_ei", "C_ii", "W_e", "W_i")


def rows():
    out = []
    # (1) isolated node: 2 regions, no coupling weight at all
    W = np.zeros((2, 2)); L = np.zeros((2, 2))
    for b_e in (0.0, 60.0, 120.0):
        P = wl.param_vector(G=0.0, b_e=b_e)[None, :]
        o = orc.OracleSweep(W, L, P, seed=0)
        o.run(20000, 0.1, noise_on=False, ds=0)
        y = o.state(0)[0]
        for q, nm in enumerate(NAMES):
            out.append((f"node b_e={b_e:g} step=20000 {nm}", y[q][0]))
    # (2) cfg 1
    cfg = wl.config(1)
    Wc, Lc = wl.config_connectome(cfg)
    P = wl.grid_params(cfg)
    for noise in (0, 1):
        o = orc.OracleSweep(Wc, Lc, P, seed=cfg["seed"])
        o.run(1000, cfg["dt"], noise_on=bool(noise), ds=10)
        for s in (0, 7):
            y, ou = o.state(s)
            for k in (0, 33, 67):
                for q, nm in enumerate(NAMES):
                    out.append((f"cfg1 noise={noise} sim={s} region={k} step=1000 {nm}", y[q][k]))
                if noise:
                    out.append((f"cfg1 noise={noise} sim={s} region={k} step=1000 OU", ou[k]))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only (FP64); key : value (17 significant digits)\n")
        for k, v in rows():
            f.write(f"{k} : {float(v):.17e}\n")
    print("wrote", path)
