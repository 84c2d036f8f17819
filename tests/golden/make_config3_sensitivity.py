#!/usr/bin/env python
"""Writes tests/golden/config3_full_sensitivity.txt: how far the ORACLE's own result of BASELINE config 3 at full size
(192 x 128 x 128, WENO5, 100 steps) moves when its input is perturbed by 1 ulp (P0 (1 +- 2^-52), seeded signs) -- the L1
difference per primitive in the S23 metric (tests/parity_util.l1_diff).  Calls only oracle/ and the input generators.
The GPU test test_full_size_hundred_step_runs_l1[3] allows the CUDA path K_SENS = 10 times these numbers where they exceed the
flat 1e-8 bar (S23c).  ~10 minutes on 8 cores.

    python tests/golden/make_config3_sensitivity.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import kharm_inputs as ki                      # noqa: E402
from kharm_inputs import torus                 # noqa: E402
from oracle import kho                         # noqa: E402
from parity_util import l1_diff                # noqa: E402


def run(p, P):
    g = kho.Grid(p, omp=True)
    g.set_prims(P)
    dt = g.estimate_dt()
    for _ in range(100):
        dt = g.step(dt)
    return g.get_prims()


def main():
    p = ki.config_params(3)
    P0 = torus.torus_state(p, seed=1)
    ref = run(p, P0)
    rng = np.random.default_rng(100)
    l1 = l1_diff(p, run(p, P0 * (1.0 + 2.0 ** -52 * rng.choice([-1.0, 1.0], size=P0.shape))), ref)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config3_full_sensitivity.txt")
    with open(out, "w") as f:
        f.write("# BASELINE config 3 (192x128x128, WENO5, seed 1), 100 steps: L1 difference per primitive (S23 metric) between the oracle's\n"
                "# result from P0 and from P0 (1 +- 2^-52) (numpy default_rng(100) signs).  Written by tests/golden/make_config3_sensitivity.py\n"
                "# (oracle only).  Order: rho u ut1 ut2 ut3 B1 B2 B3\n")
        f.write(" ".join("%.6e" % v for v in l1) + "\n")
    print(l1)


if __name__ == "__main__":
    main()
