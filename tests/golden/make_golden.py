"""Writes tests/golden/config1_oracle.txt from the fp64 oracle ALONE (no CUDA path involved).

The paper (arXiv 2011.04332) prints no numeric value of its solid solver, so
there is nothing of the paper's to store; this fixture freezes the oracle's own result for
BASELINE.json config 1 (one 162-vertex RBC, 1 step x 10 iterations, N(0,(1 pN)^2) forces, seed 0)
so that a later change to the oracle's arithmetic shows up as a diff against a committed file.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import workloads as W                      # noqa: E402  (input generators only)
from oracle import npfem_oracle as O      # noqa: E402


def compute():
    w = W.make_config(1)
    g = w.groups[0]
    oc = O.OracleCell(g.tris, g.rest, g.material, w.dt)
    pos, vel = oc.step(g.pos0, g.vel0, w.forces(0, 0), w.n_iters)
    disp = pos[0] - g.pos0[0].astype(np.float64)
    return disp, vel[0]


if __name__ == "__main__":
    disp, vel = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config1_oracle.txt")
    with open(path, "w") as fh:
        fh.write("# oracle (fp64) result of BASELINE.json config 1: per-vertex displacement x1 - x0 [um] and\n"
                 "# velocity [um/us] after 1 step x 10 iterations; written by tests/golden/make_golden.py\n"
                 "# (calls only oracle/ and the input generators).  The paper prints no value to cite.\n")
        for d, v in zip(disp, vel):
            fh.write(" ".join(f"{x:.17e}" for x in list(d) + list(v)) + "\n")
    print("wrote", path, disp.shape)
