"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ and the input
generators -- never the CUDA path.

  python tests/golden/make_golden.py

  c0_error_curve.txt : 50 rows [eps_F, eps_psi, eps_P1, eps_O1] of the FP64 oracle on config 0
                       (BASELINE.json configs[0]; defaults beta=1, a_O=a_P=1e-3, eps_F=1e-30).
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from paper_1808_10375_b200 import synth  # noqa: E402


def main():
    pr = synth.make_problem(0)
    c = pr.cfg
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    o.iterate(c.n_iter)
    hdr = ("FP64 oracle (oracle/dm_oracle.c) on BASELINE.json configs[0], seed 0, 50 iterations.\n"
           "columns: eps_F eps_psi eps_P[0] eps_O[0]  (DESIGN.md A10; eq. (7) PAPER.md:63-66)\n"
           "written by tests/golden/make_golden.py")
    np.savetxt(os.path.join(HERE, "c0_error_curve.txt"), o.errors(), fmt="%.17e", header=hdr)


if __name__ == "__main__":
    main()
