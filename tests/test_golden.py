"""Stored expected values: the paper's printed numbers (arithmetic cross-checks only) and the
oracle's own config-0 error curve (regression fixture written by tests/golden/make_golden.py)."""
import os

import numpy as np

import oracle
from paper_1808_10375_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def paper_values():
    out = {}
    for line in open(os.path.join(GOLD, "paper_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def test_paper_size_and_speedup_identities():
    v = paper_values()
    nbytes = v["raw_data_views"] * v["raw_data_frame_edge"] ** 2 * v["raw_data_bytes_per_pixel"]
    assert abs(nbytes / 2 ** 30 - v["raw_data_gb"]) < 0.01                 # 2.63 "GB" is GiB of float64
    assert abs(v["time_1core_h"] * 3600 / v["time_4xV100_s"] - v["speedup_4xV100"]) < 5
    # BASELINE.md's derived iteration rates
    assert abs(v["iterations"] / v["time_4xV100_s"] - 1.95) < 0.01
    assert abs(v["iterations"] / v["time_2xV100_s"] - 1.00) < 0.01


def test_oracle_reproduces_stored_config0_curve():
    gold = np.loadtxt(os.path.join(GOLD, "c0_error_curve.txt"))
    assert gold.shape == (50, 4)
    pr = synth.make_problem(0)
    c = pr.cfg
    o = oracle.OracleDM(c.N, c.K, c.L, c.obj_h, c.obj_w, pr.positions)
    o.set_data(pr.intensities, pr.probe0, pr.object0)
    o.iterate(50)
    e = o.errors()
    # early rows are insensitive; later rows may move with libm / thread-independent rounding only
    assert np.abs(e[:10] - gold[:10]).max() < 1e-9
    assert np.abs(e - gold).max() < 1e-4
    # iteration 1 from psi = P0 O0 with beta = 1: eps_F == eps_psi (Parseval; A10)
    assert abs(gold[0, 0] - gold[0, 1]) < 1e-12
