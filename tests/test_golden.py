"""Fixtures under tests/golden/: (1) the config-0 anchors SURVEY.md 8(c) records from an independent
scratch implementation, (2) a regression lock on the oracle's own config-0 output."""
import os
import subprocess
import sys

import numpy as np

from oracle import kvarn_oracle as O
from paper_2606_03458_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
GOLD = os.path.join(HERE, "golden")


def _kv(path):
    d = {}
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, v = line.split("=", 1)
        d[k.strip()] = v.split("[")[0].strip()
    return d


def test_survey_config0_anchors():
    g = _kv(os.path.join(GOLD, "survey_config0_anchors.txt"))
    K, V, q, oc = W.config0()
    assert oc.tolist() == [int(x) for x in g["outlier_channels"].split()]
    assert abs(float(K[0, 0]) - float(g["K00"])) < 1e-7
    assert abs(float(V[0, 0]) - float(g["V00"])) < 1e-7
    assert abs(float(q[0]) - float(g["q0"])) < 1e-8
    rk = O.quantize_tile(K.astype(np.float64), "k")
    rv = O.quantize_tile(V.astype(np.float64), "v")
    traj = [float(x) for x in g["K_imbalance_trajectory"].split()]
    assert np.allclose(rk.varn.I[:len(traj)], traj, rtol=5e-5)
    vt = [float(x) for x in g["V_imbalance_trajectory"].split()]
    got = list(rv.varn.I[:3]) + [rv.varn.I[-1]]
    assert np.allclose(got, vt, atol=1.5e-4)
    lo, hi = (float(x) for x in g["K_S_tok_range"].split())
    assert np.isclose(rk.varn.S_c.min(), lo, rtol=1e-3) and np.isclose(rk.varn.S_c.max(), hi, rtol=1e-3)
    lo, hi = (float(x) for x in g["K_S_ch_range"].split())
    assert np.isclose(rk.varn.S_r.min(), lo, rtol=1e-3) and np.isclose(rk.varn.S_r.max(), hi, rtol=1e-3)


def test_oracle_regression_lock_config0():
    # the committed file must be exactly what the committed script writes from oracle/ today
    sys.path.insert(0, GOLD)
    try:
        import make_config0_regression as M
    finally:
        sys.path.pop(0)
    want = [l.rstrip("\n") for l in open(os.path.join(GOLD, "config0_oracle_regression.txt")) if not l.startswith("#")]
    assert M.lines() == want


def test_golden_script_uses_only_the_oracle():
    txt = open(os.path.join(GOLD, "make_config0_regression.py")).read()
    imports = [l.strip() for l in txt.splitlines() if l.strip().startswith(("import ", "from "))]
    assert all(("workloads" in l) or ("oracle" in l) or l.split()[1].split(".")[0] in ("os", "sys", "zlib", "numpy")
               for l in imports), imports
