"""Regression guard: the oracle still reproduces the values it wrote to tests/golden/cfg1_oracle.txt."""
import os

import numpy as np

from oracle import oracle


def test_oracle_reproduces_golden(cfg1):
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    Y = oracle.apply(cfg1["dims"], cfg1["A"], cfg1["X"])
    res = oracle.block_cg(cfg1["dims"], cfg1["A"], cfg1["B"], tol=cfg1["tol"], maxiter=100)
    for row in rows:
        if row[0] == "c":
            assert float(row[1]) == cfg1["c"]
        elif row[0] == "iterations":
            assert int(row[1]) == res["iterations"]
        elif row[0] == "history":
            k = int(row[1])
            assert np.allclose(res["history"][k], [float(v) for v in row[2:]], rtol=1e-6)
        elif row[0] == "Y":
            x, i, r = int(row[1]), int(row[2]), int(row[3])
            assert abs(Y[x, i, r] - complex(float(row[4]), float(row[5]))) <= 1e-12 * abs(Y[x, i, r])
