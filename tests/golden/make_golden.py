"""Writes tests/golden/cfg1_oracle.txt from the ORACLE ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden.py
Stored values: BlockCGrQ residual history and a few entries of Y = H X for BASELINE.json configs[0]
(4^4 lattice, nbasis 8, Nrhs 4, complex128, seed 20240903), as a regression guard on the oracle and a
human-readable record of what "7 iterations to 1e-10" looks like.  The paper prints no worked example
for this path (PAPER.md has only Table 6 throughputs), so there is no paper-value fixture.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from inputs import synth          # noqa: E402
from oracle import oracle         # noqa: E402


def main():
    cfg = synth.config(0)
    A, c = synth.make_operator(cfg["dims"], cfg["nbasis"], cfg["seed"], cfg["factor"])
    X = synth.make_block(cfg["dims"], cfg["nbasis"], cfg["nrhs"], cfg["seed"], synth.TAG_X)
    B = synth.make_block(cfg["dims"], cfg["nbasis"], cfg["nrhs"], cfg["seed"], synth.TAG_B)
    Y = oracle.apply(cfg["dims"], A, X)
    res = oracle.block_cg(cfg["dims"], A, B, tol=cfg["tol"], maxiter=100)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; BASELINE.json configs[0], seed %d\n" % cfg["seed"])
        f.write("c %.17g\n" % c)
        f.write("iterations %d\n" % res["iterations"])
        for k, row in enumerate(res["history"]):
            f.write("history %d %s\n" % (k, " ".join("%.17g" % v for v in row)))
        for (x, i, r) in [(0, 0, 0), (1, 3, 2), (100, 7, 3), (255, 5, 1)]:
            f.write("Y %d %d %d %.17g %.17g\n" % (x, i, r, Y[x, i, r].real, Y[x, i, r].imag))
    print("wrote", out)


if __name__ == "__main__":
    main()
