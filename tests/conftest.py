import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg1():
    """BASELINE.json configs[0]: 4^4, nbasis 8, Nrhs 4, complex128 (values float32-exact)."""
    from inputs import synth
    cfg = synth.config(0)
    A, c = synth.make_operator(cfg["dims"], cfg["nbasis"], cfg["seed"], cfg["factor"])
    cfg["A"], cfg["c"] = A.astype(np.complex128), c
    cfg["X"] = synth.make_block(cfg["dims"], cfg["nbasis"], cfg["nrhs"], cfg["seed"], synth.TAG_X)
    cfg["B"] = synth.make_block(cfg["dims"], cfg["nbasis"], cfg["nrhs"], cfg["seed"], synth.TAG_B)
    return cfg


@pytest.fixture(scope="session")
def cfg1_dense(cfg1):
    from helpers import dense_matrix
    return dense_matrix(cfg1["dims"], cfg1["A"])
