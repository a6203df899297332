"""-m gpu: the device-side input generator (coarse_op_fill_synthetic / coarse_fill_block) reproduces the
host generator inputs/synth.py (same counter-based hash, implemented independently)."""
import numpy as np
import pytest
import torch

from inputs import synth

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


@pytest.mark.parametrize("dims,nb,dtype,factor", [((4, 4, 4, 4), 8, torch.complex128, 1.10), ((3, 2, 4, 5), 24, torch.complex64, 1.05),
                                                   ((4, 4, 4, 6), 32, torch.complex64, 0.0)])
def test_device_generator_equals_host_generator(dims, nb, dtype, factor):
    seed = 20240903
    A_h, c_h = synth.make_operator(dims, nb, seed, factor)
    A_d, c_d = cm.fill_synthetic(dims, nb, dtype, seed, factor)
    A_d = A_d.cpu().numpy().astype(np.complex64)
    assert abs(c_d - c_h) <= 1e-6 * abs(c_h)
    if c_d != c_h:                                     # compare without the shift if the last ulp of c differs
        d = np.arange(nb)
        A_d[:, 40, d, d] -= np.float32(c_d)
        A_h[:, 40, d, d] -= np.float32(c_h)
    mism = np.count_nonzero(A_d != A_h)
    assert mism <= max(2, 1e-6 * A_h.size), f"{mism} of {A_h.size} entries differ"
    assert np.max(np.abs(A_d - A_h)) <= 1e-6
    X_h = synth.make_block(dims, nb, 5, seed, synth.TAG_B)
    X_d = cm.fill_block(dims, nb, 5, dtype, seed, synth.TAG_B).cpu().numpy().astype(np.complex128)
    assert np.count_nonzero(X_d != X_h) <= 2 and np.max(np.abs(X_d - X_h)) <= 1e-6
