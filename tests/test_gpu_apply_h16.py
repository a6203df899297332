"""-m gpu parity of the FP16-split tensor-core stencil kernel (tcgen05 kind::f16, 3 products; csrc/stencil_h16.cuh)
against the CPU oracle.  Default kernel for complex64, nbasis 32, nrhs a multiple of 8 (or 4).

Metric and tolerance as in test_gpu_apply.py (complex64: <= 1e-5 relative per column, north_star); on the diagonally
dominant operators of BASELINE.json a tighter 1e-6 is asserted as well (block CG to 1e-6 needs it).

What is specific to this kernel:
 * every real number is carried as hi + 2^-11 lo with hi, lo binary16 after a power-of-two scaling (one scale per
   operator, one per right-hand-side column): 22-23 significant bits, so "exact" cases hold to ~2^-22 relative, not
   bit for bit (the SIMT kernels are bit exact, test_gpu_apply.py);
 * the scales must make the result independent of the magnitude of the operator and of each column: tested over
   40 orders of magnitude, with columns of very different norms side by side and with an all-zero column.
"""
import numpy as np
import pytest
import torch

from gpu_common import TOL, host_case, to_dev, to_np
from helpers import rel_err_cols, shifted_block
from inputs import synth
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _apply_h16(dims, A, X, nrhs_max=None):
    s = X.shape[-1]
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), nrhs_max or s)
    name = op.kernel_name(s)
    assert name.startswith("stencil_h16"), name
    Y = to_np(op.apply(to_dev(X, "c64")))
    torch.cuda.synchronize()
    op.close()
    return Y


# lattices: x extent 3 (one pair + a single site), 4 (two pairs), 5 (2 + 2 + 1); wrap in every direction;
# (8, 6, 6, 6): 864 pairs of sites = several pairs per CTA on 148 SMs x 2 CTAs (rings wrap, accumulators are reused)
@pytest.mark.parametrize("s", [4, 8, 16, 24, 32, 40, 48, 56, 64])
@pytest.mark.parametrize("dims", [(3, 3, 3, 5), (4, 4, 4, 6), (5, 2, 3, 3)])
def test_h16_kernel_matches_oracle(s, dims):
    A, c, X, _ = host_case(dims, 32, s, seed=300 + s, factor=1.05)
    Y = _apply_h16(dims, A, X)
    err = rel_err_cols(Y, oracle.apply(dims, A, X))
    assert err <= TOL["c64"], err
    assert err <= 1e-6, err


@pytest.mark.parametrize("s", [16, 64])
def test_h16_kernel_many_groups_per_cta(s):
    dims = (8, 6, 6, 6)
    A, c, X, _ = host_case(dims, 32, s, seed=77, factor=1.02)
    Y = _apply_h16(dims, A, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


@pytest.mark.parametrize("dims", [(1, 1, 1, 1), (2, 2, 2, 2), (1, 2, 3, 1), (9, 1, 2, 1), (6, 3, 1, 2)])
def test_h16_kernel_small_extents_alias_and_add(dims):
    # extents 1 and 2: several stencil points address the same neighbour and must ADD
    A, c, X, _ = host_case(dims, 32, 16, seed=41, factor=1.1)
    Y = _apply_h16(dims, A, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


def test_h16_kernel_without_diagonal_shift():
    # c = 0: nothing dominates the sum, the error is that of the split itself and of the FP32 accumulator
    dims = (3, 4, 3, 4)
    for s in (16, 32, 64):
        A, c, X, _ = host_case(dims, 32, s, seed=7, factor=0.0)
        assert c == 0.0
        err = rel_err_cols(_apply_h16(dims, A, X), oracle.apply(dims, A, X))
        assert err <= 1e-5, (s, err)


def _close(Y, ref, rel):
    y, r = Y.view(np.float64), ref.view(np.float64)
    return bool(np.all(np.abs(y - r) <= rel * np.abs(r)))


def test_h16_kernel_pure_shift():
    # A_p = delta_{p,p0} I  =>  Y(x) = X(x + delta_p0): each element is (x_hi + 2^-11 x_lo) * 1, i.e. x to 2^-22
    dims, s = (5, 4, 3, 2), 16
    V = synth.volume(dims)
    X = synth.make_block(dims, 32, s, 5, synth.TAG_X)
    off = synth.stencil_offsets()
    for p0 in list(range(0, 81, 5)) + [39, 40, 41]:
        A = np.zeros((V, 81, 32, 32), dtype=np.complex64)
        A[:, p0] = np.eye(32, dtype=np.complex64)
        Y = _apply_h16(dims, A, X)
        assert _close(Y, shifted_block(dims, X, off[p0]), 2.0 ** -21), p0


@pytest.mark.parametrize("p_only", [0, 12, 13, 14, 39, 40, 41, 67, 80])
def test_h16_kernel_one_point_at_a_time(p_only):
    dims, s = (6, 3, 3, 4), 16
    A, c, X, _ = host_case(dims, 32, s, seed=9, factor=0.0)
    A1 = np.zeros_like(A)
    A1[:, p_only] = A[:, p_only]
    Y = _apply_h16(dims, A1, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X, p_only=p_only)) <= 2e-6


def test_h16_kernel_imaginary_unit_and_single_entries():
    # A_40 = i I  =>  Y = i X (the re/im combination and its signs); a single entry A_40[i0][j0] = -2i moves row j0 to row i0
    dims, s = (4, 2, 2, 2), 16
    V = synth.volume(dims)
    X = synth.make_block(dims, 32, s, 11, synth.TAG_X)
    A = np.zeros((V, 81, 32, 32), dtype=np.complex64)
    A[:, 40] = 1j * np.eye(32, dtype=np.complex64)
    assert _close(_apply_h16(dims, A, X), 1j * X, 2.0 ** -21)
    A[:] = 0
    A[:, 40, 3, 17] = -2j
    ref = np.zeros_like(X)
    ref[:, 3, :] = -2j * X[:, 17, :]
    Y = _apply_h16(dims, A, X)
    assert np.array_equal(Y[:, :3], ref[:, :3]) and np.array_equal(Y[:, 4:], ref[:, 4:])      # exact zeros elsewhere
    assert _close(Y[:, 3], ref[:, 3], 2.0 ** -21)


def test_h16_column_scales_cover_the_float32_range():
    # columns of norm 1e-18 ... 1e+18 side by side and one all-zero column: every column keeps its own relative accuracy
    dims, s = (4, 3, 3, 4), 16
    A, c, X, _ = host_case(dims, 32, s, seed=21, factor=1.05)
    scales = np.array([10.0 ** e for e in (-18, -12, -7, -3, 0, 0, 2, 5, 9, 14, 18, -18, 18, 1, -1, 0)])
    Xs = (X * scales).astype(np.complex64).astype(np.complex128)
    Xs[:, :, 5] = 0.0
    Y = _apply_h16(dims, A, Xs)
    ref = oracle.apply(dims, A, Xs)
    assert np.all(Y[:, :, 5] == 0.0)
    keep = [r for r in range(s) if r != 5]
    assert rel_err_cols(Y[:, :, keep], ref[:, :, keep]) <= 1e-6


@pytest.mark.parametrize("exp10", [-20, -6, 6, 20])
def test_h16_operator_scale_covers_the_float32_range(exp10):
    dims, s = (4, 3, 3, 4), 16
    A, c, X, _ = host_case(dims, 32, s, seed=22, factor=1.05)
    As = (A.astype(np.complex128) * 10.0 ** exp10).astype(np.complex64)
    Y = _apply_h16(dims, As, X)
    assert rel_err_cols(Y, oracle.apply(dims, As, X)) <= 1e-6


def test_h16_and_tf32_and_simt_kernels_agree():
    dims, s = (4, 4, 4, 4), 16
    A, c, X, _ = host_case(dims, 32, s, seed=3, factor=1.02)
    ref = oracle.apply(dims, A, X)
    outs = {}
    for name, flags in [("stencil_h16", 0), ("stencil_tc", cm.binding.FLAG_TF32), ("stencil_simt", cm.binding.FLAG_NO_TENSOR)]:
        op = cm.CoarseOperator(dims, to_dev(A, "c64"), s, flags=flags)
        assert op.kernel_name(s).startswith(name), op.kernel_name(s)
        outs[name] = to_np(op.apply(to_dev(X, "c64")))
        op.close()
        assert rel_err_cols(outs[name], ref) <= 1e-6
    assert rel_err_cols(outs["stencil_h16"], outs["stencil_simt"]) <= 2e-6


def test_h16_nrhs_not_covered_falls_back_to_simt_kernels():
    dims = (4, 3, 3, 4)
    A, c, X, _ = host_case(dims, 32, 12, seed=5, factor=1.02)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), 16)
    assert op.kernel_name(16).startswith("stencil_h16") and not op.kernel_name(12).startswith("stencil_h16")
    Y = to_np(op.apply(to_dev(X, "c64")))
    op.close()
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6
