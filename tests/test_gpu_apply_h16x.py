"""-m gpu parity of the split-FP16 tensor-core stencil kernel that holds the X operand in tensor memory
(csrc/stencil_h16x.cuh: tcgen05 kind::f16 with the M-side operand from TMEM, loader warps + tcgen05.st, groups of up to 4 x-adjacent
sites, one MMA-issuing warp per site) against the CPU oracle.  Default kernel for complex64 with nbasis 8, 16, 24 (any nrhs
>= 4); nbasis 32 with COARSE_FLAG_H16X, or above nrhs 48 with COARSE_FLAG_H16X_WIDE.

Metric and tolerance as in test_gpu_apply.py (complex64: <= 1e-5 relative per column, north_star); on the diagonally
dominant operators of BASELINE.json a tighter 1e-6 is asserted as well (block CG to 1e-6 needs it).  The numbers are those
of stencil_h16.cuh (hi + 2^-11 lo in binary16 after power-of-two scalings), so the same "exact to 2^-21" bars apply.

Lattice shapes exercise every group size: x extent 1..4 = one group of G = 1..4 sites, 5 = 4 + 1, 6 = 4 + 2, 7 = 4 + 3,
9 = 4 + 4 + 1 (nbasis 32: groups of up to 3); extents 1-2 make several stencil points alias one neighbour.
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


def _apply_x(dims, A, X, nrhs_max=None, extra_flags=0):
    s, nb = X.shape[-1], A.shape[-1]
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), nrhs_max or s, flags=(cm.binding.FLAG_H16X if nb == 32 else 0) | extra_flags)
    name = op.kernel_name(s)
    assert name.startswith("stencil_h16x"), name
    Y = to_np(op.apply(to_dev(X, "c64")))
    torch.cuda.synchronize()
    op.close()
    return Y


@pytest.mark.parametrize("s", [4, 8, 16, 24, 40, 64])
@pytest.mark.parametrize("nb", [8, 16, 24, 32])
@pytest.mark.parametrize("dims", [(3, 3, 3, 5), (4, 4, 4, 6), (5, 2, 3, 3), (7, 3, 2, 2)])
def test_h16x_kernel_matches_oracle(s, nb, dims):
    A, c, X, _ = host_case(dims, nb, s, seed=500 + s + nb, factor=1.05)
    Y = _apply_x(dims, A, X)
    err = rel_err_cols(Y, oracle.apply(dims, A, X))
    assert err <= TOL["c64"], err
    assert err <= 1e-6, err


@pytest.mark.parametrize("nb,s", [(24, 5), (24, 13), (16, 7), (8, 33), (32, 63), (24, 64)])
def test_h16x_kernel_any_nrhs_on_a_wider_handle(nb, s):
    # nrhs need not be a multiple of 8; the handle was created for a wider block (scratch tiles keep stale rows of the wider use)
    dims = (6, 3, 2, 3)
    A, c, X, _ = host_case(dims, nb, s, seed=91, factor=1.05)
    A2, _, X2, _ = host_case(dims, nb, 64, seed=92, factor=1.05)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), 64, flags=(cm.binding.FLAG_H16X if nb == 32 else 0) | cm.binding.FLAG_TENSOR_ONLY)
    assert op.kernel_name(s).startswith("stencil_h16x") and op.kernel_name(64).startswith("stencil_h16x")
    op.apply(to_dev(X2, "c64"))                                   # a wide apply first
    Y = to_np(op.apply(to_dev(X, "c64")))
    op.close()
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


@pytest.mark.parametrize("nb,s", [(24, 64), (24, 16), (32, 64), (16, 32)])
def test_h16x_kernel_many_groups_per_cta(nb, s):
    # 1728 sites: several groups per CTA on 148 SMs (rings wrap, accumulator slots and X buffers are reused many times)
    dims = (8, 6, 6, 6)
    A, c, X, _ = host_case(dims, nb, s, seed=77, factor=1.02)
    Y = _apply_x(dims, A, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


@pytest.mark.parametrize("nb", [24, 32])
@pytest.mark.parametrize("dims", [(1, 1, 1, 1), (2, 2, 2, 2), (1, 2, 3, 1), (9, 1, 2, 1), (6, 3, 1, 2), (3, 1, 1, 4)])
def test_h16x_kernel_small_extents_alias_and_add(dims, nb):
    # extents 1 and 2: several stencil points address the same neighbour and must ADD
    A, c, X, _ = host_case(dims, nb, 16, seed=41, factor=1.1)
    Y = _apply_x(dims, A, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


def test_h16x_kernel_without_diagonal_shift():
    # c = 0: nothing dominates the sum, the error is that of the split itself and of the FP32 accumulator
    dims = (3, 4, 3, 4)
    for nb, s in ((24, 16), (24, 64), (32, 64), (8, 8)):
        A, c, X, _ = host_case(dims, nb, s, seed=7, factor=0.0)
        assert c == 0.0
        err = rel_err_cols(_apply_x(dims, A, X), oracle.apply(dims, A, X))
        assert err <= 1e-5, (nb, s, err)


def _close(Y, ref, rel):
    y, r = Y.view(np.float64), ref.view(np.float64)
    return bool(np.all(np.abs(y - r) <= rel * np.abs(r)))


def test_h16x_kernel_pure_shift():
    # A_p = delta_{p,p0} I  =>  Y(x) = X(x + delta_p0): each element is (x_hi + 2^-11 x_lo) * 1, i.e. x to 2^-22.
    # x extent 7 = a group of 4 and a group of 3: every (group size, site slot, dx) combination of the schedule is hit
    dims, s, nb = (7, 4, 3, 2), 16, 24
    V = synth.volume(dims)
    X = synth.make_block(dims, nb, s, 5, synth.TAG_X)
    off = synth.stencil_offsets()
    for p0 in list(range(0, 81, 5)) + [39, 40, 41]:
        A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
        A[:, p0] = np.eye(nb, dtype=np.complex64)
        Y = _apply_x(dims, A, X)
        assert _close(Y, shifted_block(dims, X, off[p0]), 2.0 ** -21), p0


@pytest.mark.parametrize("p_only", [0, 12, 13, 14, 39, 40, 41, 67, 80])
def test_h16x_kernel_one_point_at_a_time(p_only):
    dims, s, nb = (6, 3, 3, 4), 16, 24
    A, c, X, _ = host_case(dims, nb, s, seed=9, factor=0.0)
    A1 = np.zeros_like(A)
    A1[:, p_only] = A[:, p_only]
    Y = _apply_x(dims, A1, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X, p_only=p_only)) <= 2e-6


def test_h16x_kernel_imaginary_unit_and_single_entries():
    # A_40 = i I  =>  Y = i X (the re/im combination and its signs); a single entry A_40[i0][j0] = -2i moves row j0 to row i0
    dims, s, nb = (4, 2, 2, 2), 16, 24
    V = synth.volume(dims)
    X = synth.make_block(dims, nb, s, 11, synth.TAG_X)
    A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
    A[:, 40] = 1j * np.eye(nb, dtype=np.complex64)
    assert _close(_apply_x(dims, A, X), 1j * X, 2.0 ** -21)
    A[:] = 0
    A[:, 40, 3, 17] = -2j
    ref = np.zeros_like(X)
    ref[:, 3, :] = -2j * X[:, 17, :]
    Y = _apply_x(dims, A, X)
    assert np.array_equal(Y[:, :3], ref[:, :3]) and np.array_equal(Y[:, 4:], ref[:, 4:])      # exact zeros elsewhere
    assert _close(Y[:, 3], ref[:, 3], 2.0 ** -21)


def test_h16x_column_scales_cover_the_float32_range():
    # columns of norm 1e-18 ... 1e+18 side by side and one all-zero column: every column keeps its own relative accuracy
    dims, s, nb = (4, 3, 3, 4), 16, 24
    A, c, X, _ = host_case(dims, nb, s, seed=21, factor=1.05)
    scales = np.array([10.0 ** e for e in (-18, -12, -7, -3, 0, 0, 2, 5, 9, 14, 18, -18, 18, 1, -1, 0)])
    Xs = (X * scales).astype(np.complex64).astype(np.complex128)
    Xs[:, :, 5] = 0.0
    Y = _apply_x(dims, A, Xs)
    ref = oracle.apply(dims, A, Xs)
    assert np.all(Y[:, :, 5] == 0.0)
    keep = [r for r in range(s) if r != 5]
    assert rel_err_cols(Y[:, :, keep], ref[:, :, keep]) <= 1e-6


@pytest.mark.parametrize("exp10", [-20, -6, 6, 20])
def test_h16x_operator_scale_covers_the_float32_range(exp10):
    dims, s, nb = (4, 3, 3, 4), 16, 24
    A, c, X, _ = host_case(dims, nb, s, seed=22, factor=1.05)
    As = (A.astype(np.complex128) * 10.0 ** exp10).astype(np.complex64)
    Y = _apply_x(dims, As, X)
    assert rel_err_cols(Y, oracle.apply(dims, As, X)) <= 1e-6


def test_h16x_and_tf32_and_simt_and_paired_kernels_agree():
    dims, s = (4, 4, 4, 4), 16
    for nb in (24, 32):
        A, c, X, _ = host_case(dims, nb, s, seed=3, factor=1.02)
        ref = oracle.apply(dims, A, X)
        variants = [("stencil_h16x", cm.binding.FLAG_H16X if nb == 32 else 0), ("stencil_tc", cm.binding.FLAG_TF32),
                    ("stencil_", cm.binding.FLAG_NO_TENSOR)]
        if nb == 32:
            variants.append(("stencil_h16<", 0))
        outs = {}
        for name, flags in variants:
            op = cm.CoarseOperator(dims, to_dev(A, "c64"), s, flags=flags)
            assert op.kernel_name(s).startswith(name), op.kernel_name(s)
            outs[name] = to_np(op.apply(to_dev(X, "c64")))
            op.close()
            assert rel_err_cols(outs[name], ref) <= 1e-6
        assert rel_err_cols(outs["stencil_h16x"], outs["stencil_"]) <= 2e-6


def test_h16x_repeated_applies_are_bit_identical():
    # every accumulator has one issuing thread and a fixed order of stencil points: the result does not depend on timing
    dims, s, nb = (8, 6, 6, 6), 64, 24
    A, c, X, _ = host_case(dims, nb, s, seed=13, factor=1.02)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), s)
    Xd = to_dev(X, "c64")
    Y0 = op.apply(Xd).clone()
    for _ in range(5):
        assert torch.equal(op.apply(Xd), Y0)
    op.close()


def test_h16x_wide_flag_keeps_both_layouts_and_splits_the_widths():
    # COARSE_FLAG_H16X_WIDE (nbasis 32, nrhs_max > 48): stencil_h16 serves nrhs <= 48, stencil_h16x the wider blocks; the two
    # kernels share the scratch block of split X tiles in their own formats, so alternate the widths
    dims, nb = (6, 3, 3, 4), 32
    A, c = synth.make_operator(dims, nb, 61, 1.05)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), 64, flags=cm.binding.FLAG_H16X_WIDE)
    assert op.kernel_name(64).startswith("stencil_h16x<") and op.kernel_name(56).startswith("stencil_h16x<")
    assert op.kernel_name(48).startswith("stencil_h16<") and op.kernel_name(16).startswith("stencil_h16<")
    for s in (64, 16, 24, 56, 8, 64, 48):
        X = synth.make_block(dims, nb, s, 61 + s, synth.TAG_X)
        Y = to_np(op.apply(to_dev(X, "c64")))
        assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6, s
    op.close()
    # without wide blocks on the handle the flag changes nothing
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), 32, flags=cm.binding.FLAG_H16X_WIDE)
    assert op.kernel_name(32).startswith("stencil_h16<")
    op.close()
