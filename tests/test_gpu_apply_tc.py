"""-m gpu parity of the tensor-core stencil kernel (tcgen05, split TF32; csrc/stencil_tc.cuh) against the CPU oracle.

Same metric and tolerance as test_gpu_apply.py (complex64: <= 1e-5 relative per column, north_star); on the
diagonally dominant operators of BASELINE.json the measured error is asserted against a tighter 1e-6 as well, because
block CG to 1e-6 needs the apply to be that accurate.

Two properties of the tensor core shape the assertions:
 * x = hi + lo with hi rounded to TF32 and lo = x - hi cut to TF32 by the tensor core loses the last bits of x, and
   the FP32 accumulator adds with truncation: "exact" cases (pure shifts, multiplication by i) are exact to ONE
   float32 ulp per real component, not bit for bit (the SIMT kernels are bit exact, test_gpu_apply.py);
 * without a dominant diagonal (c = 0) the truncated accumulation is the leading error; the correction products have
   their own accumulators for every nrhs, which keeps it below the 1e-5 bar (measured ~6e-6).
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


def _apply_tc(dims, A, X, nrhs_max=None):
    s = X.shape[-1]
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), nrhs_max or s, flags=cm.binding.FLAG_TF32)    # nbasis 32 defaults to the FP16-split kernel
    name = op.kernel_name(s)
    assert name.startswith("stencil_tc"), name
    Y = to_np(op.apply(to_dev(X, "c64")))
    torch.cuda.synchronize()
    op.close()
    return Y


# lattices: x extent 3 (one pair + a single site), 4 (two pairs), 5 (2 + 2 + 1); wrap in every direction
@pytest.mark.parametrize("nb,s", [(32, 16), (32, 8), (32, 32), (32, 64), (32, 24), (32, 40), (24, 16), (24, 64), (16, 16), (8, 8), (8, 48)])
@pytest.mark.parametrize("dims", [(3, 3, 3, 5), (4, 4, 4, 6), (5, 2, 3, 3)])
def test_tensor_kernel_matches_oracle(nb, s, dims):
    A, c, X, _ = host_case(dims, nb, s, seed=200 + nb + s, factor=1.05)
    Y = _apply_tc(dims, A, X)
    err = rel_err_cols(Y, oracle.apply(dims, A, X))
    assert err <= TOL["c64"], err
    assert err <= 1e-6, err


@pytest.mark.parametrize("dims", [(1, 1, 1, 1), (2, 2, 2, 2), (1, 2, 3, 1), (9, 1, 2, 1), (6, 3, 1, 2)])
def test_tensor_kernel_small_extents_alias_and_add(dims):
    # extents 1 and 2: several stencil points address the same neighbour and must ADD
    A, c, X, _ = host_case(dims, 32, 16, seed=41, factor=1.1)
    Y = _apply_tc(dims, A, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= 1e-6


def test_tensor_kernel_without_diagonal_shift():
    dims = (3, 4, 3, 4)
    for nb, s, bar in [(32, 16, 1e-5), (32, 32, 1e-5), (32, 64, 1e-5), (24, 64, 1e-5)]:
        A, c, X, _ = host_case(dims, nb, s, seed=7, factor=0.0)
        assert c == 0.0
        Y = _apply_tc(dims, A, X)
        err = rel_err_cols(Y, oracle.apply(dims, A, X))
        assert err <= bar, (nb, s, err)


def _within_one_ulp(Y, ref):
    y, r = Y.view(np.float64), ref.view(np.float64)
    return bool(np.all(np.abs(y - r) <= 2.0 ** -23 * np.abs(r)))


def test_tensor_kernel_pure_shift_to_one_ulp():
    # A_p = delta_{p,p0} I  =>  Y(x) = X(x + delta_p0): every element is x_hi * 1 + x_lo * 1 (+ zeros), one float32 ulp
    dims, nb, s = (5, 4, 3, 2), 32, 16
    V = synth.volume(dims)
    X = synth.make_block(dims, nb, s, 5, synth.TAG_X)
    off = synth.stencil_offsets()
    for p0 in list(range(0, 81, 5)) + [39, 40, 41]:
        A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
        A[:, p0] = np.eye(nb, dtype=np.complex64)
        Y = _apply_tc(dims, A, X)
        assert _within_one_ulp(Y, shifted_block(dims, X, off[p0])), p0


@pytest.mark.parametrize("p_only", [0, 12, 13, 14, 39, 40, 41, 67, 80])
def test_tensor_kernel_one_point_at_a_time(p_only):
    dims, nb, s = (6, 3, 3, 4), 32, 16
    A, c, X, _ = host_case(dims, nb, s, seed=9, factor=0.0)
    A1 = np.zeros_like(A)
    A1[:, p_only] = A[:, p_only]
    Y = _apply_tc(dims, A1, X)
    assert rel_err_cols(Y, oracle.apply(dims, A, X, p_only=p_only)) <= 2e-6


def test_tensor_kernel_imaginary_unit_and_single_entries():
    # A_40 = i I  =>  Y = i X (checks the re/im panel combination and its signs);
    # a single nonzero entry A_40[i0][j0] = -2i moves row j0 of X to row i0; both to one float32 ulp
    dims, nb, s = (4, 2, 2, 2), 32, 16
    V = synth.volume(dims)
    X = synth.make_block(dims, nb, s, 11, synth.TAG_X)
    A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
    A[:, 40] = 1j * np.eye(nb, dtype=np.complex64)
    assert _within_one_ulp(_apply_tc(dims, A, X), 1j * X)
    A[:] = 0
    A[:, 40, 3, 17] = -2j
    ref = np.zeros_like(X)
    ref[:, 3, :] = -2j * X[:, 17, :]
    Y = _apply_tc(dims, A, X)
    assert np.array_equal(Y[:, :3], ref[:, :3]) and np.array_equal(Y[:, 4:], ref[:, 4:])      # exact zeros elsewhere
    assert _within_one_ulp(Y[:, 3], ref[:, 3])


def test_tensor_and_simt_kernels_agree():
    dims, nb, s = (4, 4, 4, 4), 32, 16
    A, c, X, _ = host_case(dims, nb, s, seed=3, factor=1.02)
    Yt = _apply_tc(dims, A, X)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), s, flags=cm.binding.FLAG_NO_TENSOR)
    assert op.kernel_name(s).startswith("stencil_simt")
    Ys = to_np(op.apply(to_dev(X, "c64")))
    op.close()
    ref = oracle.apply(dims, A, X)
    assert rel_err_cols(Yt, ref) <= 1e-6 and rel_err_cols(Ys, ref) <= 1e-6
    assert rel_err_cols(Yt, Ys) <= 2e-6


def test_tensor_only_operator_keeps_one_copy_and_rejects_uncovered_nrhs():
    # COARSE_FLAG_TENSOR_ONLY: only the tensor kernel's layout of A is kept; nrhs it does not cover -> UNSUPPORTED
    dims, nb, s = (4, 3, 3, 4), 24, 16
    A, c, X, _ = host_case(dims, nb, s, seed=17, factor=1.02)
    Ad, Xd = to_dev(A, "c64"), to_dev(X, "c64")
    outs, sizes = [], []
    for flags in (cm.binding.FLAG_TF32, cm.binding.FLAG_TF32 | cm.binding.FLAG_TENSOR_ONLY):
        op = cm.CoarseOperator(dims, Ad, s, flags=flags)
        assert op.kernel_name(s).startswith("stencil_tc")
        outs.append(to_np(op.apply(Xd)))
        sizes.append(op.device_bytes())
        if flags & cm.binding.FLAG_TENSOR_ONLY:
            with pytest.raises(cm.binding.CoarseError) as ei:
                op.apply(Xd[:, :, :4].contiguous())
            assert ei.value.status == cm.binding.UNSUPPORTED
        op.close()
    assert np.array_equal(outs[0], outs[1])
    assert sizes[0] - sizes[1] == Ad.numel() * 8
