"""-m gpu parity of the block-CG linear algebra on the tensor cores (csrc/blockla_tc.cuh: split-FP16 tcgen05 Gram product
G = U^H W and rotation out = beta Vin + U K for complex64 blocks; Table 6 "ThinQR") against the CPU oracle.

Widths >= 40 take this path by default; COARSE_FLAG_TENSOR_LINALG selects it for widths 16 to 32 as well.  Bars: the Gram
tolerance of test_gpu_blockcg.py (|G_gpu - G_or|_ab <= 2e-6 ||u_a|| ||w_b||, reading R11) and the apply metric (<= 1e-6 per
column here) for rotations.  What is specific to these kernels:
 * one power-of-two scale per 64-row tile (rotation) / per CTA with re-scaling (Gram): blocks whose magnitude varies by many
   orders of magnitude along the ROWS (a point source) and along the COLUMNS must keep their norm-wise accuracy;
 * the Gram kernel keeps FP32 sums in tensor memory for at most 256 rows and flushes them to float64 (measured: runs of 1024 rows put a bias of 3.7e-6 on the diagonal): more rows than that
   per CTA are covered at n = 400 000;
 * a rotation may write onto its own input (D = Q + D S^H).
"""
import numpy as np
import pytest
import torch

from gpu_common import to_dev, to_np
from helpers import rel_err_cols
from inputs import synth
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402

WIDTHS = [16, 24, 32, 40, 48, 56, 64]


def _op(s, flags=0):
    A = torch.zeros((1, 81, 4, 4), dtype=torch.complex64, device="cuda")
    return cm.CoarseOperator((1, 1, 1, 1), A, s, flags=flags | cm.binding.FLAG_TENSOR_LINALG)


def _rand_block(rng, n, s):
    z = (rng.standard_normal((n, s)) + 1j * rng.standard_normal((n, s))) / np.sqrt(2)
    return z.astype(np.complex64).astype(np.complex128)      # float32-exact


def _gram_err(G, U, W):
    un, wn = np.linalg.norm(U, axis=0), np.linalg.norm(W, axis=0)
    return float(np.max(np.abs(G - oracle.gram(U, W)) / np.outer(un, wn)))


@pytest.mark.parametrize("s", WIDTHS)
@pytest.mark.parametrize("n", [1, 63, 64, 65, 1000, 20011])
def test_tensor_gram_matches_oracle(n, s):
    rng = np.random.default_rng(n + 7 * s)
    U, W = _rand_block(rng, n, s), _rand_block(rng, n, s)
    op = _op(s)
    G = to_np(op.gram(to_dev(U, "c64"), to_dev(W, "c64")))
    Gu = to_np(op.gram(to_dev(U, "c64"), to_dev(U, "c64")))
    op.close()
    assert _gram_err(G, U, W) <= 2e-6
    assert _gram_err(Gu, U, U) <= 2e-6
    assert np.allclose(Gu, Gu.conj().T, atol=2e-6 * np.max(np.abs(Gu)))


def test_tensor_gram_long_runs_are_flushed_to_float64():
    # 400 000 rows over <= 296 CTAs: more than 256 rows per CTA, so every CTA flushes its FP32 accumulators several times; the
    # diagonal (sums of squares, all terms of one sign) is where a long FP32 run of truncated additions would show
    n, s = 400_000, 64
    rng = np.random.default_rng(5)
    U, W = _rand_block(rng, n, s), _rand_block(rng, n, s)
    op = _op(s)
    G = to_np(op.gram(to_dev(U, "c64"), to_dev(W, "c64")))
    Gu = to_np(op.gram(to_dev(U, "c64"), to_dev(U, "c64")))
    G2 = to_np(op.gram(to_dev(U, "c64"), to_dev(W, "c64")))
    op.close()
    assert _gram_err(G, U, W) <= 2e-6
    assert _gram_err(Gu, U, U) <= 2e-6
    d = np.diag(Gu).real
    assert np.max(np.abs(d - np.sum(np.abs(U) ** 2, axis=0)) / d) <= 1e-6
    assert np.array_equal(G, G2)                                  # deterministic: fixed partition, fixed order, no atomics


@pytest.mark.parametrize("s", [16, 64])
def test_tensor_gram_and_rotation_with_magnitudes_spread_over_rows_and_columns(s):
    # a "point source": a few rows carry numbers 1e+12 times larger than the rest (the CTA scales of the Gram kernel must be
    # re-set and its accumulators flushed when such a tile arrives), blocks of zero rows, and columns of very different norm
    n = 30_000
    rng = np.random.default_rng(11 + s)
    U, W = _rand_block(rng, n, s), _rand_block(rng, n, s)
    rows = np.ones(n)
    rows[:5000] = 1e-6
    rows[5000:9000] = 0.0
    rows[17000:17040] = 1e+6
    cols = 10.0 ** rng.integers(-6, 7, size=s)
    U = (U * rows[:, None] * cols[None, :]).astype(np.complex64).astype(np.complex128)
    W = (W * rows[::-1, None]).astype(np.complex64).astype(np.complex128)
    K = _rand_block(rng, s, s) * (10.0 ** rng.integers(-5, 6, size=s))[None, :]
    op = _op(s)
    G = to_np(op.gram(to_dev(U, "c64"), to_dev(W, "c64")))
    Wd = to_dev(W, "c64")
    op.rotate(to_dev(U, "c64"), to_dev(K, "c128"), Wd, 1.0)
    op.close()
    assert _gram_err(G, U, W) <= 2e-6
    ref = W + U @ K
    assert rel_err_cols(to_np(Wd).reshape(n, 1, s), ref.reshape(n, 1, s)) <= 1e-6


@pytest.mark.parametrize("s", WIDTHS)
@pytest.mark.parametrize("n", [1, 65, 4099])
@pytest.mark.parametrize("beta", [0.0, 1.0, -0.25])
def test_tensor_rotation_matches_oracle(n, s, beta):
    rng = np.random.default_rng(3 * n + s)
    U, W, K = _rand_block(rng, n, s), _rand_block(rng, n, s), _rand_block(rng, s, s)
    op = _op(s)
    Wd = to_dev(W, "c64")
    op.rotate(to_dev(U, "c64"), to_dev(K, "c128"), Wd, beta)
    op.close()
    ref = oracle.block_rotate(U, K, W, beta)
    if n >= 8:
        assert rel_err_cols(to_np(Wd).reshape(n, 1, s), ref.reshape(n, 1, s)) <= 1e-6
    else:               # a column of one row is one number (it may be a cancelling sum): compare against the size of its terms
        terms = np.abs(U) @ np.abs(K) + abs(beta) * np.abs(W)
        assert np.max(np.abs(to_np(Wd) - ref) / terms) <= 1e-6


def test_tensor_rotation_identity_and_imaginary_unit():
    # K = I reproduces U to 2^-21 per element (hi + 2^-11 lo carries 22-23 bits), K = i I multiplies by i (re/im signs)
    n, s = 777, 32
    rng = np.random.default_rng(1)
    U = _rand_block(rng, n, s)
    op = _op(s)
    for K, ref in ((np.eye(s, dtype=np.complex128), U), (1j * np.eye(s, dtype=np.complex128), 1j * U)):
        Wd = torch.zeros((n, s), dtype=torch.complex64, device="cuda")
        op.rotate(to_dev(U, "c64"), to_dev(K, "c128"), Wd, 0.0)
        Y = to_np(Wd)
        assert np.all(np.abs(Y.view(np.float64) - ref.view(np.float64)) <= 2.0 ** -21 * np.abs(ref.view(np.float64)))
    op.close()


@pytest.mark.parametrize("s,flags", [(16, cm.binding.FLAG_TENSOR_LINALG), (32, cm.binding.FLAG_TENSOR_LINALG), (64, 0)])
def test_block_cg_through_the_tensor_linear_algebra(s, flags):
    # BlockCGrQ with every Gram product and rotation on the tensor cores against the oracle: iteration count, histories, true residual
    dims, nb, tol = (4, 4, 4, 4), 32, 1e-6
    A, c = synth.make_operator(dims, nb, 20240903, 1.02)
    B = synth.make_block(dims, nb, s, 20240903, synth.TAG_B)
    ref = oracle.block_cg(dims, A, B, tol=tol, maxiter=100)
    outs = {}
    for name, fl in (("tensor", flags), ("simt", cm.binding.FLAG_NO_TENSOR)):
        op = cm.CoarseOperator(dims, to_dev(A, "c64"), s, flags=fl)
        outs[name] = op.block_cg(to_dev(B, "c64"), tol=tol, maxiter=100)
        op.close()
    out = outs["tensor"]
    assert out["status"] == 0 and out["iterations"] == ref["iterations"] == outs["simt"]["iterations"]
    assert max(out["rel_res_true"]) <= tol * 1.001 + 2e-7
    k = ref["iterations"]
    h_ref = ref["history"].max(axis=1)[:k + 1]
    mask = h_ref > 1e-5
    assert np.allclose(np.array(out["history"][:k + 1])[mask], h_ref[mask], rtol=5e-2)
    assert rel_err_cols(to_np(out["X"]), ref["X"]) <= 1e-5
