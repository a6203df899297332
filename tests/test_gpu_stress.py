"""-m gpu parity of block_cg_solve on ILL-CONDITIONED operators (SURVEY.md section 8(c) "stress operator") and on the
breakdown / long-history paths.

The BASELINE.json operators are diagonally dominant by a loose Frobenius bound (kappa ~ 1.15, 4-7 iterations), which
makes "iteration counts within 5 %" an equality on a single-digit count.  Here the diagonal shift is taken from the
spectrum instead:  c = (1 + delta) |lambda_min(off-diagonal part)|  with lambda_min from a dense `eigvalsh` of the
brute-force matrix on a small lattice (tests/helpers.dense_matrix: independent of the oracle and of the CUDA path), so
kappa(H) ~ (lambda_max - lambda_min)/(delta |lambda_min|): delta = 0.02 -> kappa ~ 100, delta = 0.001 -> kappa ~ 2000
(the paper's real coarse operator: spectrum [0.02, 40], ~120 CG iterations to 4e-2).  These
operators have NO dominant diagonal (c ~ 6 against off-diagonal blocks of norm ~ 1): the case where the split-FP16
kernel's error is largest.
"""
import numpy as np
import pytest
import torch

from gpu_common import TOL, to_dev, to_np
from helpers import rel_err_cols, stress_operator
from inputs import synth
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def stress_case(dims, nb, seed, delta):
    A, c, lmin, lmax = stress_operator(dims, nb, seed, delta)
    return A, c, lmax / lmin


def _solve_both(dims, A, B, dtype, tol, maxiter, flags=0):
    s = B.shape[-1]
    ref = oracle.block_cg(dims, A, B, tol=tol, maxiter=maxiter)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s, flags=flags)
    name = op.kernel_name(s)
    out = op.block_cg(to_dev(B, dtype), to_dev(np.zeros_like(B), dtype), tol=tol, maxiter=maxiter)
    op.close()
    out["X"] = to_np(out["X"])
    return out, ref, name


# ---- complex128: the 5 % bar bites (74-93 iterations), histories to 1e-6 -------------------------------------------------
@pytest.mark.parametrize("delta", [0.02, 0.001])
def test_stress_c128_matches_oracle(delta):
    dims, nb, s, tol = (4, 4, 4, 4), 8, 4, 1e-10
    A, c, kappa = stress_case(dims, nb, 20240903, delta)
    B = synth.make_block(dims, nb, s, 20240903, synth.TAG_B)
    out, ref, name = _solve_both(dims, A, B, "c128", tol, 1000)
    print(f"stress c128 delta={delta}: kappa={kappa:.0f} kernel={name} its gpu/oracle={out['iterations']}/{ref['iterations']} "
          f"true={max(out['rel_res_true']):.2e}/{np.max(ref['true_rel']):.2e}")
    assert kappa > (50 if delta == 0.02 else 1000)
    assert out["status"] == ref["status"] == 0
    assert ref["iterations"] >= 50
    assert abs(out["iterations"] - ref["iterations"]) <= 0.05 * ref["iterations"]
    # both reach the tolerance in the TRUE residual (recursive and true residual agree to ~kappa eps)
    assert max(out["rel_res_true"]) <= tol * 1.01 + kappa * 1e-15
    k = min(out["iterations"], ref["iterations"])
    h_ref, h_gpu = ref["history"].max(axis=1)[:k + 1], np.array(out["history"][:k + 1])
    # the two iterations are the same recurrence in different rounding (FMA, summation order): histories agree to a relative
    # error that grows with the iteration count; 1e-6 holds for the first half, 5 % to the end
    assert np.allclose(h_gpu[:k // 2], h_ref[:k // 2], rtol=1e-6)
    assert np.allclose(h_gpu, h_ref, rtol=5e-2)
    assert rel_err_cols(out["X"], ref["X"]) <= 10 * tol * kappa


# ---- complex64 through the split-FP16 tensor kernel, no dominant diagonal --------------------------------------------------
# Bars ("ill-conditioned operators in complex64"): float32 storage of the blocks limits the TRUE residual to
# ~ eps32 kappa (||B - H X|| / ||B|| <= eps32 ||H|| ||X|| / ||B||), so the bar is tol + 6e-8 kappa, and tolerances below that
# attainable level (1e-6 at kappa = 2000) are a separate, characterised case below.  The tensor kernels' apply error is
# SYSTEMATIC (the tensor core truncates when it adds into its FP32 accumulator): block CG then converges to the solution of
# a perturbed system, ||X - X_oracle|| / ||X|| <= kappa (tol + e_apply) with e_apply the apply's own measured error.
@pytest.mark.parametrize("delta,tol", [(0.02, 1e-6), (0.02, 1e-4), (0.001, 1e-5), (0.001, 1e-4)])
def test_stress_c64_through_the_tensor_kernel(delta, tol):
    dims, nb, s = (4, 4, 2, 2), 32, 16
    A, c, kappa = stress_case(dims, nb, 77, delta)
    B = synth.make_block(dims, nb, s, 77, synth.TAG_B)
    out, ref, name = _solve_both(dims, A, B, "c64", tol, 1000)
    e_apply = _apply_error(dims, A, s)
    hist = np.array(out["history"])
    print(f"stress c64 delta={delta} tol={tol}: kappa={kappa:.0f} kernel={name} e_apply={e_apply:.2e} its gpu/oracle={out['iterations']}/{ref['iterations']} "
          f"status={out['status']} true={max(out['rel_res_true']):.2e} recursive={max(out['rel_res_recursive']):.2e} "
          f"sol_err={rel_err_cols(out['X'], ref['X']):.2e}")
    assert name.startswith("stencil_h16")                           # the split-FP16 tensor kernel is underneath
    assert e_apply <= TOL["c64"]
    assert out["status"] == ref["status"] == 0
    assert ref["iterations"] >= 25
    assert abs(out["iterations"] - ref["iterations"]) <= 0.05 * ref["iterations"], (out["iterations"], ref["iterations"])
    k = min(out["iterations"], ref["iterations"])
    h_ref = ref["history"].max(axis=1)[:k + 1]
    floor = 6e-8 * kappa                                             # float32 blocks: attainable residual ~ eps32 kappa
    mask = h_ref > max(1e-5, floor)                                  # histories are compared above the attainable accuracy
    assert np.allclose(hist[:k + 1][mask], h_ref[mask], rtol=5e-2)
    assert max(out["rel_res_true"]) <= tol * 1.01 + floor, (max(out["rel_res_true"]), floor)
    assert rel_err_cols(out["X"], ref["X"]) <= kappa * (tol + e_apply)


def _apply_error(dims, A, s, flags=0):
    X = synth.make_block(dims, A.shape[-1], s, 1234, synth.TAG_X)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), s, flags=flags)
    Y = to_np(op.apply(to_dev(X, "c64")))
    op.close()
    return rel_err_cols(Y, oracle.apply(dims, A, X))


@pytest.mark.parametrize("flags", [0, cm.binding.FLAG_NO_TENSOR])
def test_stress_c64_below_the_attainable_accuracy_is_characterised_not_hidden(flags):
    # kappa = 2000, tol = 1e-6 < eps32 kappa: no float32 implementation can deliver this (the oracle works in float64: 45
    # iterations).  What the CUDA path does, measured on B200 and asserted so that a regression shows: it still reports
    # convergence of the RECURSIVE residual, needs up to 25 % more iterations (tensor kernel 54, SIMT 47-48), and the true
    # residual stalls near 2e-5 ... 5e-5 -- reported in rel_res_true, which is why the API returns both.
    dims, nb, s, tol = (4, 4, 2, 2), 32, 16, 1e-6
    A, c, kappa = stress_case(dims, nb, 77, 0.001)
    B = synth.make_block(dims, nb, s, 77, synth.TAG_B)
    out, ref, name = _solve_both(dims, A, B, "c64", tol, 1000, flags=flags)
    print(f"below attainable accuracy: kernel={name} its gpu/oracle={out['iterations']}/{ref['iterations']} true={max(out['rel_res_true']):.2e}")
    assert out["status"] == ref["status"] == 0
    assert ref["iterations"] <= out["iterations"] <= 1.25 * ref["iterations"]
    assert tol < max(out["rel_res_true"]) <= 6e-8 * kappa


# ---- breakdown, end to end, deterministic on both sides -----------------------------------------------------------------------
def _identity_like_operator(dims, nb, diag):
    V = synth.volume(dims)
    A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
    d = np.arange(nb)
    A[:, 40, d, d] = np.asarray(diag, dtype=np.complex64)[None, :]
    return A


def _integer_block(dims, nb, s):
    """s mutually orthogonal columns with entries in {0, +1, -1}, 4 nonzeros each: every Gram sum, Cholesky factor and
    rotation of the first iteration is exact in float32 and float64."""
    V = synth.volume(dims)
    B = np.zeros((V * nb, s), dtype=np.complex128)
    for r in range(s):
        B[4 * r:4 * r + 4, r] = [1, -1, 1, 1]
    return B.reshape(V, nb, s)


@pytest.mark.parametrize("dtype,nb,s", [("c128", 8, 4), ("c64", 32, 16)])
def test_breakdown_inside_the_loop_T_is_exactly_zero(dtype, nb, s):
    # H = I: the first iteration solves the system exactly, T = Q - Z M = 0 exactly, T^H T = 0 is not positive definite:
    # COARSE_BREAKDOWN from statement 11 of iteration 1 (no column deflation, R12); X holds the iterate of statement 10
    dims = (2, 2, 2, 2)
    A, B = _identity_like_operator(dims, nb, np.ones(nb)), _integer_block(dims, nb, s)
    out, ref, name = _solve_both(dims, A, B, dtype, 1e-30, 10)
    assert ref["status"] == oracle.BREAKDOWN and out["status"] == cm.binding.BREAKDOWN
    assert out["iterations"] == ref["iterations"] == 1
    assert np.array_equal(out["X"], B) and np.array_equal(ref["X"], B)          # the exact solution, bit for bit
    assert max(out["rel_res_true"]) == 0.0


@pytest.mark.parametrize("dtype,nb,s", [("c128", 8, 4), ("c64", 32, 16)])
def test_breakdown_on_an_indefinite_operator_leaves_X_at_the_last_valid_iterate(dtype, nb, s):
    # H = diag(-1, ...): D^H Z = -I is not positive definite: COARSE_BREAKDOWN from statement 9 of the first iteration;
    # the block passes already enqueued behind the s x s kernel must not touch X (coarse_mrhs.h "breakdown contract")
    dims = (2, 2, 2, 2)
    A, B = _identity_like_operator(dims, nb, -np.ones(nb)), _integer_block(dims, nb, s)
    ref = oracle.block_cg(dims, A, B, tol=1e-30, maxiter=10)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    X0 = synth.make_block(dims, nb, s, 3, synth.TAG_U)
    Xd = to_dev(X0, dtype)
    out = op.block_cg(to_dev(B, dtype), Xd, tol=1e-30, maxiter=10)
    assert ref["status"] == oracle.BREAKDOWN and ref["iterations"] == 0
    assert out["status"] == cm.binding.BREAKDOWN and out["iterations"] == 0
    assert np.array_equal(to_np(Xd), X0.astype(np.complex64 if dtype == "c64" else np.complex128).astype(np.complex128))
    # begin / step / end: further steps after the breakdown keep X frozen and end reports it
    Xd2 = to_dev(X0, dtype)
    st, _ = op.block_cg_begin(to_dev(B, dtype), Xd2, tol=1e-30)
    assert st == cm.binding.NOT_CONVERGED
    op.block_cg_step(3)
    out2 = op.block_cg_end()
    op.close()
    assert out2["status"] == cm.binding.BREAKDOWN
    assert np.array_equal(to_np(Xd2), to_np(Xd))


def test_zero_source_column_breaks_down_at_the_start_on_both_sides():
    # a zero column makes R_0^H R_0 singular: statement 5 (Q_0 C_0 = R_0) fails on both sides, iterations = 0, X = X_0
    dims, nb, s = (2, 2, 2, 2), 8, 4
    A, c = synth.make_operator(dims, nb, 5, 1.05)
    B = synth.make_block(dims, nb, s, 5, synth.TAG_B)
    B[:, :, 2] = 0.0
    out, ref, _ = _solve_both(dims, A, B, "c128", 1e-10, 10)
    assert ref["status"] == oracle.BREAKDOWN and out["status"] == cm.binding.BREAKDOWN
    assert out["iterations"] == ref["iterations"] == 0
    assert not out["X"].any()


# ---- more than COARSE_MAX_HISTORY iterations ---------------------------------------------------------------------------------
def test_history_longer_than_the_result_array():
    # kappa ~ 2e5, one right-hand side (plain CG), tolerance out of reach: exactly maxiter = 300 iterations on both sides;
    # history[] keeps the first COARSE_MAX_HISTORY = 256 entries only.  The recursive residual keeps falling (1e-21) long after
    # the true one has stalled at ~kappa eps: both are reported.
    dims, nb, s = (4, 4, 4, 4), 8, 1
    A, c, kappa = stress_case(dims, nb, 11, 1e-5)
    B = synth.make_block(dims, nb, s, 11, synth.TAG_B)
    out, ref, _ = _solve_both(dims, A, B, "c128", 1e-30, 300)
    print(f"long history: kappa={kappa:.0f} its gpu/oracle={out['iterations']}/{ref['iterations']} true={max(out['rel_res_true']):.2e}/{ref['true_rel'].max():.2e} "
          f"recursive={max(out['rel_res_recursive']):.2e}/{ref['history'][-1].max():.2e}")
    assert out["status"] == ref["status"] == cm.binding.NOT_CONVERGED
    assert out["iterations"] == ref["iterations"] == 300 > cm.binding.MAX_HISTORY
    assert len(out["history"]) == cm.binding.MAX_HISTORY and all(h >= 0.0 for h in out["history"])
    h_ref = ref["history"][:cm.binding.MAX_HISTORY, 0]
    mask = h_ref > 1e-8
    assert mask.sum() > 100 and np.allclose(np.array(out["history"])[mask], h_ref[mask], rtol=1e-4)
    assert max(out["rel_res_true"]) <= 1e-10 and ref["true_rel"].max() <= 1e-10
    assert rel_err_cols(out["X"], ref["X"]) <= 1e-8
