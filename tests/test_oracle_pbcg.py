"""Pins of the Preconditioned BlockCGrQ oracle (oracle/pbcg_oracle.py; Fig. 2 right):
 * M^-1 = identity reduces it to the unpreconditioned BlockCGrQ oracle (a different implementation: C, own Cholesky):
   same iteration count, same residual history, same iterates;
 * the solution against numpy.linalg.solve on the dense brute-force matrix;
 * s = 1 against textbook preconditioned CG (Saad, Alg. 9.1) written out in the test;
 * invariants every iteration: Q^H q = I (orthonormal in the M inner product), B - H X_k = q_k C_k;
 * M^-1 = H^-1 exactly => convergence in one iteration; the printed update without C_k does NOT solve the system.
"""
import numpy as np
import pytest

from helpers import dense_matrix, rel_err_cols
from inputs import synth
from oracle import cheby_oracle, oracle, pbcg_oracle

DIMS, NB = (2, 2, 2, 3), 6


def _case(s, seed=21, factor=1.05):
    A, c = synth.make_operator(DIMS, NB, seed, factor)
    B = synth.make_block(DIMS, NB, s, seed, synth.TAG_B)
    return A, c, B


def test_identity_preconditioner_reduces_to_block_cgrq():
    A, c, B = _case(4)
    ref = oracle.block_cg(DIMS, A, B, tol=1e-10, maxiter=100)
    out = pbcg_oracle.pblock_cg(DIMS, A, B, lambda R: R, tol=1e-10, maxiter=100)
    assert out["status"] == ref["status"] == 0 and out["iterations"] == ref["iterations"]
    assert np.allclose(out["history"], ref["history"], rtol=1e-8)
    assert rel_err_cols(out["X"], ref["X"]) <= 1e-12


@pytest.mark.parametrize("kind", ["cheby", "defl+cheby"])
def test_solution_equals_dense_solve_and_invariants_hold(kind):
    s = 3
    A, c, B = _case(s)
    Hd = dense_matrix(DIMS, A.astype(np.complex128))
    lam, U = np.linalg.eigh(Hd)
    n = Hd.shape[0]
    if kind == "cheby":
        Minv = lambda R: cheby_oracle.cheby_apply(DIMS, A, R, 0.9 * lam[0], 1.1 * lam[-1], 2)
    else:
        Minv = lambda R: cheby_oracle.cheby_defl_solve(DIMS, A, U[:, :5], lam[:5], R, 0.9 * lam[5], 1.1 * lam[-1], 2)
    b = B.reshape(n, s)

    def check(k, st):
        r = b - Hd @ st["X"].reshape(n, s)
        assert np.linalg.norm(r - st["q"] @ st["C"]) <= 1e-10 * np.linalg.norm(b)                  # r_k = q_k C_k
        # <Q|Q>_M = 1.  T = Q - Z N is a difference of O(1) blocks of size ||S|| (the reduction factor of the step), so the
        # Gram matrix T^H t is accurate to eps / ||S||^2 only: checked while the residual is far above rounding
        if np.linalg.norm(r) > 1e-7 * np.linalg.norm(b):
            assert np.allclose(st["Q"].conj().T @ st["q"], np.eye(s), atol=1e-6)

    out = pbcg_oracle.pblock_cg(DIMS, A, B, Minv, tol=1e-11, maxiter=100, callback=check)
    assert out["status"] == 0 and out["true_rel"].max() <= 1e-10
    assert rel_err_cols(out["X"].reshape(n, 1, s), np.linalg.solve(Hd, b).reshape(n, 1, s)) <= 1e-10
    plain = oracle.block_cg(DIMS, A, B, tol=1e-11, maxiter=100)
    assert out["iterations"] < plain["iterations"]                                                  # the preconditioner helps


def test_single_rhs_equals_textbook_pcg():
    A, c, B = _case(1)
    Hd = dense_matrix(DIMS, A.astype(np.complex128))
    lam = np.linalg.eigvalsh(Hd)
    lo, hi = 0.9 * lam[0], 1.1 * lam[-1]
    n = Hd.shape[0]
    Md = lambda v: cheby_oracle.cheby_apply(DIMS, A, v.reshape(B.shape), lo, hi, 3).reshape(n)
    # Saad, Iterative Methods, Algorithm 9.1
    b = B.reshape(n)
    x = np.zeros(n, dtype=np.complex128)
    r = b.copy(); zv = Md(r); p = zv.copy()
    xs = []
    for _ in range(6):
        Ap = Hd @ p
        alpha = np.vdot(r, zv) / np.vdot(p, Ap)
        x = x + alpha * p
        r_new = r - alpha * Ap
        z_new = Md(r_new)
        beta = np.vdot(r_new, z_new) / np.vdot(r, zv)
        p = z_new + beta * p
        r, zv = r_new, z_new
        xs.append(x.copy())
    got = []
    pbcg_oracle.pblock_cg(DIMS, A, B, lambda R: cheby_oracle.cheby_apply(DIMS, A, R, lo, hi, 3), tol=1e-300, maxiter=6,
                          callback=lambda k, st: got.append(st["X"].reshape(n).copy()))
    for a, bb in zip(got, xs):
        assert np.linalg.norm(a - bb) <= 1e-11 * np.linalg.norm(bb)


def test_exact_preconditioner_converges_in_one_iteration_and_printed_update_fails():
    s = 2
    A, c, B = _case(s)
    Hd = dense_matrix(DIMS, A.astype(np.complex128))
    n = Hd.shape[0]
    Hinv = np.linalg.inv(Hd)
    out = pbcg_oracle.pblock_cg(DIMS, A, B, lambda R: (Hinv @ R.reshape(n, s)).reshape(R.shape), tol=1e-10, maxiter=10)
    assert out["iterations"] == 1 and out["true_rel"].max() <= 1e-10
    # the listing as printed (X + D N, no C_k): one step with the exact preconditioner would have to give the solution
    b = B.reshape(n, s)
    Z = Hinv @ b
    G = Z.conj().T @ b
    C = np.linalg.cholesky(0.5 * (G + G.conj().T)).conj().T
    D = Z @ np.linalg.inv(C)
    N = np.linalg.inv(D.conj().T @ (Hd @ D))
    x_printed, x_read = D @ N, D @ N @ C
    assert np.linalg.norm(b - Hd @ x_read) <= 1e-10 * np.linalg.norm(b)
    assert np.linalg.norm(b - Hd @ x_printed) >= 1e-2 * np.linalg.norm(b)
