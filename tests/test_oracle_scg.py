"""Pins of the stacked single-Krylov CG oracle (oracle/scg_oracle.py):
 * scipy.sparse.linalg.cg (a library routine) on the Kronecker system (I_s (x) H) vec(X) = vec(B): same iterates;
 * numpy.linalg.solve on the dense matrix; * s = 1 is plain CG = BlockCGrQ with one column (same iterates and count);
 * the iteration count is that of the slowest single right-hand side within one or two iterations (no block gain).
"""
import numpy as np
import scipy.sparse.linalg as spla

from helpers import dense_matrix, rel_err_cols
from inputs import synth
from oracle import oracle, scg_oracle

DIMS, NB = (2, 2, 2, 3), 6


def _case(s, seed=17):
    A, c = synth.make_operator(DIMS, NB, seed, 1.05)
    return A, synth.make_block(DIMS, NB, s, seed, synth.TAG_B)


def test_iterates_equal_scipy_cg_on_the_kronecker_system():
    s = 3
    A, B = _case(s)
    Hd = dense_matrix(DIMS, A.astype(np.complex128))
    n = Hd.shape[0]
    big = np.kron(Hd, np.eye(s))                       # acts on the row-major flattening [n][s]
    b = B.reshape(n * s)
    for k in (1, 2, 4):
        xk, _ = spla.cg(big, b, x0=np.zeros_like(b), rtol=0.0, atol=0.0, maxiter=k)
        out = scg_oracle.stacked_cg(DIMS, A, B, tol=0.0, maxiter=k)
        assert out["iterations"] == k
        assert np.linalg.norm(out["X"].reshape(-1) - xk) <= 1e-11 * np.linalg.norm(xk)


def test_solution_equals_dense_solve():
    s = 4
    A, B = _case(s)
    Hd = dense_matrix(DIMS, A.astype(np.complex128))
    n = Hd.shape[0]
    out = scg_oracle.stacked_cg(DIMS, A, B, tol=1e-11, maxiter=200)
    assert out["status"] == 0 and out["true_rel"].max() <= 1e-10
    assert rel_err_cols(out["X"].reshape(n, 1, s), np.linalg.solve(Hd, B.reshape(n, s)).reshape(n, 1, s)) <= 1e-10


def test_single_rhs_equals_block_cgrq_with_one_column():
    A, B = _case(1)
    ref = oracle.block_cg(DIMS, A, B, tol=1e-10, maxiter=100)
    out = scg_oracle.stacked_cg(DIMS, A, B, tol=1e-10, maxiter=100)
    assert out["iterations"] == ref["iterations"]
    assert np.allclose(out["history"], ref["history"][:, 0], rtol=1e-7)
    assert rel_err_cols(out["X"], ref["X"]) <= 1e-11


def test_no_block_gain():
    s = 4
    A, B = _case(s)
    counts = [oracle.block_cg(DIMS, A, B[:, :, r:r + 1], tol=1e-10, maxiter=100)["iterations"] for r in range(s)]
    out = scg_oracle.stacked_cg(DIMS, A, B, tol=1e-10, maxiter=100)
    assert abs(out["iterations"] - max(counts)) <= 2
