"""-m gpu parity of pblock_cg_solve (Preconditioned BlockCGrQ, Fig. 2 right) against oracle/pbcg_oracle.py
with the same stationary preconditioner on both sides (oracle/cheby_oracle.py).  Bars as for block_cg_solve (DESIGN.md
section 6): status equal, iteration counts within 5 %, true residual <= tol, histories equal while above the dtype's
attainable accuracy, solutions equal to what the tolerance allows."""
import numpy as np
import pytest

from gpu_common import TOL, host_case, to_dev, to_np
from helpers import dense_matrix, rel_err_cols
from oracle import cheby_oracle, oracle, pbcg_oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _check(out, ref, tol, dtype):
    assert out["status"] == ref["status"] == 0
    assert abs(out["iterations"] - ref["iterations"]) <= 0.05 * ref["iterations"], (out["iterations"], ref["iterations"])
    assert max(out["rel_res_true"]) <= tol * (1.0 + 1e-3) + (0 if dtype == "c128" else 3e-7)
    k = min(out["iterations"], ref["iterations"])
    h_ref = ref["history"].max(axis=1)[:k + 1]
    h_gpu = np.array(out["history"][:k + 1])
    mask = h_ref > (1e-11 if dtype == "c128" else 1e-5)
    assert np.allclose(h_gpu[mask], h_ref[mask], rtol=1e-5 if dtype == "c128" else 5e-2)
    assert rel_err_cols(to_np(out["X"]), ref["X"]) <= max(10 * tol, TOL[dtype])


@pytest.mark.parametrize("dims,nb,s,dtype,order,tol", [
    ((4, 4, 4, 4), 8, 4, "c128", 3, 1e-10),      # BASELINE configs[0] shape
    ((3, 3, 3, 5), 24, 8, "c128", 2, 1e-10),
    ((4, 4, 4, 4), 32, 16, "c64", 2, 1e-6),      # FP16-split tensor kernel underneath
    ((3, 3, 2, 4), 13, 5, "c128", 4, 1e-10),
])
def test_pblock_cg_with_chebyshev_preconditioner_matches_oracle(dims, nb, s, dtype, order, tol):
    A, c, _, B = host_case(dims, nb, s, seed=600 + nb + s, factor=1.03)
    lo, hi = c - 12.0, c + 12.0
    ref = pbcg_oracle.pblock_cg(dims, A, B, lambda R: cheby_oracle.cheby_apply(dims, A, R, lo, hi, order), tol=tol, maxiter=100)
    plain = oracle.block_cg(dims, A, B, tol=tol, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    out = op.pblock_cg(to_dev(B, dtype), lo, hi, order, tol=tol, maxiter=100)
    op.close()
    _check(out, ref, tol, dtype)
    assert out["iterations"] <= plain["iterations"]


@pytest.mark.parametrize("dtype,tol", [("c128", 1e-10), ("c64", 1e-6)])
def test_pblock_cg_with_deflated_chebyshev_preconditioner_matches_oracle(dtype, tol):
    from inputs import synth
    dims, nb, s, nev, order = (2, 2, 2, 3), 8, 6, 6, 2
    A, c = synth.make_operator(dims, nb, 41, 1.05)
    B = synth.make_block(dims, nb, s, 41, synth.TAG_B)
    lam, U = np.linalg.eigh(dense_matrix(dims, A.astype(np.complex128)))
    Vev, lo, hi = U[:, :nev].copy(), 0.95 * lam[nev], 1.05 * lam[-1]
    Vq = Vev.astype(np.complex64).astype(np.complex128) if dtype == "c64" else Vev
    ref = pbcg_oracle.pblock_cg(dims, A, B, lambda R: cheby_oracle.cheby_defl_solve(dims, A, Vq, lam[:nev], R, lo, hi, order),
                                tol=tol, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    out = op.pblock_cg(to_dev(B, dtype), lo, hi, order, Vev=to_dev(Vev, dtype), lam=lam[:nev], tol=tol, maxiter=100)
    op.close()
    _check(out, ref, tol, dtype)


def test_pblock_cg_nonzero_start_maxiter_and_bad_arguments():
    dims, nb, s = (4, 4, 4, 4), 8, 4
    A, c, X0, B = host_case(dims, nb, s, seed=7, factor=1.05)
    lo, hi = c - 12.0, c + 12.0
    Minv = lambda R: cheby_oracle.cheby_apply(dims, A, R, lo, hi, 2)
    ref = pbcg_oracle.pblock_cg(dims, A, B, Minv, X0=X0, tol=1e-10, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), s)
    out = op.pblock_cg(to_dev(B, "c128"), lo, hi, 2, X=to_dev(X0, "c128"), tol=1e-10, maxiter=100)
    _check(out, ref, 1e-10, "c128")
    out2 = op.pblock_cg(to_dev(B, "c128"), lo, hi, 2, tol=1e-30, maxiter=2)
    assert out2["status"] == cm.binding.NOT_CONVERGED and out2["iterations"] == 2
    ref2 = pbcg_oracle.pblock_cg(dims, A, B, Minv, tol=1e-30, maxiter=2)
    assert rel_err_cols(to_np(out2["X"]), ref2["X"]) <= 1e-10
    with pytest.raises(cm.binding.CoarseError):
        op.pblock_cg(to_dev(B, "c128"), hi, lo, 2)
    op.close()
