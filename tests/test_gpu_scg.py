"""-m gpu parity of stacked_cg_solve (single-Krylov CG on the stacked system) against oracle/scg_oracle.py.
Bars as for block_cg_solve."""
import numpy as np
import pytest

from gpu_common import TOL, host_case, to_dev, to_np
from helpers import rel_err_cols
from oracle import scg_oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


@pytest.mark.parametrize("dims,nb,s,dtype,tol", [
    ((4, 4, 4, 4), 8, 4, "c128", 1e-10),
    ((3, 3, 3, 5), 24, 8, "c128", 1e-10),
    ((4, 4, 4, 4), 32, 16, "c64", 1e-6),
    ((3, 3, 2, 4), 13, 5, "c128", 1e-10),
    ((3, 3, 3, 3), 32, 64, "c64", 1e-6),
    ((4, 4, 4, 4), 32, 1, "c64", 1e-6),
])
def test_stacked_cg_matches_oracle(dims, nb, s, dtype, tol):
    A, c, _, B = host_case(dims, nb, s, seed=700 + nb + s, factor=1.03)
    ref = scg_oracle.stacked_cg(dims, A, B, tol=tol, maxiter=200)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    out = op.stacked_cg(to_dev(B, dtype), tol=tol, maxiter=200)
    op.close()
    assert out["status"] == ref["status"] == 0
    assert abs(out["iterations"] - ref["iterations"]) <= 0.05 * ref["iterations"], (out["iterations"], ref["iterations"])
    assert max(out["rel_res_true"]) <= 3 * tol + (0 if dtype == "c128" else 3e-7)      # the stop is on the stacked norm: a column may sit above it
    assert np.max(ref["true_rel"]) <= 3 * tol
    k = min(out["iterations"], ref["iterations"])
    h_ref, h_gpu = ref["history"][:k + 1], np.array(out["history"][:k + 1])
    mask = h_ref > (1e-11 if dtype == "c128" else 1e-5)
    assert np.allclose(h_gpu[mask], h_ref[mask], rtol=1e-6 if dtype == "c128" else 5e-2)
    assert rel_err_cols(to_np(out["X"]), ref["X"]) <= max(10 * tol, TOL[dtype])


def test_stacked_cg_nonzero_start_and_maxiter():
    dims, nb, s = (4, 4, 4, 4), 8, 4
    A, c, X0, B = host_case(dims, nb, s, seed=8, factor=1.05)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), s)
    out = op.stacked_cg(to_dev(B, "c128"), X=to_dev(X0, "c128"), tol=1e-30, maxiter=3)
    op.close()
    ref = scg_oracle.stacked_cg(dims, A, B, X0=X0, tol=1e-30, maxiter=3)
    assert out["status"] == cm.binding.NOT_CONVERGED and out["iterations"] == 3
    assert rel_err_cols(to_np(out["X"]), ref["X"]) <= 1e-12
    assert np.allclose(out["history"][:4], ref["history"][:4], rtol=1e-9)
