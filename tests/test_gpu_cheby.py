"""-m gpu parity of coarse_cheby_apply (Chebyshev polynomial coarse solve) against oracle/cheby_oracle.py.

Tolerances: the polynomial is evaluated by a three-term recurrence with order - 1 applications of the operator; rounding
errors of the apply (1e-15 complex128, ~1.5e-7 complex64 per application) accumulate at most linearly in
the order while the terms T_j(y(H)) B stay bounded by ||B|| (spectrum inside [lo, hi]); the result is compared norm-wise per
column: <= 1e-12 (complex128), <= 1e-5 (complex64) -- north_star's figures -- for orders up to 120 (the paper's coarse solve).
"""
import numpy as np
import pytest
import torch

from gpu_common import TOL, host_case, to_dev, to_np
from helpers import rel_err_cols
from oracle import cheby_oracle, oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _gpu(dims, A, B, dtype, lo, hi, order, flags=0):
    s = B.shape[-1]
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s, flags=flags)
    name = op.kernel_name(s)
    Bd = to_dev(B, dtype)
    X = to_np(op.cheby_apply(Bd, lo, hi, order))
    assert np.array_equal(to_np(Bd), B.astype(np.complex64 if dtype == "c64" else np.complex128).astype(np.complex128))   # B untouched
    op.close()
    return X, name


@pytest.mark.parametrize("dims,nb,s,dtype,order", [
    ((4, 4, 4, 4), 8, 4, "c128", 12),       # BASELINE configs[0] shape
    ((3, 3, 3, 5), 24, 8, "c128", 9),       # configs[1] shape, ragged lattice
    ((4, 4, 4, 4), 32, 16, "c64", 8),       # configs[2] shape: FP16-split tensor kernel underneath; the paper's smoother order
    ((3, 3, 2, 4), 32, 64, "c64", 16),      # transposed tensor form underneath
    ((3, 2, 2, 3), 13, 5, "c128", 32),      # generic stencil kernel, odd sizes
    ((4, 3, 3, 4), 24, 16, "c64", 1),       # order 1: X = B / midpoint
    ((4, 3, 3, 4), 24, 16, "c64", 2),       # order 2: one application
])
def test_cheby_apply_matches_oracle(dims, nb, s, dtype, order):
    A, c, _, B = host_case(dims, nb, s, seed=500 + nb + s, factor=1.05)
    # the synthetic operator's spectrum lies within c +- 7 (off-diagonal part ~ +-2 sqrt(80/nb)); take a safe interval
    lo, hi = c - 12.0, c + 12.0
    X, name = _gpu(dims, A, B, dtype, lo, hi, order)
    ref = cheby_oracle.cheby_apply(dims, A, B, lo, hi, order)
    assert rel_err_cols(X, ref) <= TOL[dtype], (name, rel_err_cols(X, ref))


@pytest.mark.parametrize("dims,nb,s,dtype", [((4, 4, 4, 4), 8, 4, "c128"), ((4, 4, 2, 2), 32, 16, "c64")])
def test_cheby_order_120_on_an_ill_conditioned_operator(dims, nb, s, dtype):
    # the paper's coarse solve is P^Cheby of order 120 on an eigenspan of ratio 2000 ([0.02, 40]); here: the
    # stress operator (kappa ~ 100, no dominant diagonal), [lo, hi] = [0.9 lambda_min, 1.1 lambda_max], order 120 = 119 applications
    from helpers import stress_operator
    from inputs import synth
    A, c, lmin, lmax = stress_operator(dims, nb, 123, 0.02)
    B = synth.make_block(dims, nb, s, 123, synth.TAG_B)
    lo, hi = 0.9 * lmin, 1.1 * lmax
    X, name = _gpu(dims, A, B, dtype, lo, hi, 120)
    ref = cheby_oracle.cheby_apply(dims, A, B, lo, hi, 120)
    err = rel_err_cols(X, ref)
    # the apply's own error on this operator (no dominant diagonal), measured here against the oracle
    Xv = synth.make_block(dims, nb, s, 124, synth.TAG_X)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    e_apply = rel_err_cols(to_np(op.apply(to_dev(Xv, dtype))), oracle.apply(dims, A, Xv))
    op.close()
    kappa = lmax / lmin
    print(f"cheby order 120 {dtype}: kernel={name} kappa={kappa:.0f} e_apply={e_apply:.2e} err={err:.2e}")
    assert e_apply <= TOL[dtype]
    # P approximates 1/x: a perturbed operator H~ = H + E, ||E|| <= e ||H||, moves P(H) B by ~ kappa e relative (d(1/x) = -dx/x^2);
    # the tensor kernels' error is systematic (FP32 accumulator truncation), so it does not average out over the 119 applications:
    # bar = 2 kappa e_apply with e_apply measured above (and never below the apply's own bar)
    assert err <= max(TOL[dtype], 2.0 * kappa * e_apply), (name, err, e_apply)
    # and the polynomial is the approximate inverse it should be: ||B - H X|| <= ||B|| / |T_n(y(0))| + rounding
    R = B - oracle.apply(dims, A, X)
    y0 = (hi + lo) / (hi - lo)
    bound = 1.0 / np.cosh(120 * np.arccosh(y0))
    rel = np.linalg.norm(R.reshape(-1, s), axis=0) / np.linalg.norm(B.reshape(-1, s), axis=0)
    # (complex64: plus ||H (X - X_oracle)|| <= lambda_max ||X - X_oracle||, the part of the residual the perturbed operator explains)
    dx = np.linalg.norm((X - ref).reshape(-1, s), axis=0) / np.linalg.norm(B.reshape(-1, s), axis=0)
    assert np.all(rel <= bound + (1e-12 if dtype == "c128" else lmax * dx + 1e-7)), (rel.max(), bound)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_cheby_apply_is_an_approximate_inverse(dtype):
    # property that holds at any size: ||B - H P(H) B|| <= ||B|| / |T_n(y(0))| (+ rounding) when spec(H) is inside [lo, hi]
    dims, nb, s, order = (4, 4, 4, 6), 32, 16, 10
    A, c, _, B = host_case(dims, nb, s, seed=9, factor=1.02)
    lo, hi = c - 12.0, c + 12.0
    X, _ = _gpu(dims, A, B, dtype, lo, hi, order)
    R = B - oracle.apply(dims, A, X)
    y0 = (hi + lo) / (hi - lo)
    bound = 1.0 / np.cosh(order * np.arccosh(y0))
    floor = 1e-13 if dtype == "c128" else 5e-7
    rel = np.linalg.norm(R.reshape(-1, s), axis=0) / np.linalg.norm(B.reshape(-1, s), axis=0)
    assert np.all(rel <= bound + floor), (rel.max(), bound)


def test_cheby_apply_rejects_bad_arguments():
    dims, nb, s = (2, 2, 2, 2), 8, 4
    A, c, _, B = host_case(dims, nb, s, seed=1, factor=1.05)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), s)
    Bd = to_dev(B, "c128")
    for lo, hi, order in [(0.0, 1.0, 4), (2.0, 1.0, 4), (1.0, 2.0, 0), (-1.0, 2.0, 3)]:
        with pytest.raises(cm.binding.CoarseError) as ei:
            op.cheby_apply(Bd, lo, hi, order)
        assert ei.value.status == cm.binding.INVALID_ARG
    with pytest.raises(cm.binding.CoarseError):
        op.cheby_apply(Bd, 1.0, 2.0, 4, X=Bd)
    op.close()


# ---- deflation and the composite Defl + Cheby solve (Eq. 7-12) -------------------------------------------------
def _eigenpairs(dims, nb, seed, nev):
    """lowest nev eigenpairs of the synthetic operator from a dense eigendecomposition of the brute-force matrix (tiny lattices)."""
    from helpers import dense_matrix
    from inputs import synth
    A, c = synth.make_operator(dims, nb, seed, 1.05)
    lam, U = np.linalg.eigh(dense_matrix(dims, A.astype(np.complex128)))
    return A, lam, U[:, :nev].copy(), lam[:nev].copy()


@pytest.mark.parametrize("dims,nb,s,nev,dtype", [((2, 2, 2, 2), 8, 4, 6, "c128"), ((2, 2, 2, 3), 8, 16, 16, "c64"),
                                                 ((2, 2, 2, 2), 4, 5, 3, "c128"), ((2, 2, 2, 2), 8, 64, 33, "c64")])
def test_deflate_matches_oracle(dims, nb, s, nev, dtype):
    from inputs import synth
    A, lam_all, Vev, lam = _eigenpairs(dims, nb, 31, nev)
    B = synth.make_block(dims, nb, s, 31, synth.TAG_B)
    n = B.shape[0] * B.shape[1]
    Vq = Vev.astype(np.complex64).astype(np.complex128) if dtype == "c64" else Vev       # what the device sees
    q_ref, perp_ref = cheby_oracle.deflate(Vq, lam, B.reshape(n, s))
    op = cm.CoarseOperator(dims, to_dev(A, dtype), max(s, nev))
    q, perp = op.deflate(to_dev(Vev, dtype), lam, to_dev(B, dtype))
    op.close()
    tol = 1e-12 if dtype == "c128" else 2e-6
    assert rel_err_cols(to_np(q).reshape(n, 1, s), q_ref.reshape(n, 1, s)) <= tol
    assert rel_err_cols(to_np(perp).reshape(n, 1, s), perp_ref.reshape(n, 1, s)) <= tol


@pytest.mark.parametrize("dims,nb,s,nev,nrhs_max,dtype", [((2, 2, 2, 4), 16, 12, 192, 12, "c128"),      # 16 chunks of 12 eigenvectors
                                                          ((4, 2, 2, 4), 8, 16, 200, 64, "c64"),         # chunks 64, 64, 64, 8
                                                          ((2, 2, 2, 4), 16, 5, 65, 64, "c128"),         # 64 + 1
                                                          ((2, 2, 2, 4), 16, 32, 128, 32, "c64"),        # wide blocks: 4 rows per thread in stage 2
                                                          ((2, 2, 2, 4), 16, 64, 96, 64, "c64")])        # chunks 64, 32 at width 64
def test_deflate_with_hundreds_of_eigenvectors(dims, nb, s, nev, nrhs_max, dtype):
    # the paper deflates the coarse solve with "several hundred" eigenvectors (192 in its production runs, up to 1000 computed:
    # PAPER.md:118, 196, 384-388): more than one chunk of <= min(64, nrhs_max) vectors, in place as well (Bperp aliases B)
    from inputs import synth
    A, lam_all, Vev, lam = _eigenpairs(dims, nb, 35, nev)
    B = synth.make_block(dims, nb, s, 35, synth.TAG_B)
    n = B.shape[0] * B.shape[1]
    assert n >= 512 and nev > 64
    Vq = Vev.astype(np.complex64).astype(np.complex128) if dtype == "c64" else Vev
    q_ref, perp_ref = cheby_oracle.deflate(Vq, lam, B.reshape(n, s))
    op = cm.CoarseOperator(dims, to_dev(A, dtype), nrhs_max)
    Vd, Bd = to_dev(Vev, dtype), to_dev(B, dtype)
    q, perp = op.deflate(Vd, lam, Bd)
    tol = 1e-12 if dtype == "c128" else 2e-6
    assert rel_err_cols(to_np(q).reshape(n, 1, s), q_ref.reshape(n, 1, s)) <= tol
    assert rel_err_cols(to_np(perp).reshape(n, 1, s), perp_ref.reshape(n, 1, s)) <= tol
    # projector identities on the device result: V^H b_perp = 0, b_perp + V V^H b = b
    assert np.abs(Vq.conj().T @ to_np(perp).reshape(n, s)).max() <= (1e-12 if dtype == "c128" else 3e-6)
    q2 = torch.empty_like(Bd)
    lam_c = (cm.binding.C.c_double * nev)(*[float(x) for x in lam])
    st = cm.lib().coarse_deflate(op._h, Vd.data_ptr(), lam_c, nev, Bd.data_ptr(), q2.data_ptr(), Bd.data_ptr(), s, None)
    torch.cuda.synchronize()
    op.close()
    assert st == 0
    assert torch.equal(q2, q) and torch.equal(Bd, perp)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_deflate_in_place_Bperp_aliases_B(dtype):
    # coarse_mrhs.h: "Bperp may alias B" -- the projection written over its own input
    from inputs import synth
    dims, nb, s, nev = (2, 2, 2, 2), 8, 8, 5
    A, lam_all, Vev, lam = _eigenpairs(dims, nb, 33, nev)
    B = synth.make_block(dims, nb, s, 33, synth.TAG_B)
    n = B.shape[0] * B.shape[1]
    Vq = Vev.astype(np.complex64).astype(np.complex128) if dtype == "c64" else Vev
    q_ref, perp_ref = cheby_oracle.deflate(Vq, lam, B.reshape(n, s))
    op = cm.CoarseOperator(dims, to_dev(A, dtype), max(s, nev))
    Bd, Vd = to_dev(B, dtype), to_dev(Vev, dtype)
    q = torch.empty_like(Bd)
    lam_c = (cm.binding.C.c_double * nev)(*[float(x) for x in lam])
    st = cm.lib().coarse_deflate(op._h, Vd.data_ptr(), lam_c, nev, Bd.data_ptr(), q.data_ptr(), Bd.data_ptr(), s, None)
    torch.cuda.synchronize()
    op.close()
    assert st == 0
    tol = 1e-12 if dtype == "c128" else 2e-6
    assert rel_err_cols(to_np(q).reshape(n, 1, s), q_ref.reshape(n, 1, s)) <= tol
    assert rel_err_cols(to_np(Bd).reshape(n, 1, s), perp_ref.reshape(n, 1, s)) <= tol


@pytest.mark.parametrize("dims,nb,s,nev,order,dtype", [((2, 2, 2, 2), 8, 4, 6, 10, "c128"), ((2, 2, 2, 3), 8, 16, 12, 8, "c64")])
def test_cheby_defl_solve_matches_oracle(dims, nb, s, nev, order, dtype):
    from inputs import synth
    A, lam_all, Vev, lam = _eigenpairs(dims, nb, 32, nev)
    B = synth.make_block(dims, nb, s, 32, synth.TAG_B)
    lo, hi = 0.95 * lam_all[nev], 1.05 * lam_all[-1]
    Vq = Vev.astype(np.complex64).astype(np.complex128) if dtype == "c64" else Vev
    ref = cheby_oracle.cheby_defl_solve(dims, A, Vq, lam, B, lo, hi, order)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), max(s, nev))
    X = to_np(op.cheby_defl_solve(to_dev(Vev, dtype), lam, to_dev(B, dtype), lo, hi, order))
    with pytest.raises(cm.binding.CoarseError):
        op.cheby_defl_solve(to_dev(Vev, dtype), -lam, to_dev(B, dtype), lo, hi, order)          # non-positive eigenvalues
    op.close()
    assert rel_err_cols(X, ref) <= TOL[dtype]
