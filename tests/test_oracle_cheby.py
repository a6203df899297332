"""Pins of the Chebyshev coarse-solve oracle (oracle/cheby_oracle.py) against things other than itself:
 * numpy.polynomial.chebyshev.chebinterpolate / chebval (a library routine) for the coefficients and for P on the spectrum;
 * the closed form of the interpolation error of 1/x:  1 - x P(x) = T_n(y(x)) / T_n(y(0))  (degree-n polynomial that vanishes
   at the n nodes and equals 1 at x = 0), for any x;
 * P(H) B through a dense eigendecomposition of the brute-force matrix of a tiny lattice;
 * orders 1 and 2 worked by hand; the residual bound ||B - H P(H) B|| <= ||B|| / |T_n(y(0))| when spec(H) is inside [lo, hi].
"""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

from helpers import dense_matrix, rel_err_cols
from inputs import synth
from oracle import cheby_oracle


def _T(n, y):
    y = np.asarray(y, dtype=np.float64)
    out = np.empty_like(y)
    inside = np.abs(y) <= 1
    out[inside] = np.cos(n * np.arccos(y[inside]))
    yo = y[~inside]
    out[~inside] = np.sign(yo) ** n * np.cosh(n * np.arccosh(np.abs(yo)))
    return out


@pytest.mark.parametrize("lo,hi,order", [(0.02, 40.0, 120), (2.0, 92.0, 8), (70.0, 95.0, 12), (1.0, 3.0, 1), (0.5, 7.0, 2)])
def test_coefficients_equal_numpy_chebinterpolate(lo, hi, order):
    c = cheby_oracle.coefficients(lo, hi, order)
    a = npcheb.chebinterpolate(lambda y: 1.0 / (0.5 * (hi + lo) + 0.5 * (hi - lo) * y), order - 1)
    ours = c.copy()
    ours[0] *= 0.5
    assert np.allclose(ours, a, rtol=1e-9, atol=1e-12 * np.abs(a).max())


@pytest.mark.parametrize("lo,hi,order", [(0.02, 40.0, 120), (2.0, 92.0, 8), (70.0, 95.0, 12), (0.5, 7.0, 2)])
def test_error_closed_form_one_minus_xP_is_Tn_ratio(lo, hi, order):
    rng = np.random.default_rng(order)
    x = np.concatenate([rng.uniform(lo, hi, 200), rng.uniform(0.3 * lo, lo, 20), rng.uniform(hi, 1.1 * hi, 20)])
    y = (2 * x - hi - lo) / (hi - lo)
    y0 = -(hi + lo) / (hi - lo)
    expect = _T(order, y) / _T(order, np.array([y0]))[0]
    got = 1.0 - x * cheby_oracle.scalar_polynomial(x, lo, hi, order)
    inside = (x >= lo) & (x <= hi)
    # inside [lo, hi] |T_j| <= 1: float64 rounding of 1 - x P(x) only; outside, T_j(y) amplifies the rounding of the c_j
    assert np.allclose(got[inside], expect[inside], rtol=1e-7, atol=2e-13)
    assert np.allclose(got[~inside], expect[~inside], rtol=5e-3, atol=2e-13)


def test_orders_one_and_two_by_hand():
    lo, hi = 1.0, 3.0
    x = np.array([0.7, 1.0, 2.0, 2.9])
    assert np.allclose(cheby_oracle.scalar_polynomial(x, lo, hi, 1), 0.5)          # constant 1 / midpoint
    n0, n1 = 2.0 + np.cos(np.pi / 4), 2.0 + np.cos(3 * np.pi / 4)                    # the two nodes
    line = 1 / n0 + (x - n0) * (1 / n1 - 1 / n0) / (n1 - n0)
    assert np.allclose(cheby_oracle.scalar_polynomial(x, lo, hi, 2), line, rtol=1e-13)


@pytest.mark.parametrize("dims,nb,s,order", [((2, 2, 2, 2), 4, 3, 9), ((2, 3, 1, 2), 6, 2, 16), ((3, 2, 2, 2), 5, 4, 2)])
def test_block_polynomial_equals_dense_eigendecomposition(dims, nb, s, order):
    A, c = synth.make_operator(dims, nb, 11, 1.05)
    B = synth.make_block(dims, nb, s, 11, synth.TAG_B)
    H = dense_matrix(dims, A.astype(np.complex128))
    lam, U = np.linalg.eigh(H)
    lo, hi = 0.9 * lam[0], 1.1 * lam[-1]
    a = npcheb.chebinterpolate(lambda y: 1.0 / (0.5 * (hi + lo) + 0.5 * (hi - lo) * y), order - 1)
    p_lam = npcheb.chebval((2 * lam - hi - lo) / (hi - lo), a)
    n = H.shape[0]
    ref = (U * p_lam) @ (U.conj().T @ B.reshape(n, s))
    X = cheby_oracle.cheby_apply(dims, A, B, lo, hi, order)
    assert rel_err_cols(X.reshape(n, 1, s), ref.reshape(n, 1, s)) <= 1e-12
    # residual bound: ||B - H X|| <= ||B|| / |T_n(y(0))| column by column (spectrum inside [lo, hi])
    y0 = -(hi + lo) / (hi - lo)
    bound = 1.0 / abs(_T(order, np.array([y0]))[0])
    R = B.reshape(n, s) - H @ X.reshape(n, s)
    assert np.all(np.linalg.norm(R, axis=0) <= (1 + 1e-9) * bound * np.linalg.norm(B.reshape(n, s), axis=0) + 1e-13)


def test_columns_are_independent_and_map_is_linear():
    dims, nb, s = (2, 2, 2, 3), 4, 3
    A, c = synth.make_operator(dims, nb, 5, 1.05)
    B = synth.make_block(dims, nb, s, 5, synth.TAG_B)
    lo, hi, order = 0.8 * c, 1.3 * c, 7
    X = cheby_oracle.cheby_apply(dims, A, B, lo, hi, order)
    for r in range(s):
        Xr = cheby_oracle.cheby_apply(dims, A, B[:, :, r:r + 1], lo, hi, order)
        assert np.allclose(Xr[:, :, 0], X[:, :, r], rtol=1e-13, atol=1e-15)
    X2 = cheby_oracle.cheby_apply(dims, A, (2 - 1j) * B, lo, hi, order)
    assert np.allclose(X2, (2 - 1j) * X, rtol=1e-13, atol=1e-15)


# ---- deflation and the composite solve (Eq. 7-12) ------------------------------------------------------------
def _tiny_eigensystem(dims=(2, 2, 2, 2), nb=4, seed=13):
    A, c = synth.make_operator(dims, nb, seed, 1.05)
    H = dense_matrix(dims, A.astype(np.complex128))
    lam, U = np.linalg.eigh(H)
    return A, H, lam, U


def test_deflation_with_the_full_basis_is_the_inverse():
    A, H, lam, U = _tiny_eigensystem()
    rng = np.random.default_rng(0)
    B = rng.standard_normal((H.shape[0], 3)) + 1j * rng.standard_normal((H.shape[0], 3))
    q, perp = cheby_oracle.deflate(U, lam, B)
    assert np.allclose(q, np.linalg.solve(H, B), rtol=1e-11, atol=1e-13)
    assert np.linalg.norm(perp) <= 1e-12 * np.linalg.norm(B)


@pytest.mark.parametrize("nev", [1, 5, 16])
def test_deflation_splits_the_source(nev):
    A, H, lam, U = _tiny_eigensystem()
    rng = np.random.default_rng(nev)
    B = rng.standard_normal((H.shape[0], 4)) + 1j * rng.standard_normal((H.shape[0], 4))
    V = U[:, :nev]
    q, perp = cheby_oracle.deflate(V, lam[:nev], B)
    assert np.linalg.norm(V.conj().T @ perp) <= 1e-12 * np.linalg.norm(B)            # b_perp is orthogonal to the space
    assert np.allclose(H @ q + perp, B, rtol=1e-11, atol=1e-12)                       # H Q b_par = b_par, b_par + b_perp = b
    q2, perp2 = cheby_oracle.deflate(V, lam[:nev], perp)                              # projecting twice changes nothing
    assert np.linalg.norm(q2) <= 1e-12 * np.linalg.norm(B) and np.allclose(perp2, perp, atol=1e-12)


@pytest.mark.parametrize("nev,order", [(4, 6), (10, 12)])
def test_composite_solve_is_diagonal_in_the_eigenbasis(nev, order):
    # Eq. 11: Q = diag(1/lambda_1 .. 1/lambda_nev, P(lambda_nev+1) .. P(lambda_max)) in the eigenbasis
    dims, nb, s = (2, 2, 2, 2), 4, 3
    A, H, lam, U = _tiny_eigensystem(dims, nb)
    B = synth.make_block(dims, nb, s, 3, synth.TAG_B)
    lo, hi = 0.9 * lam[nev], 1.1 * lam[-1]
    a = npcheb.chebinterpolate(lambda y: 1.0 / (0.5 * (hi + lo) + 0.5 * (hi - lo) * y), order - 1)
    qdiag = npcheb.chebval((2 * lam - hi - lo) / (hi - lo), a)
    qdiag[:nev] = 1.0 / lam[:nev]
    n = H.shape[0]
    ref = (U * qdiag) @ (U.conj().T @ B.reshape(n, s))
    X = cheby_oracle.cheby_defl_solve(dims, A, U[:, :nev], lam[:nev], B, lo, hi, order)
    assert rel_err_cols(X.reshape(n, 1, s), ref.reshape(n, 1, s)) <= 1e-11
