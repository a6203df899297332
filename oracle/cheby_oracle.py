"""CPU oracle for the Chebyshev polynomial coarse solve, plain numpy, complex128.

TEST INFRASTRUCTURE ONLY (tests/ and bench legs may import it; the CUDA package does not, and this file does not
import the CUDA package).

What it computes (section 2.3): the coarse solve "replaced ... with a ... Chebyshev approximation to
1/x over eigenspan [lo, hi]", "with coefficients chose[n] according to the usual Chebyshev approximation obtained by
determining coefficients at the Chebyshev interpolation points from the target function 1/x", tuned parameters
[lo, hi, order] ([0.02, 40, 120] for the coarse solve, [2.0, 92.0] order 8 for the smoother).

Reading taken (R16): "order" n = number of coefficients (polynomial degree n - 1), the "usual"
approximation is interpolation at the n first-kind Chebyshev points of [lo, hi] (Numerical-Recipes form):
    y(x)  = (2 x - hi - lo) / (hi - lo)                               maps [lo, hi] to [-1, 1]
    x_k   = (hi + lo)/2 + (hi - lo)/2 * cos(pi (k + 1/2) / n),         k = 0 .. n-1
    c_j   = (2/n) sum_k (1 / x_k) cos(pi j (k + 1/2) / n),             j = 0 .. n-1
    P(x)  = c_0 / 2 + sum_{j=1}^{n-1} c_j T_j(y(x))
and P(H) B is evaluated with the three-term recurrence T_{j+1} = 2 y T_j - T_{j-1} applied to blocks, one operator
application per term, in this order, no reordering:
    T_0 = B ;  T_1 = y(H) B ;  X = (c_0/2) T_0 + c_1 T_1 ;  T_{j+1} = 2 y(H) T_j - T_{j-1} ;  X += c_{j+1} T_{j+1}.
Pins: tests/test_oracle_cheby.py (numpy.polynomial.chebyshev interpolation of 1/x evaluated on the eigenvalues of a
dense H; the closed-form error bound of the interpolant; order 1 and 2 by hand).
"""
from __future__ import annotations

import numpy as np

from . import oracle


def coefficients(lo: float, hi: float, order: int) -> np.ndarray:
    """c_j, j = 0 .. order-1, of the interpolant of 1/x at the first-kind Chebyshev points of [lo, hi]."""
    n = int(order)
    c = np.zeros(n, dtype=np.float64)
    for j in range(n):
        acc = 0.0
        for k in range(n):
            xk = 0.5 * (hi + lo) + 0.5 * (hi - lo) * np.cos(np.pi * (k + 0.5) / n)
            acc += (1.0 / xk) * np.cos(np.pi * j * (k + 0.5) / n)
        c[j] = 2.0 * acc / n
    return c


def scalar_polynomial(x, lo: float, hi: float, order: int):
    """P(x) for real x (array), by the same recurrence on scalars."""
    c = coefficients(lo, hi, order)
    x = np.asarray(x, dtype=np.float64)
    y = (2.0 * x - hi - lo) / (hi - lo)
    t_prev, t_cur = np.ones_like(y), y
    out = 0.5 * c[0] * t_prev
    if order > 1:
        out = out + c[1] * t_cur
    for j in range(1, order - 1):
        t_next = 2.0 * y * t_cur - t_prev
        out = out + c[j + 1] * t_next
        t_prev, t_cur = t_cur, t_next
    return out


def cheby_apply(dims, A, B, lo: float, hi: float, order: int) -> np.ndarray:
    """X = P(H) B for a block B [V][nb][s] (complex128); order - 1 applications of the coarse operator."""
    c = coefficients(lo, hi, order)
    B = np.ascontiguousarray(B, dtype=np.complex128)
    alpha, beta = 2.0 / (hi - lo), -(hi + lo) / (hi - lo)         # y(H) = alpha H + beta
    t_prev = B
    X = 0.5 * c[0] * t_prev
    if order == 1:
        return X
    t_cur = alpha * oracle.apply(dims, A, t_prev) + beta * t_prev
    X = X + c[1] * t_cur
    for j in range(1, order - 1):
        t_next = 2.0 * (alpha * oracle.apply(dims, A, t_cur) + beta * t_cur) - t_prev
        X = X + c[j + 1] * t_next
        t_prev, t_cur = t_cur, t_next
    return X


# ---- multi-RHS deflation and the composite "Defl + Cheby" coarse solve (Eq. 7-12) ----
# Definitions written out (complex128): with the n_ev lowest eigenpairs (|i>, lambda_i) of H as columns of Vev [n][nev],
#   b_par  = (sum_i |i><i|) b                      (Eq. 8)
#   b_perp = (1 - sum_i |i><i|) b                  (Eq. 9)
#   Q b_par = (sum_i |i><i| / lambda_i) b          (Eq. 10)
#   Q^{Cheby+defl} b = Defl(b_par) + P^{Cheby}(b_perp)     (Eq. 12)
# applied to a block of right-hand sides at once (two tall-skinny products).
# Pins: tests/test_oracle_cheby.py (full basis => H^-1 b by numpy.linalg.solve; b_par + b_perp = b; V^H b_perp = 0;
# Eq. 11's diagonal form through a dense eigendecomposition).

def deflate(Vev, lam, B):
    """Vev [n][nev] (orthonormal columns), lam [nev], B [n][s]  ->  (Q b_par, b_perp), both [n][s]."""
    Vev = np.asarray(Vev, dtype=np.complex128)
    B = np.asarray(B, dtype=np.complex128)
    C = Vev.conj().T @ B                                  # <i|b>
    b_par = Vev @ C
    b_perp = B - b_par
    q_b_par = Vev @ (C / np.asarray(lam, dtype=np.float64)[:, None])
    return q_b_par, b_perp


def cheby_defl_solve(dims, A, Vev, lam, B, lo: float, hi: float, order: int) -> np.ndarray:
    """Eq. 12 on a block B [V][nb][s]; Vev [V*nb][nev]."""
    shape = B.shape
    n, s = shape[0] * shape[1], shape[2]
    q_b_par, b_perp = deflate(Vev, lam, np.asarray(B, dtype=np.complex128).reshape(n, s))
    return q_b_par.reshape(shape) + cheby_apply(dims, A, b_perp.reshape(shape), lo, hi, order)
