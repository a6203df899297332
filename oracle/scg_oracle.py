"""CPU oracle for the stacked single-Krylov coarse CG (second half), plain numpy, complex128.

TEST INFRASTRUCTURE ONLY.

What it computes (section 2.1): "we find it simplest to treat the coarse solve as an enlarged five
dimensional system with a single Krylov solve, albeit with a block diagonal structure" -- plain conjugate gradients
(Hestenes-Stiefel, PAPER.md ref [52]) on  (I_s (x) H) vec(X) = vec(B), i.e. ONE alpha and ONE beta per iteration from inner
products over all right-hand sides at once (Frobenius inner product <U, W> = sum_r <U[:,r], W[:,r]>):
    R = B - H X ;  P = R ;  rho = <R, R>
    loop:  Z = H P ;  alpha = rho / <P, Z> ;  X += alpha P ;  R -= alpha Z ;  rho' = <R, R> ;
           stop if sqrt(rho') / ||B||_F <= tol ;  beta = rho' / rho ;  P = R + beta P ;  rho = rho'
Reading (R18): the stop quantity of a single Krylov process is the norm of the stacked residual, ||R||_F / ||B||_F
(the paper quotes one tolerance per coarse solve); per-column true residuals are reported as well.
Pins: tests/test_oracle_scg.py (scipy.sparse.linalg.cg on the Kronecker system; dense solve; s = 1 equals BlockCGrQ).
"""
from __future__ import annotations

import numpy as np

from . import oracle


def stacked_cg(dims, A, B, X0=None, tol: float = 1e-10, maxiter: int = 1000, callback=None):
    B = np.ascontiguousarray(B, dtype=np.complex128)
    shape = B.shape
    H = lambda Y: oracle.apply(dims, A, np.ascontiguousarray(Y))
    fdot = lambda U, W: float(np.real(np.vdot(U, W)))
    X = np.zeros_like(B) if X0 is None else np.array(X0, dtype=np.complex128)
    bn = np.sqrt(fdot(B, B)) or 1.0
    R = B - H(X)
    rho = fdot(R, R)
    history = [np.sqrt(rho) / bn]
    status, its = -5, 0
    if history[0] <= tol:
        status = 0
    else:
        P = R.copy()
        for k in range(maxiter):
            Z = H(P)
            alpha = rho / fdot(P, Z)
            X = X + alpha * P
            R = R - alpha * Z
            rho_new = fdot(R, R)
            its = k + 1
            history.append(np.sqrt(rho_new) / bn)
            if callback is not None:
                callback(its, X)
            if history[-1] <= tol:
                status = 0
                break
            beta = rho_new / rho
            P = R + beta * P
            rho = rho_new
    s = shape[-1]
    bcol = np.linalg.norm(B.reshape(-1, s), axis=0)
    bcol[bcol == 0] = 1.0
    true_rel = np.linalg.norm((B - H(X)).reshape(-1, s), axis=0) / bcol
    return dict(X=X, iterations=its, status=status, history=np.array(history), true_rel=true_rel)
