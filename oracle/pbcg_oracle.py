"""CPU oracle for Preconditioned BlockCGrQ, plain numpy, complex128.

TEST INFRASTRUCTURE ONLY (tests/ may import it; the CUDA package does not, and this file does not import the CUDA package).

Follows Fig. 2 (right) of the paper statement by statement, lower case = unpreconditioned vectors,
upper case = preconditioned ones, M^-1 a Hermitian positive definite STATIONARY preconditioner (the
Chebyshev / deflated-Chebyshev polynomial of the coarse operator):
    z_0 = B - H X_0 ;  Z_0 = M^-1 z_0
    C_0^H C_0 = Z_0^H z_0 = <Z_0|Z_0>_M                    (Cholesky, C_0 upper triangular, real positive diagonal)
    q_0 = z_0 C_0^-1 ;  Q_0 = Z_0 C_0^-1 ;  D_0 = Q_0
    for k = 0, 1, ...:
        z_k = H D_k ;  Z_k = M^-1 z_k
        N_k = [D_k^H z_k]^-1
        X_{k+1} = X_k + D_k N_k C_k                         (*)
        t_k = q_k - z_k N_k ;  T_k = Q_k - Z_k N_k
        S^H S = T_k^H t_k = <T|T>_M                         (Cholesky)                                     (**)
        q_{k+1} = t_k S^-1 ;  Q_{k+1} = T_k S^-1
        D_{k+1} = Q_{k+1} + D_k S^H
        C_{k+1} = S C_k
Readings: (*) the printed update "X + D_k N_k" lacks the factor C_k exactly as in the unpreconditioned
listing (R1): with r_k = q_k C_k the residual recurrence only closes with it.  (**) the printed line "S_k^dagger S_{k+1} =
T_k^dagger . t_k" and the mixed indices S_k / S_{k+1} are read as ONE factor S per iteration, S^H S = T^H t (R2).
Stop test (the paper gives none, R17): the Euclidean residual is r_k = q_k C_k, so ||r_k[:,r]||^2 = (C^H (q^H q) C)_rr -- one
extra Gram product q^H q per iteration; stop when max_r ||r_k[:,r]|| / ||B[:,r]|| <= tol.
Gram matrices are symmetrised, (G + G^H)/2, before factoring (as in the unpreconditioned oracle).
Pins: tests/test_oracle_pbcg.py.
"""
from __future__ import annotations

import numpy as np

from . import oracle


def _chol_upper(G):
    G = 0.5 * (G + G.conj().T)
    return np.linalg.cholesky(G).conj().T          # numpy returns lower L with G = L L^H;  upper factor = L^H


def pblock_cg(dims, A, B, Minv, X0=None, tol: float = 1e-10, maxiter: int = 200, callback=None):
    """Returns dict(X, iterations, status (0 / -5 not converged), history [k][s] relative residuals, true_rel [s])."""
    B = np.ascontiguousarray(B, dtype=np.complex128)
    shape = B.shape
    n, s = shape[0] * shape[1], shape[2]
    flat = lambda Y: Y.reshape(n, s)
    H = lambda Y: oracle.apply(dims, A, np.ascontiguousarray(Y.reshape(shape))).reshape(n, s)
    Mi = lambda Y: np.asarray(Minv(np.ascontiguousarray(Y.reshape(shape))), dtype=np.complex128).reshape(n, s)
    b = flat(B)
    bnorm = np.linalg.norm(b, axis=0)
    bnorm[bnorm == 0] = 1.0
    X = np.zeros((n, s), dtype=np.complex128) if X0 is None else flat(np.array(X0, dtype=np.complex128)).copy()
    z = b - H(X)
    history = [np.linalg.norm(z, axis=0) / bnorm]
    status, its = -5, 0
    if history[0].max() <= tol:
        status = 0
    else:
        Z = Mi(z)
        C = _chol_upper(Z.conj().T @ z)
        Cinv = np.linalg.inv(C)
        q, Q = z @ Cinv, Z @ Cinv
        D = Q.copy()
        for k in range(maxiter):
            zk = H(D)
            Zk = Mi(zk)
            G = D.conj().T @ zk
            N = np.linalg.inv(0.5 * (G + G.conj().T))
            X = X + D @ (N @ C)
            t, T = q - zk @ N, Q - Zk @ N
            S = _chol_upper(T.conj().T @ t)
            Sinv = np.linalg.inv(S)
            q, Q = t @ Sinv, T @ Sinv
            D = Q + D @ S.conj().T
            C = S @ C
            its = k + 1
            Gq = q.conj().T @ q
            rel = np.sqrt(np.maximum(np.real(np.einsum("ar,ab,br->r", C.conj(), Gq, C)), 0.0)) / bnorm
            history.append(rel)
            if callback is not None:
                callback(its, dict(X=X.reshape(shape), q=q, Q=Q, D=D, C=C))
            if rel.max() <= tol:
                status = 0
                break
    true_rel = np.linalg.norm(b - H(X), axis=0) / bnorm
    return dict(X=X.reshape(shape), iterations=its, status=status, history=np.array(history), true_rel=true_rel)
