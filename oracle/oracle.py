"""ctypes loader and numpy-facing wrappers for the C oracle (oracle/coarse_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  It does not import the CUDA package and the CUDA package does not import it.
This file does argument marshalling only; every number is computed in coarse_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "coarse_oracle.c"
_LIB = _HERE / "libcoarse_oracle.so"

OK, NOT_CONVERGED, BREAKDOWN = 0, -5, -6
A_C64, A_C128 = 0, 1

_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, OpenMP).  -ffp-contract=off: no fused multiply-adds, so the
    arithmetic is exactly the loop nests as written."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", str(_LIB), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_CB = C.CFUNCTYPE(None, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.oracle_num_threads.restype = C.c_int
        L.oracle_neighbour.restype = C.c_int64
        L.oracle_neighbour.argtypes = [C.c_void_p, C.c_int64, C.c_int32]
        L.oracle_apply_sites.restype = None
        L.oracle_apply_sites.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                         C.c_void_p, C.c_int64, C.c_void_p, C.c_int32]
        L.oracle_gram.restype = None
        L.oracle_gram.argtypes = [C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.oracle_cholesky_upper.restype = C.c_int
        L.oracle_cholesky_upper.argtypes = [C.c_int32, C.c_void_p, C.c_void_p]
        L.oracle_upper_inverse.restype = None
        L.oracle_upper_inverse.argtypes = [C.c_int32, C.c_void_p, C.c_void_p]
        L.oracle_hpd_inverse.restype = C.c_int
        L.oracle_hpd_inverse.argtypes = [C.c_int32, C.c_void_p, C.c_void_p]
        L.oracle_block_rotate.restype = None
        L.oracle_block_rotate.argtypes = [C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.oracle_block_cg.restype = C.c_int
        L.oracle_block_cg.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_double, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                      _CB, C.c_void_p]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _dims(dims):
    return np.ascontiguousarray(np.asarray(dims, dtype=np.int32))


def _a_arg(A):
    A = np.ascontiguousarray(A)
    if A.dtype == np.complex64:
        return A, A_C64
    if A.dtype == np.complex128:
        return A, A_C128
    raise TypeError("A must be complex64 or complex128")


def _z(x):
    return np.ascontiguousarray(x, dtype=np.complex128)


def neighbour(dims, x: int, p: int) -> int:
    d = _dims(dims)
    return int(lib().oracle_neighbour(d.ctypes.data, int(x), int(p)))


def apply(dims, A, X, sites=None, p_only: int = -1) -> np.ndarray:
    """Y = H X (Eq. 19 summed over the 81 points).  A: [n_sites][81][nb][nb] for the listed sites
    (all sites if sites is None); X: [V][nb][s]; returns [n_sites][nb][s] complex128."""
    d = _dims(dims)
    A, adt = _a_arg(A)
    X = _z(X)
    nb, s = X.shape[1], X.shape[2]
    n_sites = A.shape[0]
    assert A.shape[1:] == (81, nb, nb)
    if sites is None:
        assert n_sites == X.shape[0]
        sp = None
    else:
        sites = np.ascontiguousarray(sites, dtype=np.int64)
        assert len(sites) == n_sites
        sp = sites.ctypes.data
    Y = np.empty((n_sites, nb, s), dtype=np.complex128)
    lib().oracle_apply_sites(d.ctypes.data, nb, s, adt, A.ctypes.data, X.ctypes.data, Y.ctypes.data,
                             n_sites, sp, int(p_only))
    return Y


def gram(U, W) -> np.ndarray:
    U, W = _z(U), _z(W)
    s = U.shape[-1]
    n = U.size // s
    G = np.empty((s, s), dtype=np.complex128)
    lib().oracle_gram(n, s, U.ctypes.data, W.ctypes.data, G.ctypes.data)
    return G


def cholesky_upper(G):
    G = _z(G)
    s = G.shape[0]
    S = np.empty((s, s), dtype=np.complex128)
    st = lib().oracle_cholesky_upper(s, G.ctypes.data, S.ctypes.data)
    return st, S


def upper_inverse(S) -> np.ndarray:
    S = _z(S)
    s = S.shape[0]
    out = np.empty((s, s), dtype=np.complex128)
    lib().oracle_upper_inverse(s, S.ctypes.data, out.ctypes.data)
    return out


def hpd_inverse(G):
    G = _z(G)
    s = G.shape[0]
    out = np.empty((s, s), dtype=np.complex128)
    st = lib().oracle_hpd_inverse(s, G.ctypes.data, out.ctypes.data)
    return st, out


def block_rotate(U, K, W, beta: float) -> np.ndarray:
    """returns beta*W + U K (a new array); U, W: [...][s], K: [s][s]."""
    U, K = _z(U), _z(K)
    out = _z(W).copy()
    s = U.shape[-1]
    lib().oracle_block_rotate(U.size // s, s, U.ctypes.data, K.ctypes.data, float(beta), out.ctypes.data)
    return out


def block_cg(dims, A, B, X0=None, tol: float = 1e-10, maxiter: int = 1000, callback=None):
    """BlockCGrQ (Fig. 2 left).  Returns dict(X, iterations, status, history[(its+1), s], true_rel[s]).
    callback(k, X, Q, D, C) receives numpy views valid only during the call."""
    d = _dims(dims)
    A, adt = _a_arg(A)
    B = _z(B)
    V, nb, s = B.shape
    X = np.zeros_like(B) if X0 is None else _z(X0).copy()
    its = C.c_int32(0)
    hist = np.full((maxiter + 1, s), np.nan, dtype=np.float64)
    true_rel = np.empty(s, dtype=np.float64)

    def _view(ptr, shape):
        n = int(np.prod(shape))
        buf = (C.c_double * (2 * n)).from_address(ptr)
        return np.frombuffer(buf, dtype=np.complex128).reshape(shape)

    if callback is not None:
        def _cb(k, px, pq, pd, pc, _user):
            callback(int(k), _view(px, (V, nb, s)), _view(pq, (V, nb, s)), _view(pd, (V, nb, s)), _view(pc, (s, s)))
        cb = _CB(_cb)
    else:
        cb = _CB()
    st = lib().oracle_block_cg(d.ctypes.data, nb, s, adt, A.ctypes.data, B.ctypes.data, X.ctypes.data,
                               float(tol), int(maxiter), C.byref(its), hist.ctypes.data, true_rel.ctypes.data,
                               cb, None)
    k = its.value
    return dict(X=X, iterations=k, status=int(st), history=hist[:k + 1].copy(), true_rel=true_rel)
