"""Thin ctypes binding of the C ABI in include/coarse_mrhs.h -- argument marshalling only.

Every step of the path (neighbour table, stencil-GEMM apply, Gram products, s x s algebra, block
rotations, the BlockCGrQ loop) runs in the CUDA kernels behind the C entry points; nothing here
computes.  PyTorch is used for device memory and streams only.  There is no CPU fallback: if the shared
library is missing or a call fails, a CoarseError is raised.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import torch

from . import build as _build

C64, C128 = 0, 1
OK, INVALID_ARG, UNSUPPORTED, CUDA_ERROR, OUT_OF_MEMORY, NOT_CONVERGED, BREAKDOWN = 0, -1, -2, -3, -4, -5, -6
FLAG_FORCE_GENERIC, FLAG_NO_TENSOR, FLAG_TENSOR_ONLY, FLAG_TF32, FLAG_UNFUSED_LINALG, FLAG_H16X, FLAG_TENSOR_LINALG, FLAG_H16X_WIDE, FLAG_NO_GRAPH = 1, 2, 4, 8, 16, 32, 64, 128, 256
MAX_NRHS, MAX_HISTORY = 64, 256
SOLVE_ZERO_GUESS = 1

EXPORTS = [
    "coarse_op_create", "coarse_op_destroy", "coarse_op_apply", "coarse_op_apply_host", "block_cg_solve",
    "block_cg_solve_host", "block_cg_begin", "block_cg_step", "block_cg_end", "coarse_block_gram", "coarse_small_cholesky", "coarse_small_hpd_inverse",
    "coarse_block_rotate", "coarse_op_fill_synthetic", "coarse_fill_block", "coarse_op_kernel_name",
    "coarse_op_device_bytes", "coarse_launch_count", "coarse_last_error", "coarse_op_profile", "coarse_op_profile_read",
    "coarse_cheby_apply", "coarse_deflate", "coarse_cheby_defl_solve", "pblock_cg_solve", "stacked_cg_solve", "coarse_block_project", "coarse_block_promote",
    "block_cg_solve_ex", "block_cg_solve_host_ex", "coarse_measure_peaks", "coarse_block_gram_noalloc",
]


class CoarseError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"coarse_mrhs status {status}: {msg}")
        self.status = status


class BlockCGResult(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("status", C.c_int32),
                ("rel_res_recursive", C.c_double * MAX_NRHS), ("rel_res_true", C.c_double * MAX_NRHS),
                ("history", C.c_double * MAX_HISTORY), ("seconds", C.c_double)]


class CoarsePrecond(C.Structure):
    _fields_ = [("kind", C.c_int32), ("order", C.c_int32), ("lo", C.c_double), ("hi", C.c_double),
                ("Vev_dev", C.c_void_p), ("lambda_host", C.POINTER(C.c_double)), ("nev", C.c_int32)]


PRECOND_CHEBY, PRECOND_DEFL_CHEBY = 0, 1

_lib = None


def library_path() -> Path:
    return _build.LIB


def lib():
    """Loads libcoarse_mrhs.so (building it with nvcc when the sources are newer).  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        vp, i32, i64, u32, u64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_double
        sig = {
            "coarse_op_create": (C.c_int, [C.POINTER(vp), vp, i32, i32, i32, vp, u32, vp]),
            "coarse_op_destroy": (C.c_int, [vp]),
            "coarse_op_apply": (C.c_int, [vp, vp, vp, i32, vp]),
            "coarse_op_apply_host": (C.c_int, [vp, vp, vp, i32, vp]),
            "block_cg_solve": (C.c_int, [vp, vp, vp, i32, dbl, i32, C.POINTER(BlockCGResult), vp]),
            "block_cg_solve_host": (C.c_int, [vp, vp, vp, i32, dbl, i32, C.POINTER(BlockCGResult), vp]),
            "block_cg_begin": (C.c_int, [vp, vp, vp, i32, dbl, C.POINTER(dbl), vp]),
            "block_cg_step": (C.c_int, [vp, i32, vp]),
            "block_cg_end": (C.c_int, [vp, C.POINTER(BlockCGResult), vp]),
            "coarse_block_gram": (C.c_int, [vp, vp, vp, vp, i64, i32, vp]),
            "coarse_small_cholesky": (C.c_int, [vp, vp, vp, i32, vp, vp]),
            "coarse_small_hpd_inverse": (C.c_int, [vp, vp, i32, vp, vp]),
            "coarse_block_rotate": (C.c_int, [vp, vp, vp, vp, dbl, i64, i32, vp]),
            "coarse_op_fill_synthetic": (C.c_int, [vp, vp, i32, i32, u64, dbl, C.POINTER(dbl), vp]),
            "coarse_fill_block": (C.c_int, [vp, vp, i32, i32, i32, u64, i32, vp]),
            "coarse_op_kernel_name": (C.c_char_p, [vp, i32]),
            "coarse_op_device_bytes": (i64, [vp]),
            "coarse_launch_count": (i64, []),
            "coarse_last_error": (C.c_char_p, []),
            "coarse_op_profile": (C.c_int, [vp, i32]),
            "coarse_op_profile_read": (C.c_int, [vp, C.POINTER(dbl), i32, C.POINTER(i32)]),
            "coarse_cheby_apply": (C.c_int, [vp, vp, vp, i32, dbl, dbl, i32, vp]),
            "coarse_deflate": (C.c_int, [vp, vp, C.POINTER(dbl), i32, vp, vp, vp, i32, vp]),
            "coarse_block_project": (C.c_int, [vp, vp, vp, i64, i32, i32, i32, i32, vp]),
            "coarse_block_promote": (C.c_int, [vp, vp, vp, i64, i32, i32, i32, i32, vp]),
            "block_cg_solve_ex": (C.c_int, [vp, vp, vp, i32, dbl, i32, u32, C.POINTER(BlockCGResult), vp]),
            "block_cg_solve_host_ex": (C.c_int, [vp, vp, vp, i32, dbl, i32, u32, C.POINTER(BlockCGResult), vp]),
            "stacked_cg_solve": (C.c_int, [vp, vp, vp, i32, dbl, i32, C.POINTER(BlockCGResult), vp]),
            "pblock_cg_solve": (C.c_int, [vp, vp, vp, i32, dbl, i32, C.POINTER(CoarsePrecond), C.POINTER(BlockCGResult), vp]),
            "coarse_cheby_defl_solve": (C.c_int, [vp, vp, C.POINTER(dbl), i32, vp, vp, i32, dbl, dbl, i32, vp]),
            "coarse_measure_peaks": (C.c_int, [C.POINTER(dbl), i32, vp, i64, vp]),
            "coarse_block_gram_noalloc": (C.c_int, [i32, vp, vp, vp, i64, i32, vp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(st: int, allow=()):
    if st != OK and st not in allow:
        raise CoarseError(st, lib().coarse_last_error().decode())
    return st


def _stream(stream=None) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.complex64:
        return C64
    if t.dtype == torch.complex128:
        return C128
    raise TypeError("tensors must be complex64 or complex128")


def _dims(dims):
    return (C.c_int32 * 4)(*[int(d) for d in dims])


def _dev(t: torch.Tensor) -> int:
    if not (t.is_cuda and t.is_contiguous()):
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def launch_count() -> int:
    return int(lib().coarse_launch_count())


def measure_peaks(scratch_bytes: int = 4 << 30, stream=None) -> dict:
    """coarse_measure_peaks on the current device: read-only HBM stream GB/s and FFMA / FFMA2 / DFMA / DMMA TFLOP/s."""
    scratch = torch.randint(0, 2 ** 31 - 1, (int(scratch_bytes) // 4,), dtype=torch.int32, device="cuda")
    out = (C.c_double * 5)()
    _check(lib().coarse_measure_peaks(out, 5, _dev(scratch), C.c_int64(scratch.numel() * 4), _stream(stream)))
    del scratch
    return dict(hbm_read_gbs=out[0], ffma_tflops=out[1], ffma2_tflops=out[2], dfma_tflops=out[3], dmma_tflops=out[4])


NOALLOC_MAX_NRHS, NOALLOC_SCRATCH_BYTES = 32, 256 * 32 * 32 * 16


def block_gram_noalloc(U: torch.Tensor, W: torch.Tensor, G: torch.Tensor, stream=None) -> torch.Tensor:
    """coarse_block_gram_noalloc: G = U^H W into the caller's [s][s] complex128 CUDA tensor, without a handle and without any
    allocation (the reduction scratch is a static device array of NOALLOC_SCRATCH_BYTES; s <= NOALLOC_MAX_NRHS; calls that
    overlap on the GPU race on it).  This wrapper allocates nothing either."""
    s = int(U.shape[-1])
    if U.dtype not in (torch.complex64, torch.complex128) or W.dtype != U.dtype or W.shape != U.shape:
        raise ValueError("U and W: complex64 or complex128 blocks of one shape")
    if G.dtype != torch.complex128 or tuple(G.shape) != (s, s):
        raise ValueError("G: [s][s] complex128")
    _check(lib().coarse_block_gram_noalloc(C64 if U.dtype == torch.complex64 else C128, _dev(U), _dev(W), _dev(G), U.numel() // s, s,
                                           _stream(stream)))
    return G


class CoarseOperator:
    """Handle of coarse_op_create.  A: [V][81][nb][nb] complex CUDA tensor (canonical layout; copied into the
    kernels' own layouts, so the caller may release it afterwards)."""

    def __init__(self, dims, A: torch.Tensor, nrhs_max: int, flags: int = 0, stream=None):
        self.dims = tuple(int(d) for d in dims)
        V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        if A.dim() != 4 or A.shape[0] != V or A.shape[1] != 81 or A.shape[2] != A.shape[3]:
            raise ValueError("A must be [V][81][nbasis][nbasis]")
        self.V, self.nbasis, self.nrhs_max, self.dtype = V, int(A.shape[2]), int(nrhs_max), A.dtype
        self._h = C.c_void_p()
        _check(lib().coarse_op_create(C.byref(self._h), _dims(self.dims), self.nbasis, self.nrhs_max, _dtype_code(A),
                                      _dev(A), flags, _stream(stream)))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().coarse_op_destroy(self._h)
            self._h = None

    __del__ = close

    def _block_ok(self, X: torch.Tensor) -> int:
        if X.dtype != self.dtype or X.dim() != 3 or X.shape[0] != self.V or X.shape[1] != self.nbasis:
            raise ValueError("blocks must be [V][nbasis][nrhs] in the operator's dtype")
        return int(X.shape[2])

    def kernel_name(self, nrhs: int) -> str:
        return lib().coarse_op_kernel_name(self._h, int(nrhs)).decode()

    def device_bytes(self) -> int:
        return int(lib().coarse_op_device_bytes(self._h))

    def profile(self, enable: bool):
        _check(lib().coarse_op_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """milliseconds of each stencil-kernel launch since the last read (CUDA events on the launch stream)."""
        ms = (C.c_double * 64)()
        n = C.c_int32(0)
        _check(lib().coarse_op_profile_read(self._h, ms, 64, C.byref(n)))
        return [ms[i] for i in range(n.value)]

    def apply(self, X: torch.Tensor, Y: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """coarse_op_apply: Y(x) = sum_p A_p(x) X(x + delta_p)  (Eq. 19)."""
        s = self._block_ok(X)
        if Y is None:
            Y = torch.empty_like(X)
        self._block_ok(Y)
        _check(lib().coarse_op_apply(self._h, _dev(X), _dev(Y), s, _stream(stream)))
        return Y

    def cheby_apply(self, B: torch.Tensor, lo: float, hi: float, order: int, X: torch.Tensor | None = None, stream=None) -> torch.Tensor:
        """coarse_cheby_apply: X = P(H) B, P the order-`order` Chebyshev interpolant of 1/x on [lo, hi]."""
        s = self._block_ok(B)
        if X is None:
            X = torch.empty_like(B)
        self._block_ok(X)
        _check(lib().coarse_cheby_apply(self._h, _dev(B), _dev(X), s, float(lo), float(hi), int(order), _stream(stream)))
        return X

    def _evecs_ok(self, Vev: torch.Tensor, lam):
        n = self.V * self.nbasis
        if Vev.dtype != self.dtype or not Vev.is_cuda or not Vev.is_contiguous() or Vev.dim() != 2 or Vev.shape[0] != n:
            raise ValueError(f"Vev must be a contiguous device tensor [{n}][nev] of dtype {self.dtype}")
        nev = int(Vev.shape[1])
        if len(lam) != nev:
            raise ValueError("one eigenvalue per column of Vev")
        return nev, (C.c_double * nev)(*[float(x) for x in lam])

    def deflate(self, Vev: torch.Tensor, lam, B: torch.Tensor, stream=None):
        """coarse_deflate: (Q b_par, b_perp) for a block B (Eq. 7-10)."""
        s = self._block_ok(B)
        nev, lam_c = self._evecs_ok(Vev, lam)
        q, perp = torch.empty_like(B), torch.empty_like(B)
        _check(lib().coarse_deflate(self._h, _dev(Vev), lam_c, nev, _dev(B), _dev(q), _dev(perp), s, _stream(stream)))
        return q, perp

    def cheby_defl_solve(self, Vev: torch.Tensor, lam, B: torch.Tensor, lo: float, hi: float, order: int, stream=None) -> torch.Tensor:
        """coarse_cheby_defl_solve: X = Defl(b_par) + P^Cheby(b_perp) (Eq. 11-12)."""
        s = self._block_ok(B)
        nev, lam_c = self._evecs_ok(Vev, lam)
        X = torch.empty_like(B)
        _check(lib().coarse_cheby_defl_solve(self._h, _dev(Vev), lam_c, nev, _dev(B), _dev(X), s, float(lo), float(hi), int(order), _stream(stream)))
        return X

    def apply_host(self, X: torch.Tensor, Y: torch.Tensor, stream=None) -> torch.Tensor:
        """coarse_op_apply_host: X, Y are (pinned) HOST tensors; H2D + apply + D2H + sync."""
        s = self._block_ok(X)
        self._block_ok(Y)
        if X.is_cuda or Y.is_cuda or not X.is_contiguous() or not Y.is_contiguous():
            raise ValueError("apply_host takes contiguous host tensors")
        _check(lib().coarse_op_apply_host(self._h, X.data_ptr(), Y.data_ptr(), s, _stream(stream)))
        return Y

    def _result(self, res: BlockCGResult, s: int, X):
        k = res.iterations
        return dict(X=X, iterations=int(k), status=int(res.status), seconds=float(res.seconds),
                    history=[res.history[i] for i in range(min(k + 1, MAX_HISTORY))],
                    rel_res_recursive=[res.rel_res_recursive[r] for r in range(s)],
                    rel_res_true=[res.rel_res_true[r] for r in range(s)])

    def block_cg(self, B: torch.Tensor, X: torch.Tensor | None = None, tol: float = 1e-6, maxiter: int = 1000, stream=None,
                 zero_guess: bool = False):
        """block_cg_solve(_ex): BlockCGrQ (Fig. 2 left).  X in: X0 (zeros if None), out: solution;
        zero_guess: X is an output only (X_0 = 0: R_0 = B, one application of the operator less)."""
        s = self._block_ok(B)
        if X is None:
            X = torch.empty_like(B) if zero_guess else torch.zeros_like(B)
        self._block_ok(X)
        res = BlockCGResult()
        _check(lib().block_cg_solve_ex(self._h, _dev(B), _dev(X), s, float(tol), int(maxiter), SOLVE_ZERO_GUESS if zero_guess else 0,
                                       C.byref(res), _stream(stream)), allow=(NOT_CONVERGED, BREAKDOWN))
        return self._result(res, s, X)

    def stacked_cg(self, B: torch.Tensor, X: torch.Tensor | None = None, tol: float = 1e-6, maxiter: int = 1000, stream=None):
        """stacked_cg_solve: single-Krylov CG on the stacked system."""
        s = self._block_ok(B)
        if X is None:
            X = torch.zeros_like(B)
        self._block_ok(X)
        res = BlockCGResult()
        _check(lib().stacked_cg_solve(self._h, _dev(B), _dev(X), s, float(tol), int(maxiter), C.byref(res), _stream(stream)),
               allow=(NOT_CONVERGED, BREAKDOWN))
        return self._result(res, s, X)

    def pblock_cg(self, B: torch.Tensor, lo: float, hi: float, order: int, Vev: torch.Tensor | None = None, lam=None,
                  X: torch.Tensor | None = None, tol: float = 1e-6, maxiter: int = 1000, stream=None):
        """pblock_cg_solve: Preconditioned BlockCGrQ (Fig. 2 right); preconditioner = Chebyshev polynomial of
        the operator on [lo, hi], deflated with the eigenpairs (Vev, lam) when given."""
        s = self._block_ok(B)
        if X is None:
            X = torch.zeros_like(B)
        self._block_ok(X)
        M = CoarsePrecond(kind=PRECOND_CHEBY, order=int(order), lo=float(lo), hi=float(hi), Vev_dev=None, lambda_host=None, nev=0)
        keep = None
        if Vev is not None:
            nev, keep = self._evecs_ok(Vev, lam)
            M.kind, M.Vev_dev, M.lambda_host, M.nev = PRECOND_DEFL_CHEBY, _dev(Vev), C.cast(keep, C.POINTER(C.c_double)), nev
        res = BlockCGResult()
        _check(lib().pblock_cg_solve(self._h, _dev(B), _dev(X), s, float(tol), int(maxiter), C.byref(M), C.byref(res), _stream(stream)),
               allow=(NOT_CONVERGED, BREAKDOWN))
        return self._result(res, s, X)

    def block_cg_begin(self, B: torch.Tensor, X: torch.Tensor, tol: float = 1e-6, stream=None):
        """block_cg_begin: returns (status, initial max relative residual)."""
        s = self._block_ok(B)
        self._block_ok(X)
        self._bcg_keep = (B, X)
        r0 = C.c_double(0.0)
        st = _check(lib().block_cg_begin(self._h, _dev(B), _dev(X), s, float(tol), C.byref(r0), _stream(stream)),
                    allow=(NOT_CONVERGED, BREAKDOWN))
        return st, float(r0.value)

    def block_cg_step(self, count: int = 1, stream=None):
        _check(lib().block_cg_step(self._h, int(count), _stream(stream)))

    def block_cg_end(self, stream=None):
        res = BlockCGResult()
        _check(lib().block_cg_end(self._h, C.byref(res), _stream(stream)), allow=(BREAKDOWN,))
        B, X = self._bcg_keep
        return self._result(res, int(B.shape[2]), X)

    def block_cg_host(self, B: torch.Tensor, X: torch.Tensor, tol: float = 1e-6, maxiter: int = 1000, stream=None, zero_guess: bool = False):
        """block_cg_solve_host(_ex): B, X are (pinned) HOST tensors; zero_guess: X is an output only (X_0 = 0, no copy in)."""
        s = self._block_ok(B)
        self._block_ok(X)
        if B.is_cuda or X.is_cuda:
            raise ValueError("block_cg_host takes host tensors")
        res = BlockCGResult()
        _check(lib().block_cg_solve_host_ex(self._h, B.data_ptr(), X.data_ptr(), s, float(tol), int(maxiter),
                                            SOLVE_ZERO_GUESS if zero_guess else 0, C.byref(res), _stream(stream)),
               allow=(NOT_CONVERGED, BREAKDOWN))
        return self._result(res, s, X)

    # ---- block-CG building blocks (each parity-tested on its own) ----
    def gram(self, U: torch.Tensor, W: torch.Tensor, stream=None) -> torch.Tensor:
        s = int(U.shape[-1])
        n = U.numel() // s
        G = torch.empty((s, s), dtype=torch.complex128, device=U.device)
        _check(lib().coarse_block_gram(self._h, _dev(U), _dev(W), _dev(G), n, s, _stream(stream)))
        return G

    def rotate(self, U: torch.Tensor, K: torch.Tensor, W: torch.Tensor, beta: float, stream=None) -> torch.Tensor:
        """W = beta*W + U K, K s x s complex128 on the device."""
        s = int(U.shape[-1])
        n = U.numel() // s
        _check(lib().coarse_block_rotate(self._h, _dev(U), _dev(K), _dev(W), float(beta), n, s, _stream(stream)))
        return W


def small_cholesky(G: torch.Tensor, want_inverse: bool = True, stream=None):
    s = int(G.shape[0])
    S = torch.empty_like(G)
    Sinv = torch.empty_like(G) if want_inverse else None
    info = torch.zeros(1, dtype=torch.int32, device=G.device)
    _check(lib().coarse_small_cholesky(_dev(G), _dev(S), _dev(Sinv) if want_inverse else None, s, _dev(info), _stream(stream)))
    return S, Sinv, int(info.item())


def small_hpd_inverse(G: torch.Tensor, stream=None):
    s = int(G.shape[0])
    M = torch.empty_like(G)
    info = torch.zeros(1, dtype=torch.int32, device=G.device)
    _check(lib().coarse_small_hpd_inverse(_dev(G), _dev(M), s, _dev(info), _stream(stream)))
    return M, int(info.item())


def fill_synthetic(dims, nbasis: int, dtype: torch.dtype, seed: int, c_factor: float, device="cuda", stream=None):
    """coarse_op_fill_synthetic: device-side seeded HPD operator (input generation).  Returns (A, c)."""
    V = int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])
    A = torch.empty((V, 81, nbasis, nbasis), dtype=dtype, device=device)
    c = C.c_double(0.0)
    _check(lib().coarse_op_fill_synthetic(_dev(A), _dims(dims), nbasis, _dtype_code(A), int(seed), float(c_factor),
                                          C.byref(c), _stream(stream)))
    return A, float(c.value)


def fill_block(dims, nbasis: int, nrhs: int, dtype: torch.dtype, seed: int, tag: int, device="cuda", stream=None):
    V = int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])
    X = torch.empty((V, nbasis, nrhs), dtype=dtype, device=device)
    _check(lib().coarse_fill_block(_dev(X), _dims(dims), nbasis, nrhs, _dtype_code(X), int(seed), int(tag), _stream(stream)))
    return X


def _transfer(fn, Basis: torch.Tensor, src: torch.Tensor, out_rows: int, stream=None) -> torch.Tensor:
    if Basis.dim() != 3 or src.dim() != 3 or Basis.shape[0] != src.shape[0] or Basis.dtype != src.dtype:
        raise ValueError("Basis [Vc][vblock][nbasis] and the vector block must share Vc and dtype")
    dt = C64 if Basis.dtype == torch.complex64 else C128
    Vc, vb, nb = (int(x) for x in Basis.shape)
    out = torch.empty((Vc, out_rows, int(src.shape[2])), dtype=src.dtype, device=src.device)
    _check(fn(_dev(Basis), _dev(src), _dev(out), Vc, vb, nb, int(src.shape[2]), dt, _stream(stream)))
    return out


def block_project(Basis: torch.Tensor, F: torch.Tensor, stream=None) -> torch.Tensor:
    """coarse_block_project (Eq. 14): C[x] = Basis[x]^dagger F[x]."""
    if F.shape[1] != Basis.shape[1]:
        raise ValueError("F must be [Vc][vblock][nrhs]")
    return _transfer(lib().coarse_block_project, Basis, F, int(Basis.shape[2]), stream)


def block_promote(Basis: torch.Tensor, Cc: torch.Tensor, stream=None) -> torch.Tensor:
    """coarse_block_promote (Eq. 15): F[x] = Basis[x] C[x]."""
    if Cc.shape[1] != Basis.shape[2]:
        raise ValueError("C must be [Vc][nbasis][nrhs]")
    return _transfer(lib().coarse_block_promote, Basis, Cc, int(Basis.shape[1]), stream)
