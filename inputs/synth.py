"""Seeded synthetic inputs for the coarse multi-RHS operator (shared by tests, bench and smoke).

This module is the ONLY code that both the CPU oracle's tests and the CUDA path's tests use.
It holds input *generation* only: a counter-based integer hash, a Box-Muller transform and the
index bookkeeping that makes the synthetic operator Hermitian positive definite.  It contains
none of the method's arithmetic (no operator apply, no Gram product, no solver) and imports
neither `oracle/` nor the CUDA package.

Recipe (BASELINE.json configs; SURVEY.md section 8(c) readings 13-15):

* lattice site index  x = x0 + L0*(x1 + L1*(x2 + L2*x3))            (dims[0] fastest)
* stencil point       p = (d0+1) + 3*(d1+1) + 9*(d2+1) + 27*(d3+1),  d in {-1,0,1}^4,
                      centre p = 40, opposite point 80 - p
* p < 40 :  A_p(x)[i][j] = z / nbasis,  z ~ complex N(0,1)  (E|z|^2 = 1)
* p > 40 :  A_p(x)[i][j] = conj( A_{80-p}(x + delta_p)[j][i] )   so the assembled matrix is Hermitian
            (the operator being coarsened is Hermitian)
* p = 40 :  A_40(x) = (G + G^H)/2 + c*I,  G entries complex N(0,1)/nbasis,
            c = factor * max_x [ ||Hrand(x)||_F + sum_{p != 40} ||A_p(x)||_F ]   (block Gershgorin => HPD)
* every value is rounded to float32 and stored/widened from there, so complex64 and complex128
  runs see bit-identical inputs.

Random numbers: element `idx` of stream (seed, tag) is  mix64(K + (idx+1)*GOLDEN),
K = mix64(seed + tag*TAGMUL)  (the splitmix64 output function), split into two 32-bit uniforms
u = (k + 0.5) / 2^32 and turned into one complex normal by Box-Muller in float64.
"""
from __future__ import annotations

import numpy as np

GOLDEN = np.uint64(0x9E3779B97F4A7C15)
TAGMUL = np.uint64(0xD1B54A32D192ED03)
M1 = np.uint64(0xBF58476D1CE4E5B9)
M2 = np.uint64(0x94D049BB133111EB)

TAG_A = 1      # off-diagonal stencil matrices, p < 40
TAG_G = 2      # Hermitian random part of the centre matrix
TAG_X = 3      # a block of vectors (X)
TAG_B = 4      # a block of sources (B)
TAG_U = 5      # extra blocks for invariants
TAG_W = 6

NPOINT = 81
CENTRE = 40


def mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 output function on uint64 arrays (wrap-around arithmetic)."""
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * M1
        z = (z ^ (z >> np.uint64(27))) * M2
        z = z ^ (z >> np.uint64(31))
    return z


def stream_key(seed: int, tag: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = np.array([seed], dtype=np.uint64) + np.array([tag], dtype=np.uint64) * TAGMUL
    return mix64(k)[0]


def complex_normal(seed: int, tag: int, idx: np.ndarray) -> np.ndarray:
    """complex N(0,1) samples (E|z|^2 = 1) for element indices `idx` of stream (seed, tag); complex128."""
    idx = np.asarray(idx, dtype=np.uint64)
    key = stream_key(seed, tag)
    with np.errstate(over="ignore"):
        h = mix64(key + (idx + np.uint64(1)) * GOLDEN)
    u1 = ((h >> np.uint64(32)).astype(np.float64) + 0.5) * (1.0 / 4294967296.0)
    u2 = ((h & np.uint64(0xFFFFFFFF)).astype(np.float64) + 0.5) * (1.0 / 4294967296.0)
    # Box-Muller; radius scaled so that re, im ~ N(0, 1/2)
    r = np.sqrt(-np.log(u1))
    ang = (2.0 * np.pi) * u2
    return r * np.cos(ang) + 1j * (r * np.sin(ang))


def stencil_offsets() -> np.ndarray:
    """(81, 4) int array: offsets[p] = (d0, d1, d2, d3) with p = sum (d_k+1) 3^k."""
    p = np.arange(NPOINT)
    return np.stack([(p // 3 ** k) % 3 - 1 for k in range(4)], axis=1).astype(np.int64)


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


def site_coords(dims, sites: np.ndarray) -> np.ndarray:
    """(len(sites), 4) coordinates of linear site indices (dims[0] fastest)."""
    sites = np.asarray(sites, dtype=np.int64)
    c = np.empty((sites.size, 4), dtype=np.int64)
    rem = sites.copy()
    for k in range(4):
        c[:, k] = rem % dims[k]
        rem //= dims[k]
    return c


def shifted_sites(dims, sites: np.ndarray, p: int) -> np.ndarray:
    """linear index of x + delta_p with periodic wrap, for each x in `sites`."""
    off = stencil_offsets()[p]
    c = site_coords(dims, sites)
    out = np.zeros(len(c), dtype=np.int64)
    stride = 1
    for k in range(4):
        out += ((c[:, k] + off[k]) % dims[k]) * stride
        stride *= dims[k]
    return out


def _raw_offdiag(dims, nb: int, seed: int, sites: np.ndarray, p: int) -> np.ndarray:
    """independent half (p < 40): float32-rounded z/nb, shape (len(sites), nb, nb) complex64."""
    assert p < CENTRE
    sites = np.asarray(sites, dtype=np.int64)
    ij = np.arange(nb * nb, dtype=np.int64)
    idx = (sites[:, None] * NPOINT + p) * (nb * nb) + ij[None, :]
    z = complex_normal(seed, TAG_A, idx) / nb
    return z.astype(np.complex64).reshape(len(sites), nb, nb)


def _raw_hrand(nb: int, seed: int, sites: np.ndarray) -> np.ndarray:
    """Hrand(x) = (G + G^H)/2 with float32-rounded G; result float32-exact and exactly Hermitian."""
    sites = np.asarray(sites, dtype=np.int64)
    ij = np.arange(nb * nb, dtype=np.int64)
    idx = sites[:, None] * (nb * nb) + ij[None, :]
    g = (complex_normal(seed, TAG_G, idx) / nb).astype(np.complex64).reshape(len(sites), nb, nb)
    g = g.astype(np.complex128)
    h = 0.5 * (g + np.conj(np.transpose(g, (0, 2, 1))))
    return h.astype(np.complex64)


def stencil_matrices(dims, nb: int, seed: int, sites=None) -> np.ndarray:
    """A[x][p] for the listed sites WITHOUT the c*I shift: (len(sites), 81, nb, nb) complex64.

    A pure function of (dims, nb, seed, site index): any subset of sites can be generated
    without generating the rest (used for sampled checks at the large configurations).
    """
    V = volume(dims)
    sites = np.arange(V, dtype=np.int64) if sites is None else np.asarray(sites, dtype=np.int64)
    A = np.empty((len(sites), NPOINT, nb, nb), dtype=np.complex64)
    for p in range(NPOINT):
        if p < CENTRE:
            A[:, p] = _raw_offdiag(dims, nb, seed, sites, p)
        elif p == CENTRE:
            A[:, p] = _raw_hrand(nb, seed, sites)
        else:
            y = shifted_sites(dims, sites, p)
            A[:, p] = np.conj(np.transpose(_raw_offdiag(dims, nb, seed, y, NPOINT - 1 - p), (0, 2, 1)))
    return A


def offdiag_bound(dims, nb: int, seed: int, chunk: int = 2048) -> float:
    """max_x [ ||Hrand(x)||_F + sum_{p != 40} ||A_p(x)||_F ]  (float64, from the float32 values)."""
    V = volume(dims)
    best = 0.0
    for s0 in range(0, V, chunk):
        sites = np.arange(s0, min(V, s0 + chunk), dtype=np.int64)
        A = stencil_matrices(dims, nb, seed, sites).astype(np.complex128)
        fro = np.sqrt(np.sum(A.real ** 2 + A.imag ** 2, axis=(2, 3)))   # (sites, 81)
        best = max(best, float(np.max(np.sum(fro, axis=1))))
    return best


def diagonal_shift(dims, nb: int, seed: int, factor: float) -> float:
    """c = factor * bound, rounded to float32 (returned as a Python float holding that value)."""
    return float(np.float32(factor * offdiag_bound(dims, nb, seed)))


def add_shift(A: np.ndarray, c: float) -> np.ndarray:
    """in place: A[:, 40] += c*I, result rounded to float32 (A is complex64)."""
    nb = A.shape[-1]
    d = np.arange(nb)
    A[:, CENTRE, d, d] = (A[:, CENTRE, d, d].astype(np.complex128) + c).astype(np.complex64)
    return A


def make_operator(dims, nb: int, seed: int, factor: float, chunk: int = 2048):
    """Full synthetic HPD operator: (A complex64 [V][81][nb][nb], c).  factor = 0 gives c = 0.

    Same values as stencil_matrices() + add_shift(); the dependent half (p > 40) is filled by a gather
    from the independent half instead of re-hashing."""
    V = volume(dims)
    A = np.empty((V, NPOINT, nb, nb), dtype=np.complex64)
    allsites = np.arange(V, dtype=np.int64)
    for s0 in range(0, V, chunk):
        sites = allsites[s0:s0 + chunk]
        for p in range(CENTRE):
            A[s0:s0 + len(sites), p] = _raw_offdiag(dims, nb, seed, sites, p)
        A[s0:s0 + len(sites), CENTRE] = _raw_hrand(nb, seed, sites)
    for p in range(CENTRE + 1, NPOINT):
        y = shifted_sites(dims, allsites, p)
        A[:, p] = np.conj(np.transpose(A[y, NPOINT - 1 - p], (0, 2, 1)))
    best = 0.0
    for s0 in range(0, V, chunk):
        b = A[s0:s0 + chunk].astype(np.complex128)
        fro = np.sqrt(np.sum(b.real ** 2 + b.imag ** 2, axis=(2, 3)))
        best = max(best, float(np.max(np.sum(fro, axis=1))))
    c = float(np.float32(factor * best))
    if c != 0.0:
        add_shift(A, c)
    return A, c


def make_block(dims, nb: int, s: int, seed: int, tag: int = TAG_X, sites=None) -> np.ndarray:
    """A block of vectors [V][nb][s], entries complex N(0,1) rounded to float32; complex128."""
    V = volume(dims)
    sites = np.arange(V, dtype=np.int64) if sites is None else np.asarray(sites, dtype=np.int64)
    ir = np.arange(nb * s, dtype=np.int64)
    idx = sites[:, None] * (nb * s) + ir[None, :]
    z = complex_normal(seed, tag, idx).astype(np.complex64)
    return z.astype(np.complex128).reshape(len(sites), nb, s)


# BASELINE.json configs (index = position in BASELINE.json "configs"); seed = 20240903 + index
CONFIGS = [
    dict(name="cfg1_4^4_nb8_s4_c128", dims=(4, 4, 4, 4), nbasis=8, nrhs=4, dtype="c128", factor=1.10, tol=1e-10),
    dict(name="cfg2_8^4_nb24_s8_c128", dims=(8, 8, 8, 8), nbasis=24, nrhs=8, dtype="c128", factor=1.05, tol=1e-10),
    dict(name="cfg3_8^3x16_nb32_s16_c64", dims=(8, 8, 8, 16), nbasis=32, nrhs=16, dtype="c64", factor=1.02, tol=1e-6),
    dict(name="cfg4_12^3x24_nb32_sweep_c64", dims=(12, 12, 12, 24), nbasis=32, nrhs=16, dtype="c64", factor=1.02,
         tol=1e-6, sweep=(1, 4, 8, 16, 32, 64)),
    dict(name="cfg5_16^3x32_nb24_s64_c64", dims=(16, 16, 16, 32), nbasis=24, nrhs=64, dtype="c64", factor=1.01, tol=1e-6),
]
BASE_SEED = 20240903


def config(index: int) -> dict:
    cfg = dict(CONFIGS[index])
    cfg["seed"] = BASE_SEED + index
    cfg["index"] = index
    return cfg
