"""Pins for the oracle's coarse-operator apply (Eq. 19) -- CPU only.

Each test checks oracle/coarse_oracle.c against something that is NOT the oracle: a dense brute-force
matrix assembled with independent index arithmetic, closed forms (pure shift, Fourier symbol),
invariants (Hermiticity, column independence) and a library routine (scipy BSR).
"""
import itertools

import numpy as np
import pytest

from helpers import dense_matrix, rel_err_cols, shifted_block
from inputs import synth
from oracle import oracle


def _rand_A(rng, V, nb):
    return (rng.standard_normal((V, 81, nb, nb)) + 1j * rng.standard_normal((V, 81, nb, nb))) / nb


def _rand_X(rng, V, nb, s):
    return rng.standard_normal((V, nb, s)) + 1j * rng.standard_normal((V, nb, s))


# --- brute force on tiny lattices, including extents 1 and 2 where stencil points alias -------------
@pytest.mark.parametrize("dims,nb,s", [
    ((4, 4, 4, 4), 8, 4),        # BASELINE.json configs[0] shape: 2048 x 2048
    ((2, 3, 4, 5), 3, 2),
    ((3, 3, 3, 3), 4, 3),
    ((2, 2, 2, 2), 5, 1),
    ((1, 2, 3, 1), 2, 7),
    ((1, 1, 1, 1), 6, 2),
    ((5, 1, 1, 2), 1, 1),
])
def test_apply_equals_dense_bruteforce(dims, nb, s):
    rng = np.random.default_rng(hash((dims, nb, s)) % 2 ** 32)
    V = synth.volume(dims)
    A = _rand_A(rng, V, nb)            # generic (non-Hermitian) matrices: no symmetry can hide a transpose
    X = _rand_X(rng, V, nb, s)
    H = dense_matrix(dims, A)
    Yd = (H @ X.reshape(V * nb, s)).reshape(V, nb, s)
    Y = oracle.apply(dims, A, X)
    assert rel_err_cols(Y, Yd) <= 1e-13


def test_apply_cfg1_synthetic_equals_dense(cfg1, cfg1_dense):
    V, nb, s = cfg1["X"].shape
    Yd = (cfg1_dense @ cfg1["X"].reshape(V * nb, s)).reshape(V, nb, s)
    assert rel_err_cols(oracle.apply(cfg1["dims"], cfg1["A"], cfg1["X"]), Yd) <= 1e-13
    # with the dominant diagonal shift removed the off-diagonal terms are not scaled down in the norm
    A0 = cfg1["A"].copy()
    d = np.arange(nb)
    A0[:, 40, d, d] -= cfg1["c"]
    H0 = dense_matrix(cfg1["dims"], A0)
    Yd0 = (H0 @ cfg1["X"].reshape(V * nb, s)).reshape(V, nb, s)
    assert rel_err_cols(oracle.apply(cfg1["dims"], A0, cfg1["X"]), Yd0) <= 1e-13


def test_apply_complex64_storage_matches_complex128_storage(cfg1):
    A64 = cfg1["A"].astype(np.complex64)          # values are float32-exact by construction
    Y64 = oracle.apply(cfg1["dims"], A64, cfg1["X"])
    Y128 = oracle.apply(cfg1["dims"], cfg1["A"], cfg1["X"])
    assert np.array_equal(Y64, Y128)


# --- closed form: a single identity stencil point is a pure periodic shift, bit-exact ----------------
@pytest.mark.parametrize("dims", [(3, 4, 5, 2), (2, 1, 3, 4)])
def test_single_point_identity_is_a_shift(dims):
    rng = np.random.default_rng(7)
    V, nb, s = synth.volume(dims), 3, 2
    X = _rand_X(rng, V, nb, s)
    offs = synth.stencil_offsets()
    for p0 in range(81):
        A = np.zeros((V, 81, nb, nb), dtype=np.complex128)
        A[:, p0] = np.eye(nb)
        Y = oracle.apply(dims, A, X)
        assert np.array_equal(Y, shifted_block(dims, X, offs[p0])), f"p0={p0} delta={offs[p0]}"
        # p_only selects exactly that point out of a full stencil
        assert np.array_equal(oracle.apply(dims, A + 0.0, X, p_only=p0), Y)


def test_neighbour_convention():
    dims = (3, 4, 5, 6)
    for x, p in itertools.product((0, 7, 59, 359), (0, 1, 3, 9, 27, 40, 80)):
        c = [(x // int(np.prod(dims[:k]))) % dims[k] for k in range(4)]
        d = [(p // 3 ** k) % 3 - 1 for k in range(4)]
        y = sum(((c[k] + d[k]) % dims[k]) * int(np.prod(dims[:k])) for k in range(4))
        assert oracle.neighbour(dims, x, p) == y
    assert oracle.neighbour(dims, 0, 40) == 0
    assert oracle.neighbour(dims, 0, 41) == 1               # +1 in the fastest dimension
    assert oracle.neighbour(dims, 0, 39) == dims[0] - 1     # -1 wraps


# --- closed form: constant-coefficient stencil acting on a plane wave (Fourier symbol) ---------------
def test_fourier_symbol():
    dims = (3, 4, 5, 6)
    rng = np.random.default_rng(11)
    V, nb, s = synth.volume(dims), 2, 3
    a = rng.standard_normal(81) + 1j * rng.standard_normal(81)
    A = np.zeros((V, 81, nb, nb), dtype=np.complex128)
    A[:, :, np.arange(nb), np.arange(nb)] = a[None, :, None]
    offs = synth.stencil_offsets()
    coords = synth.site_coords(dims, np.arange(V))
    for mode in [(0, 0, 0, 0), (1, 0, 2, 0), (2, 3, 4, 5), (1, 1, 1, 1)]:
        k = 2 * np.pi * np.array(mode) / np.array(dims)
        v = rng.standard_normal((nb, s)) + 1j * rng.standard_normal((nb, s))
        X = np.exp(1j * coords @ k)[:, None, None] * v[None]
        symbol = np.sum(a * np.exp(1j * offs @ k))
        Y = oracle.apply(dims, A, X)
        assert rel_err_cols(Y, symbol * X) <= 1e-13


# --- invariants ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims,nb", [((4, 4, 4, 4), 8), ((2, 3, 2, 5), 4), ((1, 2, 3, 3), 3)])
def test_synthetic_operator_is_hermitian(dims, nb):
    """<U, H V> = <H U, V>: checks the apply AND the A_{80-p}(x+delta_p) = A_p(x)^H pairing."""
    seed, s = 5, 3
    A, c = synth.make_operator(dims, nb, seed, 1.05)
    U = synth.make_block(dims, nb, s, seed, synth.TAG_U)
    W = synth.make_block(dims, nb, s, seed, synth.TAG_W)
    HU, HW = oracle.apply(dims, A, U), oracle.apply(dims, A, W)
    lhs = np.vdot(U, HW)
    rhs = np.vdot(HU, W)
    assert abs(lhs - rhs) <= 1e-13 * abs(lhs)
    assert abs(np.vdot(U, HU).imag) <= 1e-13 * abs(np.vdot(U, HU))
    assert np.vdot(U, HU).real > 0                      # positive definite by block Gershgorin


def test_block_apply_is_columnwise_apply(cfg1):
    dims, A, X = cfg1["dims"], cfg1["A"], cfg1["X"]
    Y = oracle.apply(dims, A, X)
    for r in range(X.shape[2]):
        yr = oracle.apply(dims, A, X[:, :, r:r + 1].copy())
        assert np.array_equal(yr[:, :, 0], Y[:, :, r])
    perm = np.array([2, 0, 3, 1])
    assert np.array_equal(oracle.apply(dims, A, X[:, :, perm].copy()), Y[:, :, perm])


def test_apply_on_site_subset(cfg1):
    dims, A, X = cfg1["dims"], cfg1["A"], cfg1["X"]
    Y = oracle.apply(dims, A, X)
    sites = np.array([0, 3, 17, 100, 255, 64])
    Ys = oracle.apply(dims, A[sites].copy(), X, sites=sites)
    assert np.array_equal(Ys, Y[sites])


# --- library routine at a mid size: scipy block-sparse-row product (BASELINE.json configs[1] shape, reduced) ----
def test_apply_equals_scipy_bsr():
    import scipy.sparse as sp
    dims, nb, s, seed = (6, 4, 4, 6), 12, 5, 99
    V = synth.volume(dims)
    A, c = synth.make_operator(dims, nb, seed, 1.05)
    X = synth.make_block(dims, nb, s, seed)
    nbr = np.stack([synth.shifted_sites(dims, np.arange(V), p) for p in range(81)], axis=1)   # [V][81]
    H = sp.bsr_matrix((A.reshape(V * 81, nb, nb).astype(np.complex128), nbr.reshape(-1), 81 * np.arange(V + 1)),
                      shape=(V * nb, V * nb))
    Yl = (H @ X.reshape(V * nb, s)).reshape(V, nb, s)
    assert rel_err_cols(oracle.apply(dims, A, X), Yl) <= 1e-13
