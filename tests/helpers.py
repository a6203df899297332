"""Test-side helpers that are independent of BOTH the oracle and the CUDA path.

dense_matrix() assembles the n x n matrix of the coarse operator by brute force with its own
coordinate arithmetic (python ints, itertools) -- the pin for the oracle's apply on tiny lattices.
"""
import itertools

import numpy as np


def dense_matrix(dims, A):
    """H[(x,i),(y,j)] += A[x][p][i][j] for y = x + delta_p (periodic), p = sum (d_k+1) 3^k."""
    L = [int(d) for d in dims]
    V = L[0] * L[1] * L[2] * L[3]
    nb = A.shape[-1]
    H = np.zeros((V * nb, V * nb), dtype=np.complex128)

    def lin(c):
        return c[0] + L[0] * (c[1] + L[1] * (c[2] + L[2] * c[3]))

    for c3, c2, c1, c0 in itertools.product(range(L[3]), range(L[2]), range(L[1]), range(L[0])):
        x = lin((c0, c1, c2, c3))
        for d3, d2, d1, d0 in itertools.product((-1, 0, 1), repeat=4):
            p = (d0 + 1) + 3 * (d1 + 1) + 9 * (d2 + 1) + 27 * (d3 + 1)
            y = lin(((c0 + d0) % L[0], (c1 + d1) % L[1], (c2 + d2) % L[2], (c3 + d3) % L[3]))
            H[x * nb:(x + 1) * nb, y * nb:(y + 1) * nb] += A[x, p]
    return H


def lattice_view(dims, X):
    """[V][nb][s] -> [L3][L2][L1][L0][nb][s] (dims[0] fastest)."""
    return X.reshape(dims[3], dims[2], dims[1], dims[0], X.shape[1], X.shape[2])


def shifted_block(dims, X, delta):
    """Z(x) = X(x + delta) with periodic wrap, via numpy.roll on the lattice view."""
    v = lattice_view(dims, X)
    for k in range(4):
        v = np.roll(v, -int(delta[k]), axis=3 - k)
    return v.reshape(X.shape)


def rel_err_cols(Y, Yref):
    """max over columns r of ||Y[:,r] - Yref[:,r]||_2 / ||Yref[:,r]||_2  (the parity metric)."""
    s = Y.shape[-1]
    d = (Y - Yref).reshape(-1, s)
    r = Yref.reshape(-1, s)
    return float(np.max(np.linalg.norm(d, axis=0) / np.linalg.norm(r, axis=0)))


def stress_operator(dims, nb, seed, delta):
    """The synthetic stencil matrices with the diagonal shift taken from the SPECTRUM instead of the loose Frobenius bound
    ("optional stress operator"): c = (1 + delta) |lambda_min(off-diagonal part)|, lambda_min from a
    dense eigvalsh of the brute-force matrix (small lattices only).  Returns (A complex64 float32-exact, c, lambda_min(H),
    lambda_max(H)); kappa(H) ~ (lambda_max - lambda_min) / (delta |lambda_min|): delta 0.02 -> ~100, 0.001 -> ~2000."""
    from inputs import synth
    A, _ = synth.make_operator(dims, nb, seed, 0.0)
    lam = np.linalg.eigvalsh(dense_matrix(dims, A.astype(np.complex128)))
    c = float(np.float32((1.0 + delta) * abs(lam[0])))
    synth.add_shift(A, c)
    return A, c, float(lam[0] + c), float(lam[-1] + c)
