"""Pins for the oracle's BlockCGrQ (Fig. 2 left) and its small dense algebra -- CPU only.

Pins: numpy.linalg (cholesky / inv / solve), textbook CG for s = 1, O'Leary's block CG written
independently in numpy on the dense matrix, algebraic invariants of the iterates, the Chebyshev
convergence bound (Eq. 20), and the demonstration that the printed X-update
without C_k cannot be what is meant (reading R1).
"""
import numpy as np
import pytest

from helpers import dense_matrix
from inputs import synth
from oracle import oracle


def _hpd(rng, s):
    M = rng.standard_normal((s + 3, s)) + 1j * rng.standard_normal((s + 3, s))
    return M.conj().T @ M + 0.1 * np.eye(s)


# --- small dense algebra ------------------------------------------------------------------------------
@pytest.mark.parametrize("s", [1, 2, 4, 12, 16, 64])
def test_cholesky_and_inverses_match_numpy(s):
    rng = np.random.default_rng(s)
    G = _hpd(rng, s)
    st, S = oracle.cholesky_upper(G)
    assert st == oracle.OK
    L = np.linalg.cholesky(G)                      # G = L L^H, L lower, positive diagonal => S = L^H
    assert np.allclose(S, L.conj().T, rtol=1e-12, atol=1e-12)
    assert np.all(np.tril(S, -1) == 0) and np.all(S.diagonal().imag == 0) and np.all(S.diagonal().real > 0)
    assert np.allclose(oracle.upper_inverse(S) @ S, np.eye(s), atol=1e-10)
    st, Gi = oracle.hpd_inverse(G)
    assert st == oracle.OK
    assert np.allclose(Gi, np.linalg.inv(G), rtol=1e-9, atol=1e-11)


def test_cholesky_breakdown_on_indefinite():
    G = np.array([[1.0, 2.0], [2.0, 1.0]], dtype=complex)
    st, _ = oracle.cholesky_upper(G)
    assert st == oracle.BREAKDOWN
    st, _ = oracle.cholesky_upper(np.zeros((3, 3), dtype=complex))
    assert st == oracle.BREAKDOWN


def test_gram_matches_numpy():
    rng = np.random.default_rng(3)
    U = rng.standard_normal((50, 4, 6)) + 1j * rng.standard_normal((50, 4, 6))
    W = rng.standard_normal((50, 4, 6)) + 1j * rng.standard_normal((50, 4, 6))
    G = oracle.gram(U, W)
    assert np.allclose(G, U.reshape(-1, 6).conj().T @ W.reshape(-1, 6), rtol=1e-13, atol=1e-13)


# --- the solve against a dense direct solve (BASELINE.json configs[0]) -------------------------------------
def test_block_rotate_matches_numpy_matmul():
    # pin: library routine (numpy matmul) for W = beta W + U K
    rng = np.random.default_rng(11)
    n, s = 301, 5
    U = rng.standard_normal((n, s)) + 1j * rng.standard_normal((n, s))
    W = rng.standard_normal((n, s)) + 1j * rng.standard_normal((n, s))
    K = rng.standard_normal((s, s)) + 1j * rng.standard_normal((s, s))
    for beta in (0.0, 1.0, -0.5):
        out = oracle.block_rotate(U, K, W, beta)
        ref = beta * W + U @ K
        assert np.linalg.norm(out - ref) <= 1e-14 * np.linalg.norm(ref)


def test_block_cg_matches_dense_solve(cfg1, cfg1_dense):
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"]
    V, nb, s = B.shape
    res = oracle.block_cg(dims, A, B, tol=cfg1["tol"], maxiter=100)
    assert res["status"] == oracle.OK
    Xd = np.linalg.solve(cfg1_dense, B.reshape(V * nb, s)).reshape(B.shape)
    kappa = np.linalg.cond(cfg1_dense)
    err = np.linalg.norm(res["X"] - Xd) / np.linalg.norm(Xd)
    assert err <= kappa * cfg1["tol"]
    assert np.max(res["true_rel"]) <= 1.5 * cfg1["tol"]
    # recursive and true residuals agree at convergence
    assert np.allclose(res["history"][-1], res["true_rel"], rtol=1e-3)
    assert res["history"].shape == (res["iterations"] + 1, s)
    assert 5 <= res["iterations"] <= 9           # kappa ~ 1.15: SURVEY.md section 8(c) measured 7


def test_block_cg_nonzero_initial_guess_and_zero_column(cfg1, cfg1_dense):
    dims, A = cfg1["dims"], cfg1["A"]
    B = cfg1["B"].copy()
    V, nb, s = B.shape
    X0 = synth.make_block(dims, nb, s, 1234, synth.TAG_U)
    res = oracle.block_cg(dims, A, B, X0=X0, tol=1e-10, maxiter=100)
    Xd = np.linalg.solve(cfg1_dense, B.reshape(V * nb, s)).reshape(B.shape)
    assert res["status"] == oracle.OK
    assert np.linalg.norm(res["X"] - Xd) / np.linalg.norm(Xd) <= 1e-9
    # already-converged start: zero iterations, no factorisation of a zero Gram matrix
    res2 = oracle.block_cg(dims, A, B, X0=Xd, tol=1e-10, maxiter=100)
    assert res2["status"] == oracle.OK and res2["iterations"] == 0


def test_block_cg_maxiter_reports_not_converged(cfg1):
    res = oracle.block_cg(cfg1["dims"], cfg1["A"], cfg1["B"], tol=1e-10, maxiter=3)
    assert res["status"] == oracle.NOT_CONVERGED and res["iterations"] == 3
    assert np.max(res["true_rel"]) > 1e-10


# --- s = 1 reduces to textbook conjugate gradients (Hestenes-Stiefel), iterate by iterate ------------------
def _textbook_cg(H, b, tol, maxiter):
    x = np.zeros_like(b)
    r = b.copy()
    p = r.copy()
    rr = np.vdot(r, r).real
    xs = [x.copy()]
    bn = np.linalg.norm(b)
    for k in range(maxiter):
        Hp = H @ p
        alpha = rr / np.vdot(p, Hp).real
        x = x + alpha * p
        r = r - alpha * Hp
        rr_new = np.vdot(r, r).real
        xs.append(x.copy())
        if np.sqrt(rr_new) / bn <= tol:
            break
        p = r + (rr_new / rr) * p
        rr = rr_new
    return xs


def test_single_rhs_is_textbook_cg(cfg1, cfg1_dense):
    dims, A = cfg1["dims"], cfg1["A"]
    b = cfg1["B"][:, :, :1].copy()
    V, nb, _ = b.shape
    iterates = []
    res = oracle.block_cg(dims, A, b, tol=1e-10, maxiter=100, callback=lambda k, X, Q, D, C: iterates.append(X.copy()))
    xs = _textbook_cg(cfg1_dense, b.reshape(-1), 1e-10, 100)
    assert res["iterations"] == len(xs) - 1
    for k in range(len(xs)):
        assert np.linalg.norm(iterates[k].reshape(-1) - xs[k]) <= 1e-13 * max(1.0, np.linalg.norm(xs[k]))
    import scipy.sparse.linalg as spla
    xsp, info = spla.cg(cfg1_dense, b.reshape(-1), rtol=1e-10, atol=0.0, maxiter=100)
    assert info == 0
    assert np.linalg.norm(res["X"].reshape(-1) - xsp) / np.linalg.norm(xsp) <= 1e-9


# --- iterates equal O'Leary's block CG (P, alpha, beta form) on an ill-conditioned dense HPD matrix ---------
def _oleary_block_cg(H, B, iters):
    X = np.zeros_like(B)
    R = B.copy()
    P = R.copy()
    out = [X.copy()]
    for _ in range(iters):
        HP = H @ P
        alpha = np.linalg.solve(P.conj().T @ HP, R.conj().T @ R)
        X = X + P @ alpha
        Rn = R - HP @ alpha
        beta = np.linalg.solve(R.conj().T @ R, Rn.conj().T @ Rn)
        P = Rn + P @ beta
        R = Rn
        out.append(X.copy())
    return out


def test_iterates_equal_oleary_block_cg():
    """BlockCGrQ with P_k = D_k C_k is O'Leary's block CG in exact arithmetic (reading R1)."""
    dims, nb, s, seed = (2, 2, 2, 2), 4, 3, 77
    V = synth.volume(dims)
    A, _ = synth.make_operator(dims, nb, seed, 0.0)
    A = A.astype(np.complex128)
    H0 = dense_matrix(dims, A)
    lam = np.linalg.eigvalsh(H0)
    shift = 1.02 * abs(lam[0])                       # kappa ~ 100: many iterations, real block effects
    d = np.arange(nb)
    A[:, 40, d, d] += shift
    H = H0 + shift * np.eye(V * nb)
    B = synth.make_block(dims, nb, s, seed, synth.TAG_B)
    iterates = []
    res = oracle.block_cg(dims, A, B, tol=1e-30, maxiter=12, callback=lambda k, X, Q, D, C: iterates.append(X.copy()))
    ref = _oleary_block_cg(H, B.reshape(V * nb, s), 12)
    assert res["iterations"] == 12
    xn = np.linalg.norm(ref[-1])
    for k in range(13):
        assert np.linalg.norm(iterates[k].reshape(V * nb, s) - ref[k]) <= 1e-10 * xn, k


# --- invariants of the iterates ---------------------------------------------------------------------------
def test_iterate_invariants(cfg1, cfg1_dense):
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"]
    V, nb, s = B.shape
    H = cfg1_dense
    Bm = B.reshape(V * nb, s)
    Xd = np.linalg.solve(H, Bm)
    bn = np.linalg.norm(Bm)
    state = dict(prev_D=None, prev_err=np.inf)

    def check(k, X, Q, D, C):
        Xm, Qm, Dm = X.reshape(-1, s), Q.reshape(-1, s), D.reshape(-1, s)
        assert np.linalg.norm(Qm.conj().T @ Qm - np.eye(s)) <= 1e-12           # Q^H Q = I
        assert np.linalg.norm(Dm.conj().T @ Qm - np.eye(s)) <= 1e-11           # D^H Q = I
        assert np.linalg.norm(Bm - H @ Xm - Qm @ C) / bn <= 1e-13              # R_k = Q_k C_k
        assert np.all(np.tril(C, -1) == 0)                                      # C stays upper triangular
        if state["prev_D"] is not None:                                         # H-conjugate directions
            assert np.linalg.norm(Dm.conj().T @ (H @ state["prev_D"])) <= 1e-10 * np.linalg.norm(H, 2)
        E = Xm - Xd
        err = np.sqrt(np.trace(E.conj().T @ H @ E).real)                        # H-norm error decreases
        assert err <= state["prev_err"] * (1 + 1e-12)
        state["prev_err"] = err
        state["prev_D"] = Dm.copy()

    res = oracle.block_cg(dims, A, B, tol=1e-10, maxiter=100, callback=check)
    assert res["status"] == oracle.OK


def test_convergence_within_chebyshev_bound(cfg1, cfg1_dense):
    """||e_k||_H <= 2 sigma^k ||e_0||_H per column, sigma = (sqrt(kappa)-1)/(sqrt(kappa)+1)."""
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"]
    V, nb, s = B.shape
    H = cfg1_dense
    lam = np.linalg.eigvalsh(H)
    sigma = (np.sqrt(lam[-1] / lam[0]) - 1) / (np.sqrt(lam[-1] / lam[0]) + 1)
    Xd = np.linalg.solve(H, B.reshape(V * nb, s))
    e0 = np.sqrt(np.einsum("ir,ij,jr->r", Xd.conj(), H, Xd).real)

    def check(k, X, Q, D, C):
        E = X.reshape(-1, s) - Xd
        ek = np.sqrt(np.abs(np.einsum("ir,ij,jr->r", E.conj(), H, E).real))
        assert np.all(ek <= 2 * sigma ** k * e0 * (1 + 1e-9) + 1e-13 * e0)

    oracle.block_cg(dims, A, B, tol=1e-10, maxiter=100, callback=check)


# --- DESIGN.md reading R1: the printed update X + D M (no C_k) does not solve the system -------------------
def test_printed_update_without_Ck_fails(cfg1, cfg1_dense):
    H = cfg1_dense
    V, nb, s = cfg1["B"].shape
    B = cfg1["B"].reshape(V * nb, s)

    def run(with_c):
        X = np.zeros_like(B)
        R = B.copy()
        C = np.linalg.cholesky(R.conj().T @ R).conj().T
        Q = R @ np.linalg.inv(C)
        D = Q.copy()
        for _ in range(8):
            Z = H @ D
            M = np.linalg.inv(D.conj().T @ Z)
            X = X + (D @ M @ C if with_c else D @ M)
            T = Q - Z @ M
            S = np.linalg.cholesky(T.conj().T @ T).conj().T
            Q = T @ np.linalg.inv(S)
            D = Q + D @ S.conj().T
            C = S @ C
        return np.linalg.norm(B - H @ X) / np.linalg.norm(B)

    assert run(True) <= 1e-10
    assert run(False) >= 0.5
