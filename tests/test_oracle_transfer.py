"""Pins of the block project / promote oracle (oracle/transfer_oracle.py; Eq. 14-15)."""
import numpy as np

from oracle import transfer_oracle


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_explicit_loops_on_a_tiny_case():
    rng = np.random.default_rng(0)
    Vc, vb, nb, s = 3, 5, 4, 2
    Bas, F, Cc = _rand(rng, Vc, vb, nb), _rand(rng, Vc, vb, s), _rand(rng, Vc, nb, s)
    P = transfer_oracle.project(Bas, F)
    Q = transfer_oracle.promote(Bas, Cc)
    for x in range(Vc):
        for k in range(nb):
            for r in range(s):
                assert abs(P[x, k, r] - sum(np.conj(Bas[x, v, k]) * F[x, v, r] for v in range(vb))) <= 1e-13
        for v in range(vb):
            for r in range(s):
                assert abs(Q[x, v, r] - sum(Bas[x, v, k] * Cc[x, k, r] for k in range(nb))) <= 1e-13


def test_orthonormal_basis_projector_identities_and_adjointness():
    rng = np.random.default_rng(1)
    Vc, vb, nb, s = 4, 24, 6, 3
    Bas = np.stack([np.linalg.qr(_rand(rng, vb, nb))[0] for _ in range(Vc)])      # block-orthonormal basis
    F, Cc = _rand(rng, Vc, vb, s), _rand(rng, Vc, nb, s)
    assert np.allclose(transfer_oracle.project(Bas, transfer_oracle.promote(Bas, Cc)), Cc, atol=1e-13)
    PF = transfer_oracle.promote(Bas, transfer_oracle.project(Bas, F))            # orthogonal projector onto the subspace
    assert np.allclose(transfer_oracle.promote(Bas, transfer_oracle.project(Bas, PF)), PF, atol=1e-13)
    assert abs(np.vdot(PF, F - PF)) <= 1e-12 * np.vdot(F, F).real
    lhs = np.vdot(transfer_oracle.promote(Bas, Cc), F)                            # <promote C, F> = <C, project F>
    rhs = np.vdot(Cc, transfer_oracle.project(Bas, F))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
