"""-m gpu parity of coarse_block_project / coarse_block_promote (Eq. 14-15) against oracle/transfer_oracle.py.
Tolerance: the apply's norm-wise figures (1e-12 complex128, 1e-5 complex64; K = V_block <= 3072 products per output)."""
import numpy as np
import pytest
import torch

from gpu_common import NP_DTYPE, TOL
from helpers import rel_err_cols
from oracle import transfer_oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _rand(rng, dtype, *shape):
    a = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / np.sqrt(2)
    return a.astype(np.complex64).astype(np.complex128) if dtype == "c64" else a


@pytest.mark.parametrize("Vc,vb,nb,s,dtype", [
    (4096, 256, 64, 12, "c64"),      # Table 6 "Project" / "Promote" shape, FP32
    (64, 256, 64, 12, "c128"),       # same shape, FP64, fewer sites
    (7, 100, 24, 8, "c128"),         # ragged V_block
    (33, 37, 13, 5, "c64"),          # odd everything
    (3, 3072, 32, 16, "c64"),        # 4^4 x 12 fine degrees of freedom per block
    (1, 1, 1, 1, "c128"),
    # the tuned kernels (nbasis and nrhs multiples of 4): 8 sites per CTA with a ragged last chunk and ragged row tiles; the widest
    # promote tiling (16 column groups) with the generic project beside it; complex128 with 5 column groups
    (37, 70, 8, 4, "c64"),
    (5, 33, 64, 64, "c64"),
    (11, 129, 48, 20, "c128"),
    (300, 64, 32, 16, "c64"),
])
def test_project_and_promote_match_oracle(Vc, vb, nb, s, dtype):
    rng = np.random.default_rng(Vc + vb + nb + s)
    Bas, F, Cc = _rand(rng, dtype, Vc, vb, nb), _rand(rng, dtype, Vc, vb, s), _rand(rng, dtype, Vc, nb, s)
    dev = lambda a: torch.from_numpy(a.astype(NP_DTYPE[dtype])).cuda()
    P = cm.block_project(dev(Bas), dev(F)).cpu().numpy().astype(np.complex128)
    Q = cm.block_promote(dev(Bas), dev(Cc)).cpu().numpy().astype(np.complex128)
    assert rel_err_cols(P.reshape(-1, 1, s), transfer_oracle.project(Bas, F).reshape(-1, 1, s)) <= TOL[dtype]
    assert rel_err_cols(Q.reshape(-1, 1, s), transfer_oracle.promote(Bas, Cc).reshape(-1, 1, s)) <= TOL[dtype]


def test_orthonormal_basis_round_trip_on_the_device():
    rng = np.random.default_rng(5)
    Vc, vb, nb, s = 16, 48, 8, 4
    Bas = np.stack([np.linalg.qr(rng.standard_normal((vb, nb)) + 1j * rng.standard_normal((vb, nb)))[0] for _ in range(Vc)])
    Cc = _rand(rng, "c128", Vc, nb, s)
    d = lambda a: torch.from_numpy(a).cuda()
    back = cm.block_project(d(Bas), cm.block_promote(d(Bas), d(Cc))).cpu().numpy()
    assert np.allclose(back, Cc, atol=1e-13)
