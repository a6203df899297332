"""CPU oracle for the multi-RHS block project / promote between grids (first half), numpy,
complex128.  TEST INFRASTRUCTURE ONLY.

Definitions written out (section 2.5.1, "one matrix multiply for each coarse lattice site"):
    project (Eq. 14):  for all x^c:  C[x^c] (N_basis x N_rhs)  = B[x^c]^dagger (N_basis x V_block) . F[x^c] (V_block x N_rhs)
    promote (Eq. 15):  for all x^c:  F[x^c] (V_block x N_rhs)  = B[x^c] (V_block x N_basis) . C[x^c] (N_basis x N_rhs)
Layouts ("BLAS ready"; reading R19): the fine field is held block by block, basis [Vc][V_block][N_basis],
fine vectors [Vc][V_block][N_rhs], coarse vectors [Vc][N_basis][N_rhs] (the coarse-operator block layout).
Pins: tests/test_oracle_transfer.py (orthonormal basis: project(promote(C)) = C and promote.project is the orthogonal
projector; adjointness <promote(C), F> = <C, project(F)>; explicit loops on a tiny case).
"""
from __future__ import annotations

import numpy as np


def project(Basis, F):
    return np.einsum("xvk,xvr->xkr", np.conj(np.asarray(Basis, dtype=np.complex128)), np.asarray(F, dtype=np.complex128))


def promote(Basis, C):
    return np.einsum("xvk,xkr->xvr", np.asarray(Basis, dtype=np.complex128), np.asarray(C, dtype=np.complex128))
