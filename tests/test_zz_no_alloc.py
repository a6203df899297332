"""-m gpu test of coarse_block_gram_noalloc (include/coarse_mrhs.h): the Gram product G = U^H W for callers
that cannot call cudaMalloc -- no handle, the reduction scratch in a static device array of 4 MiB, nrhs <= 32.

Collected last on purpose (the file name): the suite runs with pytest -x, and a failure here must not hide another test.
Checks: the output against the existing path (coarse_block_gram through a handle) within the Gram tolerance of
test_gpu_blockcg.py (|dG|_ab <= 2e-6 ||u_a|| ||w_b|| for complex64, 1e-13 for complex128; reading R11) and against the CPU oracle,
on TWO calls in a row with different inputs and widths (the array keeps the first call's contents: the second call, with a
smaller and then a larger footprint, must not see them); that a call allocates no device memory; the size limit's error.
"""
import numpy as np
import pytest
import torch

from gpu_common import to_dev, to_np
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402

TOL = {"c64": 2e-6, "c128": 1e-13}


def _block(rng, n, s, name):
    z = (rng.standard_normal((n, s)) + 1j * rng.standard_normal((n, s))) / np.sqrt(2)
    return z.astype(np.complex64).astype(np.complex128) if name == "c64" else z


def _err(G, Gref, U, W):
    return float(np.max(np.abs(G - Gref) / np.outer(np.linalg.norm(U, axis=0), np.linalg.norm(W, axis=0))))


def _existing_path(U, W, name):
    s = U.shape[1]
    A = torch.zeros((1, 81, 4, 4), dtype=torch.complex64 if name == "c64" else torch.complex128, device="cuda")
    op = cm.CoarseOperator((1, 1, 1, 1), A, s)
    G = to_np(op.gram(to_dev(U, name), to_dev(W, name)))
    op.close()
    return G


@pytest.mark.parametrize("name", ["c64", "c128"])
def test_noalloc_gram_matches_the_existing_path_on_two_calls_in_a_row(name):
    rng = np.random.default_rng(20240903)
    # (rows, width): a long block that uses all 256 partials at the largest width, then a short narrow one (few partials, the rest
    # of the array still holds the first call's), then a ragged one
    cases = [(70_001, 32), (777, 5), (20_011, 16)]
    blocks = [(_block(rng, n, s, name), _block(rng, n, s, name)) for n, s in cases]
    expected = [_existing_path(U, W, name) for U, W in blocks]
    dev = [(to_dev(U, name), to_dev(W, name), torch.empty((U.shape[1], U.shape[1]), dtype=torch.complex128, device="cuda")) for U, W in blocks]
    torch.cuda.synchronize()
    launches0, bytes0 = cm.launch_count(), torch.cuda.memory_allocated()
    free0 = torch.cuda.mem_get_info()[0]
    for Ud, Wd, Gd in dev:                              # back to back on one stream, no synchronisation in between
        cm.block_gram_noalloc(Ud, Wd, Gd)
    torch.cuda.synchronize()
    assert cm.launch_count() - launches0 == 2 * len(cases)          # our kernels ran: two per call
    assert torch.cuda.memory_allocated() == bytes0                   # nothing through torch's allocator
    assert torch.cuda.mem_get_info()[0] >= free0                     # and nothing through cudaMalloc behind it
    for (U, W), Gref, (_, _, Gd) in zip(blocks, expected, dev):
        G = to_np(Gd)
        assert _err(G, Gref, U, W) <= TOL[name]
        assert _err(G, oracle.gram(U, W), U, W) <= TOL[name]
    # the same call again gives the same bits (fixed partition, fixed order, no atomics), whatever the array held before
    Ud, Wd, Gd = dev[0]
    G1 = to_np(Gd).copy()
    cm.block_gram_noalloc(Ud, Wd, Gd)
    assert np.array_equal(to_np(Gd), G1)


def test_noalloc_gram_single_row_and_width_one():
    rng = np.random.default_rng(7)
    for n, s in ((1, 1), (1, 32), (300, 1)):
        U, W = _block(rng, n, s, "c128"), _block(rng, n, s, "c128")
        Gd = torch.full((s, s), complex(np.nan, np.nan), dtype=torch.complex128, device="cuda")
        cm.block_gram_noalloc(to_dev(U, "c128"), to_dev(W, "c128"), Gd)
        assert _err(to_np(Gd), oracle.gram(U, W), U, W) <= TOL["c128"]


def test_noalloc_gram_rejects_widths_beyond_its_static_scratch():
    assert cm.binding.NOALLOC_MAX_NRHS == 32
    s = cm.binding.NOALLOC_MAX_NRHS + 1
    U = torch.zeros((64, s), dtype=torch.complex64, device="cuda")
    G = torch.full((s, s), 7.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(cm.CoarseError) as e:
        cm.block_gram_noalloc(U, U.clone(), G)
    assert "COARSE_NOALLOC_MAX_NRHS" in str(e.value) and "status -2" in str(e.value)
    assert bool((G == 7.0).all())                                     # outputs untouched on COARSE_UNSUPPORTED
