"""-m gpu parity: coarse_op_apply (CUDA, through the C ABI) against the CPU oracle, element by element.

Metric (BASELINE.json north_star): max over columns r of ||Y_gpu[:,r] - Y_or[:,r]||_2 / ||Y_or[:,r]||_2
<= 1e-12 (complex128) / 1e-5 (complex64; oracle arithmetic in complex128 on the same float32-exact inputs).
"""
import itertools

import numpy as np
import pytest
import torch

from gpu_common import TOL, TORCH_DTYPE, host_case, to_dev, to_np
from helpers import rel_err_cols, shifted_block
from inputs import synth
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _apply_gpu(dims, A, X, dtype, flags=0, nrhs_max=None):
    s = X.shape[-1]
    op = cm.CoarseOperator(dims, to_dev(A, dtype), nrhs_max or s, flags=flags)
    name = op.kernel_name(s)
    Y = to_np(op.apply(to_dev(X, dtype)))
    torch.cuda.synchronize()
    op.close()
    return Y, name


# every tiled kernel variant, on lattices that span many site groups and leave a ragged tail
# (3*3*3*5 = 135 sites: not a multiple of 2, 4 or 8), plus periodic wrap in every direction
TILED = [("c64", 32, 64), ("c64", 32, 32), ("c64", 32, 16), ("c64", 32, 8), ("c64", 32, 4), ("c64", 32, 1),
         ("c64", 24, 64), ("c64", 24, 16), ("c128", 24, 8), ("c128", 8, 4), ("c128", 32, 16)]


@pytest.mark.parametrize("dtype,nb,s", TILED)
@pytest.mark.parametrize("dims", [(3, 3, 3, 5), (4, 4, 4, 6)])
def test_tiled_variants_match_oracle(dtype, nb, s, dims):
    A, c, X, _ = host_case(dims, nb, s, seed=100 + nb + s, factor=1.05)
    Y, name = _apply_gpu(dims, A, X, dtype, flags=cm.binding.FLAG_NO_TENSOR)
    assert name.startswith("stencil_simt"), name
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= TOL[dtype]


@pytest.mark.parametrize("dtype,nb,s", [("c64", 32, 16), ("c128", 24, 8), ("c64", 24, 64)])
def test_without_diagonal_shift(dtype, nb, s):
    # c = 0: the dominant c*I term no longer scales errors of the 80 off-diagonal terms down in the norm
    dims = (3, 4, 3, 4)
    A, c, X, _ = host_case(dims, nb, s, seed=7, factor=0.0)
    assert c == 0.0
    Y, _ = _apply_gpu(dims, A, X, dtype)
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= TOL[dtype]


@pytest.mark.parametrize("dtype,nb,s,flags", [("c64", 32, 4, 2), ("c128", 8, 4, 0), ("c64", 5, 3, 0), ("c128", 24, 8, 1)])
def test_single_stencil_point_is_a_pure_shift_bit_exact(dtype, nb, s, flags):
    # A_p = delta_{p,p0} I  =>  Y(x) = X(x + delta_p0) exactly, for each of the 81 points, anisotropic lattice
    dims = (3, 4, 5, 2)
    V = synth.volume(dims)
    X = synth.make_block(dims, nb, s, 5, synth.TAG_X)
    off = synth.stencil_offsets()
    for p0 in list(range(0, 81, 7)) + [39, 40, 41, 80]:
        A = np.zeros((V, 81, nb, nb), dtype=np.complex64)
        A[:, p0] = np.eye(nb, dtype=np.complex64)
        Y, _ = _apply_gpu(dims, A, X, dtype, flags=flags)
        assert np.array_equal(Y, shifted_block(dims, X, off[p0])), p0


@pytest.mark.parametrize("p_only", [0, 13, 40, 67, 80])
def test_one_point_at_a_time_matches_oracle(p_only):
    dims, nb, s, dtype = (4, 3, 3, 5), 32, 16, "c64"
    A, c, X, _ = host_case(dims, nb, s, seed=9, factor=0.0)
    A1 = np.zeros_like(A)
    A1[:, p_only] = A[:, p_only]
    Y, _ = _apply_gpu(dims, A1, X, dtype)
    assert rel_err_cols(Y, oracle.apply(dims, A, X, p_only=p_only)) <= TOL[dtype]


# generic kernel: shapes without a tiled variant, extents 1 and 2 (stencil points alias and must ADD)
@pytest.mark.parametrize("dims,nb,s,dtype", [
    ((1, 1, 1, 1), 6, 2, "c128"), ((2, 2, 2, 2), 5, 1, "c128"), ((1, 2, 3, 1), 2, 7, "c64"),
    ((5, 1, 1, 2), 1, 1, "c128"), ((3, 3, 2, 4), 13, 11, "c64"), ((2, 3, 4, 3), 64, 64, "c64"),
    ((3, 2, 3, 3), 40, 33, "c128"), ((4, 4, 4, 4), 32, 12, "c64"),
])
def test_generic_kernel_matches_oracle(dims, nb, s, dtype):
    A, c, X, _ = host_case(dims, nb, s, seed=31, factor=1.1)
    Y, name = _apply_gpu(dims, A, X, dtype, flags=cm.binding.FLAG_NO_TENSOR)
    assert name.startswith("stencil_generic"), name
    assert rel_err_cols(Y, oracle.apply(dims, A, X)) <= TOL[dtype]


def test_forced_generic_equals_tiled_within_rounding():
    dims, nb, s, dtype = (4, 4, 2, 4), 32, 16, "c64"
    A, c, X, _ = host_case(dims, nb, s, seed=3, factor=1.02)
    Yt, nt = _apply_gpu(dims, A, X, dtype, flags=cm.binding.FLAG_NO_TENSOR)
    Yg, ng = _apply_gpu(dims, A, X, dtype, flags=cm.binding.FLAG_FORCE_GENERIC)
    assert nt.startswith("stencil_simt") and ng.startswith("stencil_generic")
    ref = oracle.apply(dims, A, X)
    assert rel_err_cols(Yt, ref) <= TOL[dtype] and rel_err_cols(Yg, ref) <= TOL[dtype]


def test_nrhs_below_nrhs_max_and_column_independence():
    # operator created for nrhs_max = 16; applying 4 of the columns gives those columns of the 16-wide result
    dims, nb, dtype = (4, 4, 4, 4), 32, "c64"
    A, c, X, _ = host_case(dims, nb, 16, seed=12, factor=1.02)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), 16)
    Y16 = to_np(op.apply(to_dev(X, dtype)))
    Y4 = to_np(op.apply(to_dev(X[:, :, 4:8], dtype)))
    op.close()
    ref = oracle.apply(dims, A, X)
    assert rel_err_cols(Y16, ref) <= TOL[dtype]
    assert rel_err_cols(Y4, ref[:, :, 4:8]) <= TOL[dtype]


def test_baseline_config1_and_host_entry_point(cfg1):
    dims = cfg1["dims"]
    A = cfg1["A"]
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), 4)
    ref = oracle.apply(dims, A, cfg1["X"])
    assert rel_err_cols(to_np(op.apply(to_dev(cfg1["X"], "c128"))), ref) <= TOL["c128"]
    Xh = torch.from_numpy(cfg1["X"]).pin_memory()
    Yh = torch.empty_like(Xh).pin_memory()
    op.apply_host(Xh, Yh)
    assert rel_err_cols(Yh.numpy(), ref) <= TOL["c128"]
    op.close()


def test_errors_are_reported_not_swallowed():
    dims, nb = (2, 2, 2, 2), 8
    A = torch.zeros((16, 81, nb, nb), dtype=torch.complex64, device="cuda")
    op = cm.CoarseOperator(dims, A, 4)
    X = torch.zeros((16, nb, 8), dtype=torch.complex64, device="cuda")
    with pytest.raises(cm.CoarseError) as e:
        op.apply(X)                                  # nrhs 8 > nrhs_max 4
    assert e.value.status == cm.binding.INVALID_ARG
    X = torch.zeros((16, nb, 4), dtype=torch.complex64, device="cuda")
    with pytest.raises(cm.CoarseError):
        op.apply(X, X)                               # aliasing
    # blocks that are not 16-byte aligned are refused before any kernel could fault on them (every kernel variant)
    for kind in ("c64", "c128"):
        dt = torch.complex64 if kind == "c64" else torch.complex128
        op2 = cm.CoarseOperator(dims, A.to(dt), 4)
        n = 16 * nb * 4
        odd = torch.zeros(n + 1, dtype=dt, device="cuda")[1:].view(16, nb, 4) if kind == "c64" else None
        if odd is not None:                          # complex64 offset by one element: 8-byte aligned only
            for args in ((odd, torch.zeros_like(X)), (X, odd)):
                with pytest.raises(cm.CoarseError) as e:
                    op2.apply(*args)
                assert e.value.status == cm.binding.INVALID_ARG
            with pytest.raises(cm.CoarseError) as e:
                op2.block_cg(odd, torch.zeros_like(X))
            assert e.value.status == cm.binding.INVALID_ARG
        op2.close()
    op.close()


# complex128 on the FP64 tensor path, lattices of 1 to 16 sites per warp: the kernel's BALANCED partition (stencil_dmma.cuh) cuts the
# (site, stencil point) sequence at equal counts, so two warps share most sites and add their parts into a zeroed Y.
# (6,6,6,6) with 8 warps per CTA: 1296 sites for 1184 warps (88.7 points each: almost every site is shared); (7,7,7,7) with 16.
@pytest.mark.parametrize("dims,nb,s", [((6, 6, 6, 6), 24, 8), ((6, 6, 6, 6), 16, 16), ((7, 7, 7, 7), 8, 8), ((6, 6, 6, 7), 24, 8)])
def test_dmma_balanced_partition_matches_oracle_and_is_reproducible(dims, nb, s):
    A, c, X, _ = host_case(dims, nb, s, seed=300 + nb + s, factor=1.05)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), s)
    assert op.kernel_name(s).startswith("stencil_dmma"), op.kernel_name(s)
    Xd = to_dev(X, "c128")
    Yd = torch.full_like(Xd, complex(np.nan, np.nan))        # the kernel's own zeroing, not the caller's
    op.apply(Xd, Yd)
    Y1 = to_np(Yd).copy()
    Yd.fill_(7.0)
    op.apply(Xd, Yd)
    Y2 = to_np(Yd)
    op.close()
    assert rel_err_cols(Y1, oracle.apply(dims, A, X)) <= TOL["c128"]
    assert np.array_equal(Y1, Y2)                            # two terms onto zero: the order of the atomic adds cannot show


def _sampled_sites(dims, n_random, rng):
    """corners / faces of the periodic lattice plus random interior sites"""
    L = dims
    picks = set()
    for c in itertools.product(*[(0, L[k] - 1) for k in range(4)]):
        picks.add(c[0] + L[0] * (c[1] + L[1] * (c[2] + L[2] * c[3])))
    V = synth.volume(dims)
    picks.update(int(v) for v in rng.integers(0, V, size=n_random))
    picks.add(V - 1)
    return np.array(sorted(picks), dtype=np.int64)


@pytest.mark.parametrize("index,nrhs", [(1, 8), (2, 16), (3, 16), (3, 1), (3, 4), (3, 32), (3, 64), (4, 64)])
def test_full_size_baseline_configs_on_sampled_sites(index, nrhs):
    """BASELINE.json configs[1..4] at full size in the launch configuration bench.py times: operator and
    block generated on the device (coarse_op_fill_synthetic), the oracle recomputes sampled sites from the
    device buffers' own bits (inputs, not results)."""
    cfg = synth.config(index)
    dims, nb, dtype = cfg["dims"], cfg["nbasis"], cfg["dtype"]
    need = synth.volume(dims) * 81 * nb * nb * (8 if dtype == "c64" else 16) * 2.1
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("not enough free device memory for this configuration")
    A, c = cm.fill_synthetic(dims, nb, TORCH_DTYPE[dtype], cfg["seed"], cfg["factor"])
    X = cm.fill_block(dims, nb, nrhs, TORCH_DTYPE[dtype], cfg["seed"], synth.TAG_X)
    # complex64: nbasis 32 -> paired-site split-FP16 kernel (nrhs 4 or a multiple of 8); nbasis 8/16/24 -> the split-FP16 kernel with
    # the X operand in tensor memory (any nrhs >= 4)
    tensor = dtype == "c64" and ((nrhs % 8 == 0 or nrhs == 4) if nb == 32 else nrhs >= 4)
    # the 49 GB configuration keeps one internal layout of A (the caller's copy is needed below for the oracle's sample)
    op = cm.CoarseOperator(dims, A, nrhs, flags=cm.binding.FLAG_TENSOR_ONLY if (tensor and index == 4) else 0)
    dmma = dtype == "c128" and nb % 8 == 0 and nrhs % 8 == 0          # complex128: the FP64 tensor path (mma.sync, SASS DMMA)
    assert op.kernel_name(nrhs).startswith(("stencil_h16<" if nb == 32 else "stencil_h16x<") if tensor else ("stencil_dmma" if dmma else "stencil_simt"))
    Y = op.apply(X)
    torch.cuda.synchronize()
    sites = _sampled_sites(dims, 24, np.random.default_rng(index))
    idx = torch.from_numpy(sites).cuda()
    A_s = A[idx].cpu().numpy()
    Y_s = to_np(Y[idx])
    Xh = to_np(X)
    # the device generator reproduces the host generator on the sampled sites (same integer hash)
    A_host = synth.stencil_matrices(dims, nb, cfg["seed"], sites)
    synth.add_shift(A_host, c)
    mism = np.count_nonzero(A_s.astype(np.complex64) != A_host)
    assert mism <= 1e-6 * A_host.size, mism
    ref = oracle.apply(dims, A_s, Xh, sites=sites)
    assert rel_err_cols(Y_s, ref) <= TOL[dtype]
    # property that holds at any size: the synthetic operator is Hermitian, <X, H X> is real
    ip = torch.sum(torch.conj(X) * Y, dim=(0, 1))
    assert float(torch.max(torch.abs(ip.imag) / torch.abs(ip.real))) <= (1e-12 if dtype == "c128" else 2e-5)
    op.close()
