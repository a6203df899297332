"""-m gpu parity: the block-CG kernels and block_cg_solve (CUDA, through the C ABI) against the CPU oracle.

Bars (BASELINE.json north_star): same true residual as the oracle (<= tol), iteration counts within 5 %
(with 7-9 iteration solves that means equal), solution within the
dtype's tolerance scaled by what the stopping tolerance allows.
"""
import numpy as np
import pytest
import torch

from gpu_common import TOL, TORCH_DTYPE, host_case, to_dev, to_np
from helpers import rel_err_cols
from inputs import synth
from oracle import oracle

pytestmark = pytest.mark.gpu

import paper_2409_03904_b200 as cm  # noqa: E402


def _dummy_op(nrhs_max, dtype):
    A = torch.zeros((1, 81, 4, 4), dtype=TORCH_DTYPE[dtype], device="cuda")
    return cm.CoarseOperator((1, 1, 1, 1), A, nrhs_max)


def _rand_block(rng, n, s):
    z = (rng.standard_normal((n, s)) + 1j * rng.standard_normal((n, s))) / np.sqrt(2)
    return z.astype(np.complex64).astype(np.complex128)      # float32-exact


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("n,s", [(1, 1), (37, 3), (5000, 4), (40001, 8), (30011, 12), (20000, 16), (9001, 33), (12345, 64)])
def test_gram_matches_oracle(dtype, n, s):
    rng = np.random.default_rng(n + s)
    U, W = _rand_block(rng, n, s), _rand_block(rng, n, s)
    op = _dummy_op(s, dtype)
    G = to_np(op.gram(to_dev(U, dtype), to_dev(W, dtype)))
    Gu = to_np(op.gram(to_dev(U, dtype), to_dev(U, dtype)))
    op.close()
    ref, refu = oracle.gram(U, W), oracle.gram(U, U)
    scale = np.sqrt(np.outer(np.diag(refu).real, np.diag(oracle.gram(W, W)).real))   # |G_ab| <= ||u_a|| ||w_b||
    tol = 1e-13 if dtype == "c128" else 2e-6
    assert np.max(np.abs(G - ref) / scale) <= tol
    assert np.max(np.abs(Gu - refu) / np.sqrt(np.outer(np.diag(refu).real, np.diag(refu).real))) <= tol


@pytest.mark.parametrize("dtype", ["c64", "c128"])
@pytest.mark.parametrize("n,s", [(1, 1), (130, 4), (7001, 8), (5003, 12), (4099, 16), (3000, 33), (2049, 64)])
@pytest.mark.parametrize("beta", [0.0, 1.0])
def test_rotate_matches_oracle(dtype, n, s, beta):
    rng = np.random.default_rng(n * 3 + s)
    U, W = _rand_block(rng, n, s), _rand_block(rng, n, s)
    K = _rand_block(rng, s, s)
    op = _dummy_op(s, dtype)
    Wd = to_dev(W, dtype)
    op.rotate(to_dev(U, dtype), torch.from_numpy(K).cuda(), Wd, beta)
    op.close()
    ref = oracle.block_rotate(U, K, W, beta)
    assert rel_err_cols(to_np(Wd).reshape(n, 1, s), ref.reshape(n, 1, s)) <= TOL[dtype]


@pytest.mark.parametrize("s", [1, 2, 4, 8, 12, 16, 33, 64])
def test_small_dense_algebra_matches_oracle(s):
    rng = np.random.default_rng(s)
    Z = rng.standard_normal((3 * s + 5, s)) + 1j * rng.standard_normal((3 * s + 5, s))
    G = Z.conj().T @ Z + 0.1 * np.eye(s)
    Gd = torch.from_numpy(G).cuda()
    S, Sinv, info = cm.small_cholesky(Gd)
    M, info2 = cm.small_hpd_inverse(Gd)
    st, S_ref = oracle.cholesky_upper(G)
    assert info == 0 and info2 == 0 and st == 0
    nrm = np.linalg.norm
    assert nrm(to_np(S) - S_ref) <= 1e-12 * nrm(S_ref)
    assert nrm(to_np(Sinv) - oracle.upper_inverse(S_ref)) <= 1e-10 * nrm(oracle.upper_inverse(S_ref))
    assert nrm(to_np(M) - oracle.hpd_inverse(G)[1]) <= 1e-10 * nrm(oracle.hpd_inverse(G)[1])
    assert np.all(np.tril(to_np(S), -1) == 0) and np.all(np.diag(to_np(S)).real > 0)


def test_small_cholesky_reports_breakdown():
    G = np.diag([1.0, -1.0, 2.0]).astype(np.complex128)
    _, _, info = cm.small_cholesky(torch.from_numpy(G).cuda())
    assert info == cm.binding.BREAKDOWN and oracle.cholesky_upper(G)[0] == oracle.BREAKDOWN


def _solve_both(dims, nb, s, dtype, seed, factor, tol, X0=None, maxiter=200, A=None, B=None):
    if A is None:
        A, c, _, B = host_case(dims, nb, s, seed, factor)
    ref = oracle.block_cg(dims, A, B, X0=X0, tol=tol, maxiter=maxiter)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    Xd = to_dev(np.zeros_like(B) if X0 is None else X0, dtype)
    out = op.block_cg(to_dev(B, dtype), Xd, tol=tol, maxiter=maxiter)
    op.close()
    out["X"] = to_np(out["X"])
    return out, ref


def _check_solve(out, ref, tol, dtype):
    assert out["status"] == ref["status"] == 0
    # iteration counts within 5 %  (BASELINE.json north_star)
    assert abs(out["iterations"] - ref["iterations"]) <= 0.05 * ref["iterations"], (out["iterations"], ref["iterations"])
    # same true residual: both reach the tolerance
    assert max(out["rel_res_true"]) <= tol * (1.0 + 1e-3) + (0 if dtype == "c128" else 2e-7)
    assert np.max(ref["true_rel"]) <= tol * (1.0 + 1e-3)
    # residual histories agree while they are above the dtype's attainable accuracy
    k = min(out["iterations"], ref["iterations"])
    h_ref = ref["history"].max(axis=1)[:k + 1]
    h_gpu = np.array(out["history"][:k + 1])
    floor = 1e-12 if dtype == "c128" else 1e-5
    mask = h_ref > floor
    assert np.allclose(h_gpu[mask], h_ref[mask], rtol=1e-6 if dtype == "c128" else 5e-2)
    # solutions agree to what the stopping tolerance allows
    assert rel_err_cols(out["X"], ref["X"]) <= max(10 * tol, TOL[dtype])


def test_block_cg_baseline_config1(cfg1):
    out, ref = _solve_both(cfg1["dims"], 8, 4, "c128", None, None, cfg1["tol"], A=cfg1["A"], B=cfg1["B"])
    _check_solve(out, ref, cfg1["tol"], "c128")
    assert out["iterations"] == ref["iterations"] == 7
    assert np.allclose(out["history"], ref["history"].max(axis=1), rtol=1e-6)


@pytest.mark.parametrize("dims,nb,s,dtype,factor,tol", [
    ((4, 4, 4, 8), 24, 8, "c128", 1.05, 1e-10),      # BASELINE configs[1] shape on a smaller lattice
    ((4, 4, 4, 8), 32, 16, "c64", 1.02, 1e-6),       # configs[2]
    ((3, 3, 3, 5), 32, 64, "c64", 1.02, 1e-6),       # configs[3] widest sweep point, ragged tail
    ((4, 4, 4, 4), 24, 64, "c64", 1.01, 1e-6),       # configs[4]
    ((3, 3, 2, 4), 13, 5, "c128", 1.05, 1e-10),      # generic stencil kernel underneath
    ((4, 4, 4, 4), 32, 1, "c64", 1.02, 1e-6),        # s = 1: plain CG
])
def test_block_cg_matches_oracle(dims, nb, s, dtype, factor, tol):
    out, ref = _solve_both(dims, nb, s, dtype, seed=77, factor=factor, tol=tol)
    _check_solve(out, ref, tol, dtype)


def test_block_cg_nonzero_initial_guess_zero_column_and_maxiter(cfg1):
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"].copy()
    X0 = synth.make_block(dims, 8, 4, 5, synth.TAG_U)
    out, ref = _solve_both(dims, 8, 4, "c128", None, None, 1e-10, X0=X0, A=A, B=B)
    _check_solve(out, ref, 1e-10, "c128")
    # maxiter hit: NOT_CONVERGED, outputs valid and equal to the oracle's after the same number of iterations
    out, ref = _solve_both(dims, 8, 4, "c128", None, None, 1e-10, maxiter=3, A=A, B=B)
    assert out["status"] == ref["status"] == cm.binding.NOT_CONVERGED and out["iterations"] == ref["iterations"] == 3
    assert rel_err_cols(out["X"], ref["X"]) <= 1e-12
    assert np.allclose(out["rel_res_true"], ref["true_rel"], rtol=1e-6)


def test_block_cg_already_converged_and_host_entry_point(cfg1):
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"]
    ref = oracle.block_cg(dims, A, B, tol=1e-10, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), 4)
    out = op.block_cg(to_dev(B, "c128"), to_dev(ref["X"], "c128"), tol=1e-9)      # X0 = solution
    assert out["iterations"] == 0 and out["status"] == 0
    Bh = torch.from_numpy(B.copy()).pin_memory()
    Xh = torch.zeros_like(Bh).pin_memory()
    out = op.block_cg_host(Bh, Xh, tol=1e-10)
    op.close()
    assert out["iterations"] == ref["iterations"]
    assert rel_err_cols(Xh.numpy(), ref["X"]) <= 1e-9


@pytest.mark.parametrize("index,nrhs", [(1, 8), (2, 16), (3, 16), (4, 64)])
def test_block_cg_full_size_properties(index, nrhs):
    """BASELINE configs[1] ... configs[4] at full size: the oracle cannot solve these in seconds, so check what
    holds at any size -- convergence flag, true residual <= tol (from the kernels' extra apply AND recomputed
    on sampled sites by the oracle), iteration count equal to the oracle's on the same construction at a
    reduced lattice (the spectrum of the synthetic operator does not depend on the volume: DESIGN.md)."""
    cfg = synth.config(index)
    dims, nb, dtype, tol = cfg["dims"], cfg["nbasis"], cfg["dtype"], cfg["tol"]
    esize = 8 if dtype == "c64" else 16
    need = synth.volume(dims) * (81 * nb * nb * esize * (2.1 if index == 4 else 3.1) + 12 * nb * nrhs * esize)
    if torch.cuda.mem_get_info()[0] < need:
        pytest.skip("not enough free device memory")
    A, c = cm.fill_synthetic(dims, nb, TORCH_DTYPE[dtype], cfg["seed"], cfg["factor"])
    B = cm.fill_block(dims, nb, nrhs, TORCH_DTYPE[dtype], cfg["seed"], synth.TAG_B)
    op = cm.CoarseOperator(dims, A, nrhs, flags=cm.binding.FLAG_TENSOR_ONLY if index == 4 else 0)
    out = op.block_cg(B, tol=tol, maxiter=100)
    assert out["status"] == 0 and max(out["rel_res_true"]) <= tol * 1.001 + (2e-7 if dtype == "c64" else 0.0)
    # sampled true residual through the oracle
    rng = np.random.default_rng(index)
    sites = np.sort(rng.choice(synth.volume(dims), size=16, replace=False)).astype(np.int64)
    idx = torch.from_numpy(sites).cuda()
    HX = oracle.apply(dims, A[idx].cpu().numpy(), to_np(out["X"]), sites=sites)
    Bs = to_np(B[idx])
    assert np.linalg.norm(Bs - HX) / np.linalg.norm(Bs) <= 10 * tol
    op.close()
    small = (4, 4, 4, 4)
    ref = oracle.block_cg(small, *[host_case(small, nb, nrhs, cfg["seed"], cfg["factor"])[i] for i in (0, 3)], tol=tol, maxiter=100)
    assert abs(out["iterations"] - ref["iterations"]) <= 1


def test_begin_step_end_equals_solve(cfg1):
    dims, A, B = cfg1["dims"], cfg1["A"], cfg1["B"]
    ref = oracle.block_cg(dims, A, B, tol=1e-10, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, "c128"), 4)
    Bd, Xd = to_dev(B, "c128"), to_dev(np.zeros_like(B), "c128")
    st, r0 = op.block_cg_begin(Bd, Xd, tol=1e-10)
    assert st == cm.binding.NOT_CONVERGED and abs(r0 - 1.0) < 1e-12
    op.block_cg_step(3)
    op.block_cg_step(ref["iterations"] - 3)
    out = op.block_cg_end()
    op.close()
    assert out["iterations"] == ref["iterations"] and out["status"] == 0
    assert rel_err_cols(to_np(Xd), ref["X"]) <= 1e-12
    assert np.allclose(out["rel_res_recursive"], ref["history"][-1], rtol=1e-6)
    assert max(out["rel_res_true"]) <= 1e-10


@pytest.mark.parametrize("dims,nb,s,dtype,tol", [
    ((4, 4, 4, 4), 32, 16, "c64", 1e-6),
    ((3, 3, 3, 5), 24, 8, "c128", 1e-10),
    ((3, 3, 2, 4), 13, 5, "c128", 1e-10),       # odd s: 8-byte cp.async chunks do not apply to complex128; ragged column groups
    ((3, 3, 2, 4), 16, 7, "c64", 1e-6),         # odd s in complex64: 8-byte chunks, ragged column groups
    ((3, 3, 3, 3), 32, 64, "c64", 1e-6),        # widest block: 4 x 4 register tiles, width-specialised kernels
    ((3, 3, 3, 3), 32, 48, "c64", 1e-6),        # 4 x 4 tiles with a run-time width
    ((3, 3, 3, 3), 24, 40, "c64", 1e-6),        # same, TF32 stencil kernel underneath
    ((3, 3, 3, 3), 8, 64, "c128", 1e-10),       # widest block in complex128 (tile height limited by shared memory)
    ((3, 3, 3, 3), 8, 33, "c128", 1e-10),       # s > 32 in complex128
])
def test_fused_passes_equal_the_unfused_kernel_sequence(dims, nb, s, dtype, tol):
    # the two fused passes of an iteration (bcg_fused1/2_kernel) against the six-kernel sequence (COARSE_FLAG_UNFUSED_LINALG)
    # and against the oracle: same iteration count, same residual history, same solution
    A, c, _, B = host_case(dims, nb, s, 91, 1.03)
    ref = oracle.block_cg(dims, A, B, tol=tol, maxiter=100)
    outs = []
    for flags in (0, cm.binding.FLAG_UNFUSED_LINALG):
        op = cm.CoarseOperator(dims, to_dev(A, dtype), s, flags=flags)
        out = op.block_cg(to_dev(B, dtype), to_dev(np.zeros_like(B), dtype), tol=tol, maxiter=100)
        op.close()
        out["X"] = to_np(out["X"])
        _check_solve(out, ref, tol, dtype)
        outs.append(out)
    assert outs[0]["iterations"] == outs[1]["iterations"]
    assert rel_err_cols(outs[0]["X"], outs[1]["X"]) <= (1e-12 if dtype == "c128" else 2e-6)
    k = outs[0]["iterations"]
    h0, h1 = np.array(outs[0]["history"][:k + 1]), np.array(outs[1]["history"][:k + 1])
    assert np.allclose(h0, h1, rtol=1e-9 if dtype == "c128" else 2e-2)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_zero_guess_option_equals_an_explicit_zero_start(dtype):
    # COARSE_SOLVE_ZERO_GUESS: X is an output only, R_0 = B, one apply less -- same iterates as X_0 = 0 passed explicitly
    dims, nb, s = (4, 4, 4, 4), 32, 16
    tol = 1e-10 if dtype == "c128" else 1e-6
    A, c, _, B = host_case(dims, nb, s, seed=55, factor=1.03)
    op = cm.CoarseOperator(dims, to_dev(A, dtype), s)
    Bd = to_dev(B, dtype)
    ref = op.block_cg(Bd, torch.zeros_like(Bd), tol=tol, maxiter=100)
    l0 = cm.launch_count()
    garbage = torch.full_like(Bd, float("nan"))
    out = op.block_cg(Bd, garbage, tol=tol, maxiter=100, zero_guess=True)
    assert out["status"] == ref["status"] == 0 and out["iterations"] == ref["iterations"]
    assert torch.equal(out["X"], ref["X"])
    assert np.array_equal(out["history"], ref["history"])
    # host entry point: X_host is not read
    Bh, Xh = Bd.cpu().pin_memory(), torch.full_like(Bd, float("nan")).cpu().pin_memory()
    outh = op.block_cg_host(Bh, Xh, tol=tol, maxiter=100, zero_guess=True)
    assert outh["iterations"] == ref["iterations"] and torch.equal(Xh, ref["X"].cpu())
    with pytest.raises(cm.binding.CoarseError):
        cm.binding._check(cm.lib().block_cg_solve_ex(op._h, Bd.data_ptr(), garbage.data_ptr(), s, tol, 10, 2, None, None))
    op.close()


def test_steps_interleaved_with_other_applies_on_the_same_handle():
    # pass 2 of an iteration leaves the column maxima of D for the next stencil launch (FP16-split kernel); an unrelated apply
    # on the same handle in between must not corrupt them
    dims, nb, s = (4, 4, 4, 4), 32, 16
    A, c, X, B = host_case(dims, nb, s, seed=61, factor=1.03)
    ref = oracle.block_cg(dims, A, B, tol=1e-6, maxiter=100)
    op = cm.CoarseOperator(dims, to_dev(A, "c64"), s)
    Bd, Xd = to_dev(B, "c64"), to_dev(np.zeros_like(B), "c64")
    big = to_dev(1e6 * X, "c64")
    st, r0 = op.block_cg_begin(Bd, Xd, tol=1e-6)
    for k in range(ref["iterations"]):
        op.block_cg_step(1)
        Y = op.apply(big)                      # very different column maxima
    out = op.block_cg_end()
    op.close()
    assert out["status"] == 0 and max(out["rel_res_true"]) <= 1e-6 + 3e-7
    assert rel_err_cols(to_np(Xd), ref["X"]) <= 1e-5


@pytest.mark.parametrize("s", [32, 64])
def test_first_solve_of_a_fresh_process_at_this_width(s):
    # Kernel attributes (dynamic shared memory opt-in) are set lazily per (device, kernel): a width whose s x s kernels sit
    # exactly at the 48 KB default (s = 32: 3 matrices x 16 KB + the kernel's static part) must work as the FIRST launch of
    # a process, not only after a wider solve has raised the limit (bench.py's Nrhs sweep runs 1, 4, 8, 16, 32, 64 in order).
    import subprocess
    import sys
    code = (
        "import sys, numpy as np, torch\n"
        f"sys.path.insert(0, {repr(str(__import__('os').path.dirname(__import__('os').path.dirname(__import__('os').path.abspath(__file__)))))})\n"
        "import paper_2409_03904_b200 as cm\n"
        "from inputs import synth\n"
        f"dims, nb, s = (4, 4, 2, 2), 32, {s}\n"
        "A, c = synth.make_operator(dims, nb, 5, 1.02)\n"
        "B = synth.make_block(dims, nb, s, 5, synth.TAG_B)\n"
        "op = cm.CoarseOperator(dims, torch.from_numpy(A.astype(np.complex64)).cuda(), 64)\n"
        "out = op.block_cg(torch.from_numpy(B.astype(np.complex64)).cuda(), tol=1e-6, maxiter=50)\n"
        "assert out['status'] == 0 and max(out['rel_res_true']) <= 1.3e-6, out\n"
        "print('ok', out['iterations'])\n")
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "ok" in r.stdout, r.stdout + r.stderr


@pytest.mark.parametrize("dims,nb,s,dtype,tol", [((4, 4, 4, 4), 8, 4, "c128", 1e-10), ((4, 4, 2, 2), 32, 16, "c64", 1e-6), ((3, 3, 2, 4), 13, 5, "c128", 1e-10)])
def test_graph_replay_of_an_iteration_equals_eager_launches(dims, nb, s, dtype, tol):
    # small blocks replay iterations 2, 3, ... of a solve as a CUDA graph (captured once per handle, block and width): same kernels in
    # the same order, so solution, iteration count and residual history are bit-identical to COARSE_FLAG_NO_GRAPH; repeated
    # solves on the handle (the graph is reused), a solve into another block (re-captured) and the begin/step/end form as well
    A, c, X0, B = host_case(dims, nb, s, seed=123, factor=1.05)
    outs = {}
    for name, flags in (("graph", 0), ("eager", cm.binding.FLAG_NO_GRAPH)):
        op = cm.CoarseOperator(dims, to_dev(A, dtype), s, flags=flags)
        Bd = to_dev(B, dtype)
        X1, X2 = torch.zeros_like(Bd), torch.zeros_like(Bd)
        r1 = op.block_cg(Bd, X1, tol=tol, maxiter=60)
        l0 = cm.launch_count()
        r2 = op.block_cg(Bd, X1.zero_(), tol=tol, maxiter=60)             # same block again
        launches = cm.launch_count() - l0
        r3 = op.block_cg(Bd, X2, tol=tol, maxiter=60)                     # another block
        st, _ = op.block_cg_begin(Bd, X2.zero_(), tol=1e-300)
        op.block_cg_step(r1["iterations"])
        r4 = op.block_cg_end()
        outs[name] = (r1, r2, r3, r4, to_np(X1), to_np(X2), launches)
        op.close()
    g, e = outs["graph"], outs["eager"]
    ref = oracle.block_cg(dims, A, B, tol=tol, maxiter=60)
    for k in range(3):
        assert g[k]["iterations"] == e[k]["iterations"] == ref["iterations"] >= 3
        assert g[k]["history"] == e[k]["history"]
        assert g[k]["rel_res_true"] == e[k]["rel_res_true"]
    assert np.array_equal(g[4], e[4]) and np.array_equal(g[5], e[5])
    assert g[3]["rel_res_recursive"] == e[3]["rel_res_recursive"]
    assert g[6] == e[6]                                                   # the launch counter counts the kernels of a replayed graph too
