"""Shared plumbing of the -m gpu parity tests: seeded inputs -> device tensors, oracle -> numpy."""
import numpy as np
import torch

from inputs import synth

# tolerances of BASELINE.json north_star: relative norm-wise error per column
TOL = {"c128": 1e-12, "c64": 1e-5}
TORCH_DTYPE = {"c128": torch.complex128, "c64": torch.complex64}
NP_DTYPE = {"c128": np.complex128, "c64": np.complex64}


def to_dev(a: np.ndarray, dtype: str) -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(a.astype(NP_DTYPE[dtype]))).cuda()


def to_np(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().astype(np.complex128)


def host_case(dims, nb, s, seed, factor):
    """(A complex64 float32-exact, c, X complex128 float32-exact, B) from the seeded generator."""
    A, c = synth.make_operator(dims, nb, seed, factor)
    X = synth.make_block(dims, nb, s, seed, synth.TAG_X)
    B = synth.make_block(dims, nb, s, seed, synth.TAG_B)
    return A, c, X, B
