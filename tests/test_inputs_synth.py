"""The seeded input generator: determinism, float32-exactness, distribution and Hermitian structure."""
import numpy as np

from inputs import synth


def test_deterministic_and_subset_consistent():
    dims, nb, seed = (3, 2, 4, 2), 4, 42
    A1 = synth.stencil_matrices(dims, nb, seed)
    A2 = synth.stencil_matrices(dims, nb, seed)
    assert np.array_equal(A1, A2)
    sites = np.array([5, 0, 47, 12])
    assert np.array_equal(synth.stencil_matrices(dims, nb, seed, sites), A1[sites])
    Afull, c = synth.make_operator(dims, nb, seed, 1.05)
    B = A1.copy()
    synth.add_shift(B, c)
    assert np.array_equal(Afull, B)
    assert c == synth.diagonal_shift(dims, nb, seed, 1.05)
    assert not np.array_equal(A1, synth.stencil_matrices(dims, nb, seed + 1))


def test_values_are_float32_exact_and_pairing_is_hermitian():
    dims, nb, seed = (3, 2, 4, 2), 4, 42
    A, c = synth.make_operator(dims, nb, seed, 1.02)
    assert A.dtype == np.complex64
    V = synth.volume(dims)
    for p in range(81):
        y = synth.shifted_sites(dims, np.arange(V), p)
        assert np.array_equal(A[:, p], np.conj(np.transpose(A[y, 80 - p], (0, 2, 1))))
    assert np.float32(c) == c and c > 0


def test_distribution_moments():
    z = synth.complex_normal(1, synth.TAG_X, np.arange(400000))
    assert abs(np.mean(np.abs(z) ** 2) - 1.0) < 0.01
    assert abs(np.mean(z.real ** 2) - 0.5) < 0.01 and abs(np.mean(z.imag ** 2) - 0.5) < 0.01
    assert abs(np.mean(z)) < 0.01 and abs(np.mean(z.real * z.imag)) < 0.01
    assert abs(np.mean(z.real ** 4) - 0.75) < 0.02          # Gaussian kurtosis: E x^4 = 3 sigma^4


def test_configs_match_baseline_shapes():
    import json, os
    base = json.load(open(os.path.join(os.path.dirname(__file__), "..", "BASELINE.json")))
    assert len(base["configs"]) == len(synth.CONFIGS) == 5
    vols = [256, 4096, 8192, 41472, 131072]
    for i, v in enumerate(vols):
        cfg = synth.config(i)
        assert synth.volume(cfg["dims"]) == v
        assert f"nbasis={cfg['nbasis']}" in base["configs"][i]
