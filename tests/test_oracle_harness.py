"""The long-run harness's fp64 FFT field (tests/longrun_harness.py) pinned to the oracle's
plain direct sum before anything relies on it, and the harness chain pinned to the oracle's own half-sweep."""
import numpy as np

from longrun_harness import fft_field_fp64, spectral_table, z_scores


def rand_spins(rng, R, L):
    s = rng.standard_normal((R, 3, L, L))
    return s / np.sqrt((s ** 2).sum(axis=1, keepdims=True))


def test_fft_field_equals_direct_sum(oracle):
    rng = np.random.default_rng(0)
    for L in (4, 8, 32):
        W = oracle.build_tensor_ewald(L)
        s = rand_spins(rng, 3, L)
        assert np.max(np.abs(fft_field_fp64(spectral_table(W), s) - oracle.dipole_field(W, s))) < 1e-12
    # a table with no symmetry at all fixes the direction rho = m - n and the xy mixing
    W = rng.standard_normal((4, 8, 8))
    s = rand_spins(rng, 2, 8)
    assert np.max(np.abs(fft_field_fp64(spectral_table(W), s) - oracle.dipole_field(W, s))) < 1e-12


def test_chain_with_fft_field_tracks_the_plain_oracle(oracle):
    """20 half-sweeps of the harness chain (field by FFT, decisions by oracle_halfsweep_given_field) against
    oracle_halfsweep (field by direct sum): identical decisions and states (a field difference of 1e-13 flips a
    decision only if a margin lies that close to zero)."""
    rng = np.random.default_rng(1)
    L, R, J, g, K2, K4 = 8, 4, 1.0, 0.2, 0.6, 0.1
    T = np.linspace(0.3, 1.5, R)
    W = oracle.build_tensor_ewald(L)
    Mh = spectral_table(W)
    a = rand_spins(rng, R, L)
    b = a.copy()
    for step in range(20):
        fa = oracle.halfsweep(W, a, T, 3, step, J, g, K2, K4, want=("accept",))
        fb = oracle.halfsweep_given_field(W, b, fft_field_fp64(Mh, b), T, 3, step, J, g, K2, K4, want=("accept",))
        assert np.array_equal(fa["accept"], fb["accept"])
        assert np.array_equal(a, b)


def test_z_scores():
    rng = np.random.default_rng(2)
    a = 1.0 + 0.1 * rng.standard_normal((4000, 2, 4))
    b = 1.0 + 0.1 * rng.standard_normal((4000, 2, 4))
    z, diff, sigma = z_scores(a, b)
    assert np.all(z < 4.5) and np.allclose(sigma, 0.1 * np.sqrt(2 / 4000), rtol=0.1)
    z, _, _ = z_scores(a + 0.05, b)                      # a bias of 0.05 = 22 sigma is seen
    assert np.all(z > 15)
