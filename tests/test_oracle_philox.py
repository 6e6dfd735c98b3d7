"""Pins for the oracle's random numbers (O4): Philox4x32-10 known answers, the uniform map,
and the uniform-on-S^2 trial spin."""
import os

import numpy as np


def test_philox_known_answers(oracle):
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert oracle.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_counter_sensitivity(oracle):
    # every counter word and key word changes the output (a dropped word in the keying would not)
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] ^= 1
        assert oracle.philox4x32_10(c, [5, 6]) != base
    assert oracle.philox4x32_10([1, 2, 3, 4], [4, 6]) != base
    assert oracle.philox4x32_10([1, 2, 3, 4], [5, 7]) != base


def test_keying_matches_contract(oracle):
    # DESIGN.md R9: key = (seed_lo, seed_hi); ctr = (site, replica, step_lo, step_hi | tag << 31)
    seed, site, rep, step = 0x0123456789ABCDEF, 77, 5, (3 << 32) | 9
    for tag in (0, 1):
        _, _, raw = oracle.trial_draw(seed, site, rep, step, tag)
        want = oracle.philox4x32_10([site, rep, 9, 3 | (tag << 31)], [0x89ABCDEF, 0x01234567])
        assert raw == want


def test_uniform_map_and_sphere(oracle):
    n = 20000
    S = np.empty((n, 3))
    U = np.empty(n)
    for i in range(n):
        sp, u, raw = oracle.trial_draw(12345, i, 0, 7)
        S[i], U[i] = sp, u
        # u is an odd multiple of 2^-24 strictly inside (0, 1), from word 2
        m = u * 2 ** 24
        assert m == int(m) and int(m) % 2 == 1 and 0 < u < 1
        assert int(m) == 2 * (raw[2] >> 9) + 1
        # z = 2 u0 - 1 from word 0, azimuth 2 pi u1 from word 1
        u0 = (2 * (raw[0] >> 9) + 1) / 2 ** 24
        u1 = (2 * (raw[1] >> 9) + 1) / 2 ** 24
        assert sp[2] == 2 * u0 - 1
        assert abs(np.arctan2(sp[1], sp[0]) % (2 * np.pi) - 2 * np.pi * u1) < 1e-9
    assert np.max(np.abs(np.linalg.norm(S, axis=1) - 1)) < 1e-14
    # uniform on S^2: <s> = 0, <s_a s_b> = delta_ab / 3  (4-sigma bands)
    assert np.all(np.abs(S.mean(0)) < 4 * np.sqrt(1 / 3 / n))
    C = S.T @ S / n
    assert np.max(np.abs(C - np.eye(3) / 3)) < 4 * np.sqrt(4 / 45 / n) + 1e-3
    assert abs(U.mean() - 0.5) < 4 * np.sqrt(1 / 12 / n)
    # Archimedes: z uniform on [-1, 1]
    hist, _ = np.histogram(S[:, 2], bins=10, range=(-1, 1))
    assert np.all(np.abs(hist - n / 10) < 5 * np.sqrt(n / 10))


def test_init_spins(oracle):
    s = oracle.init_spins(8, 2, 0, 99)
    assert np.max(np.abs((s ** 2).sum(1) - 1)) < 1e-14
    sp, _, _ = oracle.trial_draw(99, 8 * 3 + 5, 1, 0, tag=1)
    assert np.array_equal(s[1, :, 3, 5], sp)
    z = oracle.init_spins(4, 1, 1, 0)
    assert np.all(z[:, 2] == 1) and np.all(z[:, :2] == 0)
