"""Pins of the oracle's restatement of the paper's own update schedule (section 3.1,
App. A :307-361; the approximation of section 3.2, eq. 8; the Ising move of App. B)."""
import numpy as np


def rand_spins(rng, R, L):
    s = rng.standard_normal((R, 3, L, L))
    return s / np.sqrt((s ** 2).sum(axis=1, keepdims=True))


def wmat(W, rx, ry):
    return np.array([[W[0, ry, rx], W[1, ry, rx], 0.0], [W[1, ry, rx], W[2, ry, rx], 0.0], [0.0, 0.0, W[3, ry, rx]]])


def test_update_sites_are_the_stride_l_sublattice(oracle):
    """n = (L/l)^2 sites, i = (a l, b l) + i_1 with i_1 in [0, l)^2, each exactly once."""
    rng = np.random.default_rng(0)
    L, R = 12, 2
    W = oracle.build_tensor_ewald(L)
    for l in (2, 3, 4, 6, 12):
        for p in range(5):
            s = rand_spins(rng, R, L)
            out = oracle.sublattice_pass(W, s, 1.0, 77, p, l, 1.0, 0.1, 0.5, 0.0)
            ox, oy = out["offset"]
            assert 0 <= ox < l and 0 <= oy < l and (ox, oy) == oracle.sublattice_offset(77, p, l)
            visited = np.abs(out["trial"]).sum(axis=1) > 0
            yy, xx = np.nonzero(visited[0])
            assert len(xx) == (L // l) ** 2
            assert np.all(xx % l == ox) and np.all(yy % l == oy)
            assert np.array_equal(visited[0], visited[1])


def test_offsets_cover_the_cell_uniformly(oracle):
    l = 4
    counts = np.zeros((l, l))
    for p in range(3200):
        ox, oy = oracle.sublattice_offset(5, p, l)
        counts[oy, ox] += 1
    assert counts.min() > 200 * 0.7 and counts.max() < 200 * 1.3     # 200 expected per cell, sigma 14


def test_single_site_pass_is_exact(oracle):
    """l = L: one update site per pass, no simultaneous flipping, hence no approximation:
    frozen == sequential bit for bit, and dE is the full-energy difference (eq. 7)."""
    rng = np.random.default_rng(1)
    L, R = 6, 3
    W = oracle.build_tensor_ewald(L)
    J, g, K2, K4 = 1.0, 0.3, 0.4, -0.1
    T = np.array([0.3, 1.0, 5.0])
    for p in range(6):
        s0 = rand_spins(rng, R, L)
        a, b = s0.copy(), s0.copy()
        fa = oracle.sublattice_pass(W, a, T, 9, p, L, J, g, K2, K4)
        fb = oracle.sublattice_pass(W, b, T, 9, p, L, J, g, K2, K4, sequential=True)
        assert np.array_equal(a, b) and np.array_equal(fa["margin"], fb["margin"])
        ox, oy = fa["offset"]
        n = oy * L + ox
        for r in range(R):
            new = s0[r:r + 1].copy()
            new[0, :, oy, ox] = fa["trial"][r, :, oy, ox]
            dE = oracle.energy(W, new, J, g, K2, K4)[0] - oracle.energy(W, s0[r:r + 1], J, g, K2, K4)[0]
            _, u, _ = oracle.trial_draw(9, n, r, p)
            assert abs(fa["margin"][r, oy, ox] - (dE / T[r] + np.log(u))) < 1e-11


def test_no_dipole_no_approximation(oracle):
    """g = 0: update sites are never nearest neighbours, so simultaneous == sequential."""
    rng = np.random.default_rng(2)
    L, R = 8, 2
    W = oracle.build_tensor_ewald(L)
    for l in (2, 4):
        s0 = rand_spins(rng, R, L)
        a, b = s0.copy(), s0.copy()
        for p in range(4):
            fa = oracle.sublattice_pass(W, a, 0.7, 3, p, l, 1.0, 0.0, 0.5, 0.1)
            fb = oracle.sublattice_pass(W, b, 0.7, 3, p, l, 1.0, 0.0, 0.5, 0.1, sequential=True)
            assert np.array_equal(fa["accept"], fb["accept"])
        assert np.array_equal(a, b)
        assert not np.array_equal(a, s0)


def test_eq8_error_of_simultaneous_flipping(oracle):
    """PAPER.md:118-125, eq. 8: H3 - H1 - (H2 - H0) = g delta_1 . W(rho_12) . delta_2.  With every
    move accepted (T huge), the sequential margin of the k-th update site differs from the frozen one by
    the couplings to the sites updated before it, in the order a fastest."""
    rng = np.random.default_rng(3)
    L, l, g, T = 8, 4, 0.25, 1e9
    W = oracle.build_tensor_ewald(L)
    s0 = rand_spins(rng, 1, L)
    a, b = s0.copy(), s0.copy()
    fa = oracle.sublattice_pass(W, a, T, 21, 0, l, 1.0, g, 0.3, 0.0)
    fb = oracle.sublattice_pass(W, b, T, 21, 0, l, 1.0, g, 0.3, 0.0, sequential=True)
    assert fa["accept"].sum() == 4 and fb["accept"].sum() == 4
    assert np.array_equal(a, b)                                  # same trials, all accepted
    ox, oy = fa["offset"]
    sites = [(ox + l * aa, oy + l * bb) for bb in range(2) for aa in range(2)]
    delta = [fa["trial"][0, :, y, x] - s0[0, :, y, x] for (x, y) in sites]
    for k, (xk, yk) in enumerate(sites):
        expect = 0.0
        for j in range(k):
            xj, yj = sites[j]
            expect += g * delta[j] @ wmat(W, (xk - xj) % L, (yk - yj) % L) @ delta[k]
        got = (fb["margin"][0, yk, xk] - fa["margin"][0, yk, xk]) * T
        assert abs(got - expect) < 1e-6 * max(1.0, abs(expect)), (k, got, expect)
    assert abs(delta[0] @ wmat(W, l, 0) @ delta[1]) > 1e-4       # the test is not vacuous


def test_ising_flip_move(oracle):
    """App. B: every accepted update is a complete reversal; an Ising state stays one and
    dE is the full-energy difference of eq. 19 (our sign convention, R7)."""
    rng = np.random.default_rng(4)
    L, l, R = 8, 4, 2
    W = oracle.build_tensor_ewald(L)
    J, g = 0.85, 1.0                                               # J / C_D = 1.7 of eq. 19 = 0.85 per bond (R22)
    s = np.zeros((R, 3, L, L))
    s[:, 2] = rng.choice([-1.0, 1.0], size=(R, L, L))
    for p in range(20):
        before = s.copy()
        out = oracle.sublattice_pass(W, s, 0.85 * g, 31, p, l, J, g, 0.0, 0.0, flip=True)
        assert np.all(np.abs(s[:, 2]) == 1.0) and np.all(s[:, :2] == 0.0)
        changed = s[:, 2] != before[:, 2]
        assert np.array_equal(changed, out["accept"].astype(bool))
    # one isolated flip (l = L): margin T - T ln u = E(after) - E(before)
    before = s.copy()
    out = oracle.sublattice_pass(W, s, 1e9, 31, 100, L, J, g, 0.0, 0.0, flip=True)
    ox, oy = out["offset"]
    for r in range(R):
        _, u, _ = oracle.trial_draw(31, oy * L + ox, r, 100)
        dE = oracle.energy(W, s[r:r + 1], J, g, 0.0, 0.0)[0] - oracle.energy(W, before[r:r + 1], J, g, 0.0, 0.0)[0]
        assert abs((out["margin"][r, oy, ox] - np.log(u)) * 1e9 - dE) < 1e-5


def test_ising_limit_matches_onsager(oracle):
    """With g = 0, K = 0 and the reversal move the stride-l schedule is plain Metropolis sampling of the square-lattice
    Ising model, whose energy per spin is known in closed form (Onsager 1944, evaluated here with scipy's complete
    elliptic integral): pins the oracle's acceptance rule, exchange sign and neighbour indexing, its random numbers
    and its energy to something that is neither the oracle nor the GPU.  L = 16 at temperatures well away from
    T_c = 2.269, where the finite lattice is within 1e-3 of the infinite one."""
    from scipy.special import ellipk
    L, l = 16, 8
    T = np.array([1.5, 1.8, 3.2, 4.0])
    R = len(T)
    b = 1.0 / T
    k = 2.0 * np.sinh(2 * b) / np.cosh(2 * b) ** 2
    exact = -(1.0 / np.tanh(2 * b)) * (1.0 + (2.0 / np.pi) * (2.0 * np.tanh(2 * b) ** 2 - 1.0) * ellipk(k * k))
    W = np.zeros((4, L, L))                                    # g = 0: the table is never used
    s = np.zeros((R, 3, L, L))
    s[:, 2] = 1.0
    burn, rec = 200, 1200
    E = np.empty((rec, R))
    p = 0
    for step in range(burn + rec):
        for _ in range(l * l):
            oracle.sublattice_pass(W, s, T, 2024, p, l, 1.0, 0.0, 0.0, 0.0, flip=True)
            p += 1
        if step >= burn:
            E[step - burn] = oracle.energy(W, s, 1.0, 0.0, 0.0, 0.0) / (L * L)
    mean = E.mean(axis=0)
    se = 3.0 * E.std(axis=0, ddof=1) / np.sqrt(rec)            # factor 3: consecutive sweeps are correlated
    assert np.all(np.abs(mean - exact) < 3 * se + 2e-3), (mean, exact, se)
