"""Pins for the oracle's field, energy, single-spin dE, half-sweep and observables."""
import numpy as np
import pytest
from scipy.special import zeta

ZETA32 = zeta(1.5, 1.0)
BETA32 = (zeta(1.5, 0.25) - zeta(1.5, 0.75)) / 8.0
MADELUNG = 4.0 * ZETA32 * BETA32


def rand_spins(rng, R, L):
    v = rng.standard_normal((R, 3, L, L))
    return v / np.sqrt((v ** 2).sum(1, keepdims=True))


def brute_dipole_energy(s, A):
    """eq. 1 with explicit periodic images |a|,|b| <= A, written independently of
    the oracle: (1/2) sum over ordered pairs (n, m + G), n != m + G, of
    [s_n.s_m - 3 (s_n.rhat)(s_m.rhat)] / r^3, n and m in the cell."""
    L = s.shape[-1]
    ys, xs = np.divmod(np.arange(L * L), L)
    sv = s.reshape(3, L * L)
    a = np.arange(-A, A + 1) * L
    E = 0.0
    for n in range(L * L):
        for m in range(L * L):
            X = (xs[m] - xs[n]) + a[None, :]
            Y = (ys[m] - ys[n]) + a[:, None]
            r2 = (X * X + Y * Y).astype(np.float64)
            keep = r2 > 0
            r2 = np.where(keep, r2, 1.0)
            r = np.sqrt(r2)
            dot = sv[:, n] @ sv[:, m]
            sn_r = (sv[0, n] * X + sv[1, n] * Y) / r
            sm_r = (sv[0, m] * X + sv[1, m] * Y) / r
            E += (keep * (dot - 3 * sn_r * sm_r) / (r2 * r)).sum()
    return 0.5 * E


@pytest.mark.parametrize("L", [2, 4])
def test_energy_vs_brute_force_eq1(oracle, L):
    rng = np.random.default_rng(5 + L)
    s = rand_spins(rng, 1, L)
    W = oracle.build_tensor_ewald(L)
    _, parts = oracle.energy(W, s, J=0.0, g=1.0, K2=0.0, K4=0.0, parts=True)
    A1, A2 = 100, 200
    e1, e2 = brute_dipole_energy(s[0], A1), brute_dipole_energy(s[0], A2)
    x1, x2 = 1 / (A1 + .5), 1 / (A2 + .5)
    e_inf = (e2 * x1 - e1 * x2) / (x1 - x2)          # Richardson in the 1/(A+1/2) tail
    assert abs(parts[0, 2] - e_inf) < 5e-8 * L * L, (parts[0, 2], e1, e2, e_inf)


def test_uniform_states_closed_form(oracle):
    # all +z: E_dip/N = (g/2) sum' r^-3 for every L; all +x: -(g/2)/2 of that  (BASELINE.json pin)
    g = 0.1
    for L in (4, 8):
        W = oracle.build_tensor_ewald(L)
        s = np.zeros((2, 3, L, L))
        s[0, 2] = 1.0
        s[1, 0] = 1.0
        _, parts = oracle.energy(W, s, J=0.0, g=g, K2=0.0, K4=0.0, parts=True)
        assert abs(parts[0, 2] / L ** 2 - 0.5 * g * MADELUNG) < 1e-12
        assert abs(parts[1, 2] / L ** 2 + 0.25 * g * MADELUNG) < 1e-12
        h = oracle.dipole_field(W, s)
        assert np.max(np.abs(h[0, 2] - MADELUNG)) < 1e-11 and np.max(np.abs(h[0, :2])) < 1e-12


def test_field_is_the_plain_double_sum(oracle):
    # independent numpy evaluation of O2 through explicit index arithmetic
    rng = np.random.default_rng(11)
    L, R = 6, 2
    s = rand_spins(rng, R, L)
    W = oracle.build_tensor_ewald(L)
    h = oracle.dipole_field(W, s)
    x = np.arange(L)
    for (yn, xn) in ((0, 0), (2, 5), (5, 1)):
        ry = (x[:, None] - yn) % L
        rx = (x[None, :] - xn) % L
        for r in range(R):
            hx = (W[0][ry, rx] * s[r, 0] + W[1][ry, rx] * s[r, 1]).sum()
            hy = (W[1][ry, rx] * s[r, 0] + W[2][ry, rx] * s[r, 1]).sum()
            hz = (W[3][ry, rx] * s[r, 2]).sum()
            assert np.allclose(h[r, :, yn, xn], [hx, hy, hz], rtol=0, atol=1e-13)
    # colour mask: only (x+y) % 2 == colour is written
    h0 = oracle.dipole_field(W, s, colour=0)
    par = (x[:, None] + x[None, :]) % 2
    assert np.array_equal(h0[:, :, par == 0], h[:, :, par == 0]) and np.all(h0[:, :, par == 1] == 0)
    # sampled entry point agrees
    hs = oracle.dipole_field_sampled(W, s[1], [0, 17, 35])
    assert np.array_equal(hs[1], h[1, :, 17 // L, 17 % L])


def test_no_dipole_limit(oracle):
    # g = 0: all +z has E/N = -2J - K2 - K4 (each bond once, R8; sign convention R7)
    L = 6
    W = oracle.build_tensor_ewald(L)
    s = np.zeros((1, 3, L, L))
    s[0, 2] = 1.0
    E = oracle.energy(W, s, J=1.3, g=0.0, K2=0.6, K4=0.2)
    assert abs(E[0] / L ** 2 - (-2 * 1.3 - 0.6 - 0.2)) < 1e-13
    # Neel state in z: every bond antiparallel
    x = np.arange(L)
    s[0, 2] = (-1.0) ** (x[:, None] + x[None, :])
    E = oracle.energy(W, s, J=1.3, g=0.0, K2=0.6, K4=0.2)
    assert abs(E[0] / L ** 2 - (+2 * 1.3 - 0.6 - 0.2)) < 1e-13


@pytest.mark.parametrize("L", [4, 6])
def test_delta_e_is_full_energy_difference(oracle, L):
    rng = np.random.default_rng(3)
    J, g, K2, K4 = 1.0, 0.37, 0.6, -0.2
    W = oracle.build_tensor_ewald(L)
    s = rand_spins(rng, 1, L)
    h = oracle.dipole_field(W, s)
    E0 = oracle.energy(W, s, J, g, K2, K4)[0]
    for n in (0, 5, L * L - 1, L + 2):
        sp = rand_spins(rng, 1, 1)[0, :, 0, 0]
        dE = oracle.delta_e(W, s[0], h[0, :, n // L, n % L], n, sp, J, g, K2, K4)
        s2 = s.copy()
        s2[0, :, n // L, n % L] = sp
        E1 = oracle.energy(W, s2, J, g, K2, K4)[0]
        assert abs(dE - (E1 - E0)) < 2e-13 * L * L


def test_eq8_pair_identity_and_bounds(oracle):
    # PAPER.md:118-125 (eq. 8): for two sites that are not nearest neighbours,
    # H3 - H1 - H2 + H0 = g d1.W(rho_12).d2, so frozen-field dE of site 2 minus its sequential dE
    # is exactly that.  Extreme cases PAPER.md:131: D = 2 (perpendicular), D = 4 (planar).
    rng = np.random.default_rng(8)
    L, J, g, K2, K4 = 8, 1.0, 0.5, 0.3, 0.1
    W = oracle.build_tensor_ewald(L)
    s0 = rand_spins(rng, 1, L)
    n1, n2 = 0 * L + 1, 3 * L + 4
    S1, S2 = rand_spins(rng, 1, 1)[0, :, 0, 0], rand_spins(rng, 1, 1)[0, :, 0, 0]

    def with_(a, b):
        s = s0.copy()
        if a:
            s[0, :, n1 // L, n1 % L] = S1
        if b:
            s[0, :, n2 // L, n2 % L] = S2
        return s
    H = {(a, b): oracle.energy(W, with_(a, b), J, g, K2, K4)[0] for a in (0, 1) for b in (0, 1)}
    d1 = S1 - s0[0, :, n1 // L, n1 % L]
    d2 = S2 - s0[0, :, n2 // L, n2 % L]
    ry, rx = (n2 // L - n1 // L) % L, (n2 % L - n1 % L) % L
    Wm = np.array([[W[0, ry, rx], W[1, ry, rx], 0], [W[1, ry, rx], W[2, ry, rx], 0], [0, 0, W[3, ry, rx]]])
    eps = H[1, 1] - H[1, 0] - H[0, 1] + H[0, 0]
    assert abs(eps - g * d1 @ Wm @ d2) < 1e-12
    # frozen-field dE for site 2 (field of state 0) vs exact dE after site 1 flipped
    h0 = oracle.dipole_field(W, s0)
    dE_frozen = oracle.delta_e(W, s0[0], h0[0, :, n2 // L, n2 % L], n2, S2, J, g, K2, K4)
    assert abs(dE_frozen - (H[0, 1] - H[0, 0])) < 1e-12
    assert abs((H[1, 1] - H[1, 0]) - dE_frozen - eps) < 1e-12
    # bare pair bracket at separation r along x: D = |d1.d2 - 3 (d1.rhat)(d2.rhat)|
    T = lambda d1, d2: abs(d1 @ d2 - 3 * d1[0] * d2[0])
    # the paper prints D = 2 and D = 4 for these two cases; the bracket itself gives 4 and 8
    # (reading R16: the printed values carry eq. 1's factor 1/2); the 1 : 2 ratio is the pin
    D_perp = T(np.array([0, 0, 2.]), np.array([0, 0, 2.]))
    D_plan = T(np.array([2., 0, 0]), np.array([2., 0, 0]))
    assert D_perp == 4.0 and D_plan == 8.0 and D_plan / D_perp == 4.0 / 2.0


def test_halfsweep_limits(oracle):
    rng = np.random.default_rng(21)
    L, R = 6, 3
    W = oracle.build_tensor_ewald(L)
    s = rand_spins(rng, R, L)
    # T -> infinity: everything accepted; T -> 0+: accept <=> dE <= 0 (eq. 7, R14)
    s_hot = s.copy()
    out = oracle.halfsweep(W, s_hot, T=1e12, seed=1, step=0, J=1.0, g=0.1, K2=0.6, K4=0.0)
    x = np.arange(L)
    act = ((x[:, None] + x[None, :]) % 2) == 0
    assert np.all(out["accept"][:, act] == 1) and np.all(out["accept"][:, ~act] == 0)
    assert np.array_equal(s_hot[:, :, act], out["trial"][:, :, act])
    assert np.array_equal(s_hot[:, :, ~act], s[:, :, ~act])          # other colour untouched
    s_cold = s.copy()
    out = oracle.halfsweep(W, s_cold, T=1e-12, seed=1, step=1, J=1.0, g=0.1, K2=0.6, K4=0.0)
    act1 = ~act
    E_before = oracle.energy(W, s, 1.0, 0.1, 0.6, 0.0)
    for r in range(R):
        for (y, xx) in zip(*np.nonzero(act1)):
            n = y * L + xx
            h = oracle.dipole_field(W, s[r:r + 1])[0, :, y, xx]
            dE = oracle.delta_e(W, s[r], h, n, out["trial"][r, :, y, xx], 1.0, 0.1, 0.6, 0.0)
            assert bool(out["accept"][r, y, xx]) == (dE < 0)
            # margin = dE/T + ln u with the u of word 2
            _, u, _ = oracle.trial_draw(1, n, r, 1)
            assert abs(out["margin"][r, y, xx] - (dE / 1e-12 + np.log(u))) <= 1e-9 * abs(dE / 1e-12)
    assert E_before.shape == (R,)


def test_halfsweep_frozen_vs_sequential_without_dipole(oracle):
    # g = 0: active sites of one colour do not interact, so the simultaneous half-sweep is
    # exactly the sequential Metropolis sweep over those sites ("If the two
    # spins don't interact ... same statistics as the conventional sequential flipping")
    rng = np.random.default_rng(2)
    L, R = 6, 2
    W = oracle.build_tensor_ewald(L)
    s = rand_spins(rng, R, L)
    a, b = s.copy(), s.copy()
    for step in range(4):
        o1 = oracle.halfsweep(W, a, T=[0.4, 1.1], seed=7, step=step, J=1.0, g=0.0, K2=0.6, K4=0.1)
        o2 = oracle.halfsweep(W, b, T=[0.4, 1.1], seed=7, step=step, J=1.0, g=0.0, K2=0.6, K4=0.1,
                              sequential=True)
        assert np.array_equal(o1["accept"], o2["accept"])
        assert np.array_equal(a, b)
    # with dipoles the two differ by at most eq. 8 terms; decisions may differ, states stay unit
    for step in range(2):
        oracle.halfsweep(W, a, T=[0.4, 1.1], seed=7, step=step, J=1.0, g=0.3, K2=0.6, K4=0.1)
    assert np.max(np.abs((a ** 2).sum(1) - 1)) < 1e-14


def test_eq8_sequential_minus_frozen_halfsweep(oracle):
    """PAPER.md:118-125 (section 3.2, eq. 8) on the checkerboard: oracle_halfsweep_sequential differs from the
    frozen half-sweep only in that the field is recomputed from the CURRENT state.  With every move accepted
    (T huge) the margin of the k-th active site therefore exceeds the frozen one by the couplings to the
    sites updated before it (site order), term by term:
        (m_seq(k) - m_frozen(k)) T = g sum_{j<k} delta_j . W(rho_jk) . delta_k .
    Dropping the field refresh, refreshing from the wrong state or visiting in another order fails this."""
    rng = np.random.default_rng(31)
    L, J, g, K2, K4, T = 6, 1.0, 0.35, 0.4, -0.1, 1e9
    W = oracle.build_tensor_ewald(L)
    for step in (0, 1):
        s0 = rand_spins(rng, 2, L)
        a, b = s0.copy(), s0.copy()
        fa = oracle.halfsweep(W, a, T, 5, step, J, g, K2, K4)
        fb = oracle.halfsweep(W, b, T, 5, step, J, g, K2, K4, sequential=True)
        x = np.arange(L)
        act = ((x[:, None] + x[None, :]) % 2) == (step & 1)
        assert np.all(fa["accept"][:, act] == 1) and np.all(fb["accept"][:, act] == 1)
        assert np.array_equal(a, b)                                    # same trials, all accepted
        sites = [(n % L, n // L) for n in range(L * L) if act[n // L, n % L]]
        worst = 0.0
        for r in range(2):
            delta = [fa["trial"][r, :, y, xx] - s0[r, :, y, xx] for (xx, y) in sites]
            for k, (xk, yk) in enumerate(sites):
                expect = 0.0
                for j in range(k):
                    xj, yj = sites[j]
                    ry, rx = (yk - yj) % L, (xk - xj) % L
                    Wm = np.array([[W[0, ry, rx], W[1, ry, rx], 0], [W[1, ry, rx], W[2, ry, rx], 0], [0, 0, W[3, ry, rx]]])
                    expect += g * delta[j] @ Wm @ delta[k]
                got = (fb["margin"][r, yk, xk] - fa["margin"][r, yk, xk]) * T
                assert abs(got - expect) < 1e-6 * max(1.0, abs(expect)), (step, r, k, got, expect)
                worst = max(worst, abs(expect))
        assert worst > 1e-2                                            # the test is not vacuous
    # the first active site sees the state at entry in both: identical margins there
    assert fb["margin"][0, sites[0][1], sites[0][0]] == fa["margin"][0, sites[0][1], sites[0][0]]


def test_given_field_variants_equal_the_plain_calls(oracle):
    """oracle_halfsweep = "h <- O2, then oracle_halfsweep_given_field"; oracle_observables likewise.  Handing the
    plain O2 field to the given-field forms reproduces the plain calls bit for bit; a wrong field does not."""
    rng = np.random.default_rng(32)
    L, R, J, g = 6, 3, 1.0, 0.3
    K2, K4 = np.array([0.5, 0.6, 0.7]), np.array([0.1, 0.0, -0.1])
    T = np.array([0.3, 0.9, 2.0])
    W = oracle.build_tensor_ewald(L)
    s0 = rand_spins(rng, R, L)
    for step in (0, 1):
        a, b, c = s0.copy(), s0.copy(), s0.copy()
        fa = oracle.halfsweep(W, a, T, 17, step, J, g, K2, K4)
        h = oracle.dipole_field(W, s0)                                # all targets; only the active ones are read
        fb = oracle.halfsweep_given_field(W, b, h, T, 17, step, J, g, K2, K4, want=("accept", "margin", "trial"))
        assert np.array_equal(a, b)
        for k in ("accept", "margin", "trial"):
            assert np.array_equal(fa[k], fb[k]), k
        fc = oracle.halfsweep_given_field(W, c, 2.0 * h, T, 17, step, J, g, K2, K4, want=("margin",))
        assert not np.array_equal(fc["margin"], fa["margin"])
    ob = oracle.observables(W, s0, J, g, K2, K4)
    assert np.array_equal(ob, oracle.observables_given_field(s0, oracle.dipole_field(W, s0), J, g, K2, K4))


def test_detailed_balance_single_spin(oracle):
    # one spin in a fixed anisotropy field only (J = g = 0, L = 2 so the update touches isolated
    # sites): the Metropolis chain must sample exp(K2 s_z^2 / T): <s_z^2> = known 1-D integral
    from scipy.integrate import quad
    K2, T = 1.0, 0.5
    num = quad(lambda z: z * z * np.exp(K2 * z * z / T), -1, 1)[0]
    den = quad(lambda z: np.exp(K2 * z * z / T), -1, 1)[0]
    L, R = 2, 64
    W = np.zeros((4, L, L))
    s = oracle.init_spins(L, R, 0, 5)
    acc = []
    for step in range(2 * 600):
        oracle.halfsweep(W, s, T=T, seed=3, step=step, J=0.0, g=0.0, K2=K2, K4=0.0, want=())
        if step >= 200:
            acc.append((s[:, 2] ** 2).mean())
    got = np.mean(acc)
    assert abs(got - num / den) < 0.01, (got, num / den)


def test_observables_special_cases(oracle):
    L = 8
    W = oracle.build_tensor_ewald(L)
    s = np.zeros((4, 3, L, L))
    s[0, 2] = 1.0                                             # all perpendicular: eta = 1
    s[1, 0] = 1.0                                             # all in-plane: eta = 0, M_par = 1
    s[2, 2] = 1 / np.sqrt(2); s[2, 1] = 1 / np.sqrt(2)        # s_z = 1/sqrt2: eta = 1/2
    x = np.arange(L)
    s[3, 2] = (-1.0) ** (x[:, None] + x[None, :])             # +-z checkerboard: eta = 1, m_z = 0
    J, g, K2, K4 = 1.0, 0.1, 0.6, 0.1
    ob = oracle.observables(W, s, J, g, K2, K4)
    assert np.allclose(ob[:, 3], [1, 0, 0.5, 1], atol=1e-12)
    assert np.allclose(ob[:, 1], [1, 0, 1 / np.sqrt(2), 0], atol=1e-12)
    assert np.allclose(ob[:, 2], [0, 1, 1 / np.sqrt(2), 0], atol=1e-12)
    assert abs(ob[0, 0] - (-2 * J - K2 - K4 + 0.5 * g * MADELUNG)) < 1e-12
    assert abs(ob[1, 0] - (-2 * J - 0.25 * g * MADELUNG)) < 1e-12
    alt = -4.0 * (1.0 - 2.0 ** -0.5) * ZETA32 * BETA32
    assert abs(ob[3, 0] - (+2 * J - K2 - K4 + 0.5 * g * alt)) < 1e-11


def test_cone_angle_infinite_temperature(oracle):
    # eta(T -> inf) = sqrt((2/pi)^2 (pi^2 - 8)/4) = 0.43524 for spins uniform on S^2
    L = 64
    W = np.zeros((4, L, L))
    s = oracle.init_spins(L, 4, 0, 2024)
    ob = oracle.observables(W, s, 0.0, 0.0, 0.0, 0.0)
    want = np.sqrt((2 / np.pi) ** 2 * 0.25 * (np.pi ** 2 - 8))
    assert abs(want - 0.435236178254) < 1e-9
    assert np.all(np.abs(ob[:, 3] - want) < 0.01)
    assert np.all(np.abs(ob[:, 1]) < 5 * np.sqrt(1 / 3 / L ** 2))


def _stripe_ground_width(oracle, J_over_g):
    """Width h of the perpendicular stripe state (columns of alternating +-z, width h) with the lowest energy per
    spin, over every h that tiles one of the lattices L = 48 ... 80, by the oracle's energy (eq. 11, K = 0)."""
    best = {}
    for L in (48, 56, 64, 72, 80):
        W = oracle.build_tensor_ewald(L)
        widths = [h for h in range(1, L // 2 + 1) if L % (2 * h) == 0]
        s = np.zeros((len(widths), 3, L, L))
        for r, h in enumerate(widths):
            s[r, 2] = np.where((np.arange(L) // h) % 2 == 0, 1.0, -1.0)[None, :]
        E = oracle.energy(W, s, J_over_g, 1.0, 0.0, 0.0) / (L * L)
        for h, e in zip(widths, E):
            best.setdefault(h, e)
            assert abs(best[h] - e) < 1e-9          # the energy per spin of a width does not depend on the lattice
    return min(best, key=best.get)


def test_paper_stripe_widths_fix_the_unit_of_C_D(oracle):
    """The paper prints two ground-state stripe widths: w = 8 at script-J = J / C_D = 8.9 and the
    thinnest width h = 1 at J / C_D = 1.7.  With eq. 11 / eq. 19 read as every bond and every pair
    once (R7, R8, R22) both hold iff the paper's C_D is g / 2, i.e. J / g = 4.45 and 0.85; taking
    J / g = 8.9 and 1.7 literally gives widths >= 40 and 2 instead.  This pins the map from the paper's
    dimensionless script-J, script-K, script-T to the build's (J, g, K2, K4, T) and, through the stripe energies, the
    sign and size of W^zz against the exchange term."""
    assert _stripe_ground_width(oracle, 8.9 / 2) == 8
    assert _stripe_ground_width(oracle, 1.7 / 2) == 1
    assert _stripe_ground_width(oracle, 8.9) >= 40
    assert _stripe_ground_width(oracle, 1.7) == 2
