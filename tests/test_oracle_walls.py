"""Pins of the oracle's domain-wall observables (eq. 14-15) against what the paper
and the definitions fix: perfect stripes, the uniform and checkerboard states, the T -> infinity
wall density 1/2 the paper quotes, the lattice symmetries."""
import numpy as np


def _state(L, fz, fx=None, fy=None):
    s = np.zeros((1, 3, L, L))
    s[0, 2] = fz
    s[0, 0] = fz if fx is None else fx
    s[0, 1] = fz if fy is None else fy
    return s


def test_vertical_stripes_of_width_w(oracle):
    """Columns of width w alternating in sign: each row crosses L/w walls, no vertical bond does.
    n_h = 2 L (L/w), n_v = 0, wall density 1/(2w), O = 1 (perfect orientational order)."""
    L = 16
    x = np.arange(L)
    for w in (1, 2, 4, 8):
        f = np.where((x // w) % 2 == 0, 1.0, -1.0)[None, :] * np.ones((L, 1))
        c = oracle.wall_counts(_state(L, f))
        assert c[0].tolist() == [2 * L * (L // w), 0] * 3
        d = oracle.wall_order(L, c)
        assert d[0, 0] == 1.0 / (2 * w) and np.all(d[0, 1:] == 1.0)
        # rotate by 90 degrees: horizontal stripes swap the roles of n_h and n_v
        c2 = oracle.wall_counts(_state(L, f.T.copy()))
        assert c2[0].tolist() == [0, 2 * L * (L // w)] * 3
        assert np.array_equal(oracle.wall_order(L, c2), d)


def test_uniform_and_checkerboard(oracle):
    L = 8
    c = oracle.wall_counts(_state(L, np.ones((L, L))))
    assert np.all(c == 0)
    assert np.all(oracle.wall_order(L, c) == 0.0)               # no walls: O defined as 0
    x = np.arange(L)
    cb = np.where((x[:, None] + x[None, :]) % 2 == 0, 1.0, -1.0)
    c = oracle.wall_counts(_state(L, cb))
    assert np.all(c == 2 * L * L)                                # every bond is a wall
    d = oracle.wall_order(L, c)
    assert d[0, 0] == 1.0 and np.all(d[0, 1:] == 0.0)


def test_components_are_independent(oracle):
    """Each component has its own counts (robust against canting): z striped, x
    uniform, y checkerboard."""
    L = 8
    x = np.arange(L)
    fz = np.where((x // 2) % 2 == 0, 0.3, -0.9)[None, :] * np.ones((L, 1))   # magnitudes do not matter
    fy = np.where((x[:, None] + x[None, :]) % 2 == 0, 1e-30, -1e-30)          # nor does a tiny product
    c = oracle.wall_counts(_state(L, fz, fx=np.full((L, L), 0.1), fy=fy))
    assert c[0].tolist() == [0, 0, 2 * L * L, 2 * L * L, 2 * L * (L // 2), 0]


def test_zero_component_counts_one(oracle):
    """sgn(0) = 0: a bond touching an exactly-zero component contributes 1."""
    L = 4
    f = np.ones((L, L))
    f[1, 2] = 0.0
    c = oracle.wall_counts(_state(L, f))
    assert c[0, 4] == 2 and c[0, 5] == 2                       # two horizontal and two vertical bonds


def test_random_state_wall_density_one_half(oracle):
    """the wall density tends to 1/2 as T -> infinity (independent signs: a bond is a
    wall with probability 1/2, counted 2, over 2N bonds, divided by 4N)."""
    rng = np.random.default_rng(3)
    L, R = 64, 4
    s = rng.standard_normal((R, 3, L, L))
    d = oracle.wall_order(L, oracle.wall_counts(s))
    assert np.all(np.abs(d[:, 0] - 0.5) < 4 * 0.5 / np.sqrt(2 * L * L))
    assert np.all(d[:, 1:] < 0.05)                             # no orientational order


def test_counts_against_numpy_rolls(oracle):
    rng = np.random.default_rng(4)
    L, R = 12, 3
    s = rng.standard_normal((R, 3, L, L))
    c = oracle.wall_counts(s)
    sg = np.sign(s)
    nh = (1 - sg * np.roll(sg, -1, axis=3)).sum(axis=(2, 3))
    nv = (1 - sg * np.roll(sg, -1, axis=2)).sum(axis=(2, 3))
    ref = np.stack([nh[:, 0], nv[:, 0], nh[:, 1], nv[:, 1], nh[:, 2], nv[:, 2]], axis=1)
    assert np.array_equal(c, ref.astype(np.int64))


def test_staggered_magnetisation_of_stripe_states(oracle):
    """App. B: width-1 horizontal stripes give |m_h| = 1, m_v = 0; vertical ones the
    reverse; uniform, checkerboard and width-2 stripe states give m_st = 0; random Ising spins ~ N^-1/2."""
    L = 8
    x = np.arange(L)
    rows = np.where(x % 2 == 0, 1.0, -1.0)[:, None] * np.ones((1, L))        # alternates along y
    cols = rows.T.copy()
    for f, expect in ((rows, (1.0, 0.0, 1.0)), (-rows, (-1.0, 0.0, 1.0)), (cols, (0.0, 1.0, 1.0)),
                      (np.ones((L, L)), (0.0, 0.0, 0.0)),
                      (np.where((x[:, None] + x[None, :]) % 2 == 0, 1.0, -1.0), (0.0, 0.0, 0.0)),
                      (np.where((x // 2) % 2 == 0, 1.0, -1.0)[:, None] * np.ones((1, L)), (0.0, 0.0, 0.0))):
        s = np.zeros((1, 3, L, L))
        s[0, 2] = f
        s[0, 0] = 0.5                                                          # in-plane components do not enter
        assert np.allclose(oracle.staggered(s)[0], expect, atol=1e-15)
    rng = np.random.default_rng(1)
    s = np.zeros((4, 3, 64, 64))
    s[:, 2] = rng.choice([-1.0, 1.0], size=(4, 64, 64))
    m = oracle.staggered(s)
    assert np.all(m[:, 2] < 5.0 / 64) and np.allclose(m[:, 2], np.hypot(m[:, 0], m[:, 1]))
    # one defect in a perfect state lowers m_h by 2/N
    s1 = np.zeros((1, 3, L, L))
    s1[0, 2] = rows
    s1[0, 2, 3, 5] *= -1
    assert abs(oracle.staggered(s1)[0, 0] - (1.0 - 2.0 / (L * L))) < 1e-15


def test_ensemble_statistics(oracle):
    """eq. 13 / eq. 18: closed forms and the library routine."""
    m, v, se = oracle.ensemble(np.full((7, 3), 2.5))
    assert np.all(m == 2.5) and np.all(v == 0.0) and np.all(se == 0.0)
    x = np.array([[1.0], [3.0]] * 50)                              # +-1 around 2: variance 1, SE = 1/sqrt(n)
    m, v, se = oracle.ensemble(x)
    assert m[0] == 2.0 and v[0] == 1.0 and abs(se[0] - 0.1) < 1e-16
    t = np.arange(1, 11, dtype=np.float64)[:, None]                # 1..10: mean 5.5, variance (n^2-1)/12
    m, v, se = oracle.ensemble(t)
    assert m[0] == 5.5 and abs(v[0] - 99.0 / 12.0) < 1e-14 and abs(se[0] - np.sqrt(99.0 / 120.0)) < 1e-15
    rng = np.random.default_rng(0)
    y = rng.standard_normal((1000, 4, 2))
    m, v, se = oracle.ensemble(y)
    assert np.allclose(m, y.mean(0), atol=1e-15) and np.allclose(v, y.var(0), atol=1e-14)
    assert np.allclose(se, y.std(0) / np.sqrt(1000), atol=1e-15)
