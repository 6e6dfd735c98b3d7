"""Pins for the oracle's interaction table W (eq. 1-5).

Nothing here retypes the oracle's formulas: the checks are the Laplace invariant,
the lattice symmetries, closed-form lattice sums (Hurwitz-zeta evaluations from
scipy), agreement of two independent summation routes, and an independent
numpy brute force.
"""
import numpy as np
import pytest
from scipy.special import zeta

ZETA32 = zeta(1.5, 1.0)
BETA32 = (zeta(1.5, 0.25) - zeta(1.5, 0.75)) / 8.0        # Dirichlet beta(3/2)
MADELUNG = 4.0 * ZETA32 * BETA32                           # sum' (m^2+n^2)^-3/2


def test_closed_form_constant():
    # sum'_{(m,n) in Z^2} (m^2+n^2)^(-3/2) = 4 zeta(3/2) beta(3/2) = 9.0336...
    # (BASELINE.json: "lattice sum  sum 1/r^3 = 9.0336...")
    assert abs(MADELUNG - 9.0336216831) < 1e-9


@pytest.fixture(scope="module", params=[4, 8, 16])
def tables(request, oracle):
    L = request.param
    return L, oracle.build_tensor_ewald(L), oracle.build_tensor_image(L, 64, 1)


def test_laplace_invariant(tables):
    # each image term of eq. 1 is traceless, so W^xx + W^yy + W^zz = 0 for every rho
    L, We, Wi = tables
    for W, tol in ((We, 2e-13), (Wi, 2e-13)):
        tr = W[0] + W[2] + W[3]
        assert np.max(np.abs(tr)) < tol * max(1.0, np.max(np.abs(W)))


def test_laplace_invariant_no_tail(oracle):
    W = oracle.build_tensor_image(8, 16, 0)
    assert np.max(np.abs(W[0] + W[2] + W[3])) < 1e-13


def test_signs(tables):
    # eq. 1: side-by-side perpendicular spins repel (W^zz > 0), head-to-tail in-plane
    # spins attract (W^xx(1,0) < 0), side-by-side in-plane repel (W^yy(1,0) > 0).  (R1)
    L, We, _ = tables
    assert We[3, 0, 1] > 0 and We[0, 0, 1] < 0 < We[2, 0, 1]
    if L >= 8:
        assert abs(We[3, 0, 1] - 1.0) < 0.05 and abs(We[0, 0, 1] + 2.0) < 0.05


def test_symmetries(tables):
    L, We, Wi = tables
    # exact for the Ewald route; a square image cutoff is centred on the reduced rho, so on the
    # cell edge rho = L/2 the truncated sum is lopsided by about tail/A (reading R6)
    for W, tol in ((We, 1e-12), (Wi, 2e-7)):
        neg = lambda A: np.roll(np.roll(A[::-1, ::-1], 1, axis=0), 1, axis=1)   # rho -> -rho mod L
        for c in range(4):
            assert np.max(np.abs(W[c] - neg(W[c]))) < tol          # W(rho) = W(-rho)
        assert np.max(np.abs(W[0] - W[2].T)) < tol                 # xx(rx,ry) = yy(ry,rx)
        assert np.max(np.abs(W[3] - W[3].T)) < tol                 # zz symmetric under x<->y
        assert np.max(np.abs(W[1] - W[1].T)) < tol                 # xy symmetric under x<->y
        flipx = lambda A: np.roll(A[:, ::-1], 1, axis=1)           # rho_x -> -rho_x mod L
        assert np.max(np.abs(W[1] + flipx(W[1]))) < tol            # xy odd in rho_x
        assert np.max(np.abs(W[1][:, 0])) < tol and np.max(np.abs(W[1][0, :])) < tol
        assert np.max(np.abs(W[1][:, L // 2])) < tol and np.max(np.abs(W[1][L // 2, :])) < tol


def test_lattice_sum_closed_form(tables):
    # sum over the cell of W^zz = sum' over Z^2 of r^-3, independent of L (every site of the
    # infinite lattice is counted exactly once: reading R3); xx, yy get -1/2 each; xy 0.
    L, We, Wi = tables
    for W, tol in ((We, 1e-11), (Wi, 5e-7)):
        assert abs(W[3].sum() - MADELUNG) < tol
        assert abs(W[0].sum() + 0.5 * MADELUNG) < tol
        assert abs(W[2].sum() + 0.5 * MADELUNG) < tol
        assert abs(W[1].sum()) < tol


def test_self_term(tables):
    # W(0) = sum over G != 0 of T(G) = L^-3 sum' (a^2+b^2)^-3/2   (eq. 2 self-image term, R2)
    L, We, Wi = tables
    for W, tol in ((We, 1e-13), (Wi, 1e-7)):
        assert abs(W[3, 0, 0] - MADELUNG / L ** 3) < tol
        assert abs(W[0, 0, 0] + 0.5 * W[3, 0, 0]) < tol
        assert abs(W[2, 0, 0] + 0.5 * W[3, 0, 0]) < tol
        assert abs(W[1, 0, 0]) < tol


def test_two_routes_agree(tables):
    L, We, Wi = tables
    assert np.max(np.abs(We - Wi)) < 1e-7                       # image A=64 + tail vs Ewald


def test_two_routes_agree_small_cutoff(oracle):
    We = oracle.build_tensor_ewald(8)
    assert np.max(np.abs(We - oracle.build_tensor_image(8, 16, 1))) < 1e-6
    # without the tail the square cutoff is visibly short (reading R6): zz low by ~ 4 sqrt2/(A+.5)L^3
    Wn = oracle.build_tensor_image(8, 64, 0)
    d = (We - Wn)[3]
    t = 4 * np.sqrt(2) / (64.5 * 8 ** 3)
    assert np.all(np.abs(d - t) < 0.02 * t)


def test_ewald_independent_of_splitting(oracle):
    for L in (4, 8):
        ref = oracle.build_tensor_ewald(L, 2.5, 6, 12)
        for aL in (2.0, 3.0, 3.5):
            W = oracle.build_tensor_ewald(L, aL, 8, 16)
            assert np.max(np.abs(W - ref)) < 1e-13


def test_alternating_states_closed_form(oracle):
    # checkerboard +-z: sum_rho (-1)^(rx+ry) W^zz = sum' (-1)^(m+n) r^-3
    #   = -4 (1 - 2^(-1/2)) zeta(3/2) beta(3/2)   (Glasser-Zucker lattice sum)
    want = -4.0 * (1.0 - 2.0 ** -0.5) * ZETA32 * BETA32
    for L in (4, 8, 16):
        W = oracle.build_tensor_ewald(L)
        x = np.arange(L)
        sign = (-1.0) ** (x[None, :] + x[:, None])
        assert abs((sign * W[3]).sum() - want) < 1e-11
        Wi = oracle.build_tensor_image(L, 32, 0)              # tail-independent: net moment 0
        assert abs((sign * Wi[3]).sum() - want) < 1e-5


def _brute_W(L, rx, ry, A):
    a = np.arange(-A, A + 1)
    X = rx + a[None, :] * L
    Y = ry + a[:, None] * L
    r2 = (X * X + Y * Y).astype(np.float64)
    keep = r2 > 0                                            # the G = 0 term is absent at rho = 0
    r2 = np.where(keep, r2, 1.0)
    r5 = r2 ** 2.5
    return np.array([(keep * (r2 - 3 * X * X) / r5).sum(), (keep * -3 * X * Y / r5).sum(),
                     (keep * (r2 - 3 * Y * Y) / r5).sum(), (keep * r2 ** -1.5).sum()])


def test_against_numpy_brute_force_extrapolated():
    # independent numpy sum of eq. 1's bracket over images, Richardson-extrapolated in 1/(A+1/2)
    from oracle import oracle as o
    L = 4
    W = o.build_tensor_ewald(L)
    for (rx, ry) in ((0, 0), (1, 0), (1, 1), (2, 1), (2, 2), (3, 1)):
        dx = rx if rx <= L // 2 else rx - L
        dy = ry if ry <= L // 2 else ry - L
        A1, A2 = 200, 400
        w1, w2 = _brute_W(L, dx, dy, A1), _brute_W(L, dx, dy, A2)
        x1, x2 = 1 / (A1 + .5), 1 / (A2 + .5)
        wx = (w2 * x1 - w1 * x2) / (x1 - x2)
        assert np.max(np.abs(wx - W[:, ry, rx])) < 2e-8, (rx, ry, wx, W[:, ry, rx])


def test_survey_worked_entries(oracle):
    # tests/golden/w_L8_survey.txt: entries computed for SURVEY.md section 8(c) with independent
    # mpmath scripts (not by this oracle); cited there as a cross-check.
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "w_L8_survey.txt")
    W = oracle.build_tensor_ewald(8)
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        rx, ry, xx, xy, yy, zz = line.split()
        got = W[:, int(ry), int(rx)]
        want = np.array([float(xx), float(xy), float(yy), float(zz)])
        assert np.max(np.abs(got - want)) < 2e-10 * max(1, np.max(np.abs(want))) + 6e-11, (rx, ry, got, want)
        n += 1
    assert n == 7


def test_golden_table_regenerates(oracle):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "w_L8_oracle.txt")
    want = np.loadtxt(path).reshape(4, 8, 8)
    assert np.max(np.abs(oracle.build_tensor_ewald(8) - want)) < 1e-14
