"""GPU parity of the paper's own update schedule (dsmc_sublattice_pass; section 3.1,
App. A) against the oracle, pass by pass in lock-step with resync (SURVEY.md 8c parity protocol)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

BAND = 1e-4
BAND_FRACTION = 1e-4


@pytest.fixture(scope="module")
def dsmc_mod():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1211_6234_b200 as m
    from paper_1211_6234_b200 import build
    build.build()
    return m


def lockstep_passes(m, oracle, ctx, W, T, J, g, K2, K4, seed, l, n_passes, flip=False, resident=True):
    L, R = ctx.L, ctx.R
    acc_d = torch.zeros((R, L, L), dtype=torch.uint8, device="cuda")
    mar_d = torch.zeros((R, L, L), dtype=torch.float32, device="cuda")
    flags = (m.DSMC_TRIAL_FLIP if flip else 0) | (0 if resident else m.DSMC_NO_RESIDENT)
    ambiguous = trials = accepted = 0
    for p in range(n_passes):
        s_before = ctx.get_spins()
        s_or = s_before.astype(np.float64)
        out = oracle.sublattice_pass(W, s_or, T, seed, p, l, J, g, K2, K4, flip=flip)
        off = ctx.sublattice_pass(T, seed, p, l, flags=flags, accept_out=acc_d, margin_out=mar_d)
        assert off == out["offset"]                                    # integer work: bit-exact
        s_after = ctx.get_spins()
        ox, oy = off
        site = np.zeros((L, L), dtype=bool)
        site[oy::l, ox::l] = True
        assert site.sum() == (L // l) ** 2
        acc = acc_d.cpu().numpy()[:, site].astype(bool)
        mar = mar_d.cpu().numpy()[:, site]
        m_or = out["margin"][:, site]
        a_or = out["accept"][:, site].astype(bool)
        amb = np.abs(m_or) < BAND
        assert np.array_equal(acc[~amb], a_or[~amb]), (p, int(np.sum(acc[~amb] != a_or[~amb])))
        # the margin is dE / T: an fp32 dE good to ~2e-5 (field tolerance 1e-4 in h, times g |delta|) gives
        # a margin good to 2e-5 / T below T = 1
        tol = 2e-5 / np.minimum(np.asarray(T, dtype=np.float64), 1.0)[:, None] + 3e-6 * np.abs(m_or)
        assert np.all(np.abs(mar - m_or) <= tol), (p, np.abs(mar - m_or).max())
        ambiguous += int(amb.sum())
        trials += amb.size
        accepted += int(acc.sum())
        full = np.zeros((R, L, L), dtype=bool)
        full[:, site] = acc
        chg = np.broadcast_to(full[:, None], s_after.shape)
        assert np.array_equal(s_after[~chg], s_before[~chg])           # rejected and all other sites: bit-unchanged
        assert np.max(np.abs(s_after[chg].astype(np.float64) - out["trial"][chg]), initial=0.0) <= 1e-6
    assert ambiguous <= max(1, BAND_FRACTION * trials), (ambiguous, trials)
    return accepted, trials


@pytest.mark.parametrize("L,R,l,passes,fft,resident", [
    (8, 1, 4, 40, False, True), (12, 5, 3, 24, False, True), (32, 8, 8, 24, False, True), (64, 16, 32, 48, False, True),
    (64, 40, 2, 6, False, True), (16, 3, 16, 12, False, True), (64, 16, 32, 48, True, True), (32, 8, 8, 24, True, True),
    (32, 6, 2, 8, True, True), (8, 1, 4, 40, False, False), (64, 16, 32, 24, False, False), (16, 3, 16, 12, False, False),
    (12, 5, 6, 24, False, True), (74, 2, 37, 12, False, True), (64, 3, 64, 12, False, True),
    (64, 296, 32, 6, False, True), (64, 16, 16, 24, False, True), (64, 16, 16, 8, False, False), (4, 2, 2, 16, False, True), (6, 1, 3, 16, False, True), (6, 2, 6, 16, False, True)])
def test_sublattice_lockstep(dsmc_mod, oracle, L, R, l, passes, fft, resident):
    """(64, 16, 32) is the paper's own choice L = 64, l = 32; l = 2 is the densest
    schedule (n = N/4), l = L the conventional single-spin limit; R = 40 spans two replica chunks.
    With L/l in {1, 2, 4} and L <= 74 (and no FFT field) the pass runs in the shared-memory-resident kernel
    unless resident = False asks for the two-launch path: both are held to the same oracle.  (64, 296, 32) is the
    second launch configuration bench.py times (148 CTAs, one per SM); L = 4 and 6 are the smallest lattices."""
    from paper_1211_6234_b200 import inputs
    J, g, K2, K4 = 1.0, 0.25, 0.6, 0.1
    ctx = dsmc_mod.Dsmc(L, R, J=J, g=g, K2=K2, K4=K4)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    if fft:                                                     # the field of the pass through the FFT route
        ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    W = oracle.build_tensor_ewald(L)
    ctx.set_spins(inputs.random_spins(L, R, 31))
    T = np.linspace(0.2, 1.6, R).astype(np.float32)
    acc, tr = lockstep_passes(dsmc_mod, oracle, ctx, W, T, J, g, K2, K4, 0x5EED, l, passes, resident=resident)
    assert 0 < acc < tr
    ctx.close()


def test_sublattice_ising_flip(dsmc_mod, oracle):
    """App. B: L = 64, l = 32, Ising spins, J / C_D = 1.7 in eq. 19's convention (0.85 per bond in ours,
    DESIGN.md R22), T around the paper's T_c = 0.85 C_D (Table 1), starting from the
    h = 1 stripe ground state with a few defects."""
    L, R, l = 64, 8, 32
    J, g = 0.85, 1.0
    ctx = dsmc_mod.Dsmc(L, R, J=J, g=g, K2=0.0, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    W = oracle.build_tensor_ewald(L)
    rng = np.random.default_rng(6)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, None, :]
    s[:, 2] *= np.where(rng.random((R, L, L)) < 0.2, -1.0, 1.0)
    ctx.set_spins(s)
    T = (np.linspace(0.5, 1.2, R) * g).astype(np.float32)
    acc, tr = lockstep_passes(dsmc_mod, oracle, ctx, W, T, J, g, 0.0, 0.0, 99, l, 64, flip=True)
    out = ctx.get_spins()
    assert np.all(np.abs(out[:, 2]) == 1.0) and np.all(out[:, :2] == 0.0)
    assert acc > 0
    ctx.close()


def test_checkerboard_flip_flag(dsmc_mod, oracle):
    """DSMC_TRIAL_FLIP on the checkerboard half-sweep: an Ising state stays one, energy changes agree
    with the oracle's energy of the resulting state (margins are checked through the sub-lattice path)."""
    L, R = 32, 8
    J, g = 1.0, 0.5
    ctx = dsmc_mod.Dsmc(L, R, J=J, g=g, K2=0.0, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    rng = np.random.default_rng(8)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = rng.choice([-1.0, 1.0], size=(R, L, L))
    ctx.set_spins(s)
    T = np.full(R, 0.8, dtype=np.float32)
    mar_d = torch.zeros((R, L, L), dtype=torch.float32, device="cuda")
    acc_d = torch.zeros((R, L, L), dtype=torch.uint8, device="cuda")
    ctx.halfsweep(T, 4, 0, flags=dsmc_mod.DSMC_TRIAL_FLIP, accept_out=acc_d, margin_out=mar_d)
    out = ctx.get_spins()
    assert np.all(np.abs(out[:, 2]) == 1.0) and np.all(out[:, :2] == 0.0)
    x = np.arange(L)
    par = (x[:, None] + x[None, :]) % 2
    flipped = out[:, 2] != s[:, 2]
    assert np.array_equal(flipped[:, par == 0], acc_d.cpu().numpy()[:, par == 0].astype(bool))
    assert not flipped[:, par == 1].any() and flipped.any()
    # a flipped site's margin is dE/T + ln u with dE the frozen-field energy change: check one site per replica
    W = oracle.build_tensor_ewald(L)
    h = oracle.dipole_field(W, s.astype(np.float64), colour=0)
    mar = mar_d.cpu().numpy()
    for r in range(R):
        n = 2 * r * L + 2 * r                                       # (x, y) = (2r, 2r): colour 0
        sp = -s[r, :, 2 * r, 2 * r].astype(np.float64)
        dE = oracle.delta_e(W, s[r].astype(np.float64), h[r, :, 2 * r, 2 * r], n, sp, J, g, 0.0, 0.0)
        _, u, _ = oracle.trial_draw(4, n, r, 0)
        m_or = dE / 0.8 + np.log(u)
        assert abs(mar[r, 2 * r, 2 * r] - m_or) <= 2e-5 + 3e-6 * abs(m_or)
    ctx.close()


def test_sublattice_argument_errors(dsmc_mod):
    ctx = dsmc_mod.Dsmc(12, 2)
    ctx.build_tensor()
    ctx.init_spins(dsmc_mod.DSMC_INIT_RANDOM, seed=1)
    T = np.ones(2, dtype=np.float32)
    for bad_l in (1, 5, 24, 0):
        with pytest.raises(dsmc_mod.DsmcError):
            ctx.sublattice_pass(T, 1, 0, bad_l)
    ctx.sublattice_run(T, 1, 0, 9, 3)                               # 9 = l*l passes = one MC step
    ctx.close()


@pytest.mark.parametrize("L,R", [(8, 1), (12, 5), (64, 16), (256, 64)])
def test_staggered_magnetisation_parity(dsmc_mod, oracle, L, R):
    """App. B's order parameter: Ising states (exact sums) and Heisenberg states (fp64 sums of fp32 values)."""
    from paper_1211_6234_b200 import inputs
    ctx = dsmc_mod.Dsmc(L, R)
    rng = np.random.default_rng(12)
    ising = np.zeros((R, 3, L, L), dtype=np.float32)
    ising[:, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, :, None]
    ising[:, 2] *= np.where(rng.random((R, L, L)) < 0.1, -1.0, 1.0)
    ctx.set_spins(ising)
    got, ref = ctx.staggered_magnetisation(), oracle.staggered(ising.astype(np.float64))
    N = L * L                                                    # the sub-lattice sums are integers: exact
    assert np.array_equal(np.rint(got[:, :2] * N), np.rint(ref[:, :2] * N)) and np.max(np.abs(got - ref)) <= 1e-15
    assert np.all(np.abs(got[:, 0]) > 0.7)
    s = inputs.random_spins(L, R, 4)
    ctx.set_spins(s)
    assert np.max(np.abs(ctx.staggered_magnetisation() - oracle.staggered(s.astype(np.float64)))) <= 1e-13
    ctx.close()


def test_simultaneous_flipping_error_is_small(dsmc_mod, oracle):
    """App. B's question: do the errors of simultaneous flipping compound over many
    passes?  Dipolar Ising model, J / C_D = 1.7 in eq. 19's convention = 0.85 per bond in ours (DESIGN.md
    R22: inside the width-1 stripe window 0.43 < J/g < 1.26), L = 16 with l = 8 (four simultaneous
    flips per pass, a stronger approximation than the paper's l = 32), staggered magnetisation against
    T / C_D: the GPU's frozen-field schedule versus conventional sequential Metropolis in the oracle
    (independent seeds).  The paper reports shifts below 8 % in the critical values (Table 1)."""
    L, l, R = 16, 8, 8
    J, g = 0.85, 1.0
    Tn = np.linspace(0.4, 1.4, R)                                   # T / C_D: T_c ~ 0.82-0.85 (Table 1)
    T = (Tn * g).astype(np.float32)
    W = oracle.build_tensor_ewald(L)
    s0 = np.zeros((R, 3, L, L), dtype=np.float32)
    s0[:, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, :, None]
    n_steps, burn, every = 600, 200, 5
    ctx = dsmc_mod.Dsmc(L, R, J=J, g=g, K2=0.0, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    ctx.set_spins(s0)
    gpu = []
    for step in range(n_steps):
        ctx.sublattice_run(T, 4242, step * l * l, l * l, l, flags=dsmc_mod.DSMC_TRIAL_FLIP)
        if step >= burn and step % every == 0:
            gpu.append(ctx.staggered_magnetisation()[:, 2])
    ctx.close()
    s = s0.astype(np.float64)
    seq = []
    for step in range(n_steps):
        for p in range(step * l * l, (step + 1) * l * l):
            oracle.sublattice_pass(W, s, T, 1717, p, l, J, g, 0.0, 0.0, flip=True, sequential=True)
        if step >= burn and step % every == 0:
            seq.append(oracle.staggered(s)[:, 2])
    gpu, seq = np.mean(gpu, axis=0), np.mean(seq, axis=0)
    print("T/C_D      ", np.round(Tn, 2))
    print("m_st GPU   ", np.round(gpu, 3))
    print("m_st seq.  ", np.round(seq, 3))
    assert gpu[0] > 0.75 and seq[0] > 0.75 and gpu[-1] < 0.3 and seq[-1] < 0.3      # ordered -> disordered
    assert np.max(np.abs(gpu - seq)) < 0.1, np.abs(gpu - seq)                       # measured: 0.03


@pytest.mark.parametrize("L,R,l,fft,flip,resident", [
    (64, 16, 32, False, False, True), (64, 16, 32, True, True, True), (12, 5, 3, False, True, True),
    (32, 8, 2, True, False, True), (64, 16, 32, False, False, False), (64, 5, 32, False, True, True),
    (16, 4, 16, False, False, True), (12, 5, 6, False, False, True), (64, 6, 16, False, False, True)])
def test_sublattice_run_graph_replay_is_bit_identical(dsmc_mod, L, R, l, fft, flip, resident):
    """dsmc_sublattice_run either keeps the lattice in shared memory for the whole run (one kernel; L/l in
    {1, 2, 4}, L <= 74, no FFT field, resident = True) or replays a captured graph of passes whose kernels
    recompute the offset from a pass counter on the device: same trajectory, bit for bit, as pass-by-pass
    calls with the same flags."""
    from paper_1211_6234_b200 import inputs
    T = np.linspace(0.3, 1.5, R).astype(np.float32)
    flags = (dsmc_mod.DSMC_TRIAL_FLIP if flip else 0) | (0 if resident else dsmc_mod.DSMC_NO_RESIDENT)
    a = dsmc_mod.Dsmc(L, R, J=1.0, g=0.3, K2=0.5, K4=0.1)
    b = dsmc_mod.Dsmc(L, R, J=1.0, g=0.3, K2=0.5, K4=0.1)
    a.build_tensor(dsmc_mod.DSMC_W_EWALD)
    b.set_tensor(a.get_tensor())
    for ctx in (a, b):
        if fft:
            ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
        ctx.set_spins(inputs.random_spins(L, R, 3))
    for (seed, first, n) in ((5, 0, 40), (5, 40, 9), (6, 1000, 17)):
        a.sublattice_run(T, seed, first, n, l, flags=flags)
        for k in range(n):
            b.sublattice_pass(T, seed, first + k, l, flags=flags)
        assert np.array_equal(a.get_spins(), b.get_spins()), (seed, first, n)
    a.close()
    b.close()


@pytest.mark.skipif(not __import__("os").environ.get("DSMC_PAPER"),
                    reason="opt-in (DSMC_PAPER=1): compares the GPU with sentences of the paper, not with the oracle; "
                           "out of SURVEY.md section 8's scope, kept as an example run")
def test_appendix_b_critical_temperature_matches_table1(dsmc_mod):
    """The paper's own validation number: App. B puts the order-disorder transition of the dipolar Ising model
    (L = 64, l = 32, J / C_D = 1.7) at script-T_c = .85 with its algorithm and .82 by conventional Monte Carlo
    (Table 1; tests/golden/paper_table1.txt).  In the build's units script-T = 2 T / g
    (R22).  The peak of the staggered susceptibility chi_st = (L^2 / T)(<m_st^2> - <m_st>^2) over a
    temperature scan on the GPU (the paper's schedule, resident kernel) must fall between the two printed values
    give or take the scan's resolution, ordered below it and disordered above it."""
    import os
    from paper_1211_6234_b200 import appendix_b
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_table1.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                k, a, b = line.split()
                rows[k] = (float(a), float(b))
    temps = np.linspace(0.37, 0.48, 12)
    r = appendix_b.scan(32, temps, chains=16, equilibrate=1500, steps=4000, seed=7)
    tc = 2.0 * appendix_b.peak_temperature(r["T"], r["chi_st"])          # script-T_c
    print("script-T     ", np.round(2 * temps, 3))
    print("m_st         ", np.round(r["m_st"], 3))
    print("chi_st       ", np.round(r["chi_st"], 1))
    print("script-T_c   ", round(tc, 3), "paper:", rows["T_c"])
    lo, hi = min(rows["T_c"]), max(rows["T_c"])
    assert lo - 0.03 <= tc <= hi + 0.03, tc                                 # measured: 0.846
    assert r["m_st"][0] > 0.85 and r["m_st"][-1] < 0.25                     # ordered -> disordered across the peak


@pytest.mark.skipif(not __import__("os").environ.get("DSMC_PAPER"),
                    reason="opt-in (DSMC_PAPER=1): compares the GPU with sentences of the paper, not with the oracle; "
                           "out of SURVEY.md section 8's scope, kept as an example run")
def test_section4_production_run_matches_the_papers_statements(dsmc_mod):
    """The paper's production run (L = 64, l = 32, script-J = 8.9, script-K = 15, striped start) in
    a shortened protocol, against the numbers its text prints (tests/golden/paper_section4.txt): for a = 0 the
    in-plane magnetisation peaks at M_par ~ .46 near script-T = 4.5 after the orientational order is lost over
    1 < script-T < 3 and is gone by script-T = 8; for a = 2 the stripes hold up to script-T = 4 and the system then
    jumps to an in-plane ferromagnet; for a = -1 the orientational order goes over 1 < script-T < 2.5.  These are
    the only quantitative statements about Figs. 10-13; they also check the unit map script-T = 2 T / g (R7)."""
    import os
    from paper_1211_6234_b200 import section4
    g = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_section4.txt")) as f:
        for line in f:
            if not line.startswith("#"):
                k, v = line.split()[:2]
                g[k] = float(v)
    temps = np.array([1.0, 2.5, 3.0, 3.5, 4.0, 4.5, 5.0, 8.0])
    r = section4.run(temps, chains=2, equilibrate=10000, steps=4000, every=50, seed=11)
    mean = r["mean"]                                            # [a][T][quantity]
    Oz, Mpar, eta = mean[:, :, 7], mean[:, :, 2], mean[:, :, 3]
    print("script-T   ", temps)
    for ia, a in enumerate(section4.A_VALUES):
        print(f"a = {a:+.0f}: O_z  ", np.round(Oz[ia], 3))
        print(f"        M_par", np.round(Mpar[ia], 3))
        print(f"        eta  ", np.round(eta[ia], 3))
    iT = {t: i for i, t in enumerate(temps)}
    # a = 0 (index 1): ordered at the lower end of the printed window, disordered above it, peak of M_par
    assert Oz[1, iT[g["a0_Oz_loss_T_lo"]]] > 0.95 and Oz[1, iT[3.5]] < 0.1
    ipk = int(np.argmax(Mpar[1]))
    assert abs(temps[ipk] - g["a0_Mpar_peak_T"]) <= 0.5, temps[ipk]
    assert abs(Mpar[1, ipk] - g["a0_Mpar_peak_value"]) < 0.05, Mpar[1, ipk]           # measured: 0.47
    assert Mpar[1, iT[g["a0_Mpar_zero_T"]]] < 0.1
    # a = 2 (index 2): stripes up to script-T = 4, in-plane ferromagnet right above
    assert Oz[2, iT[3.5]] > 0.4 and Mpar[2, iT[3.5]] < 0.05 and eta[2, iT[3.5]] > 0.75
    assert Oz[2, iT[4.5]] < 0.05 and Mpar[2, iT[4.5]] > 0.65 and eta[2, iT[4.5]] < 0.4
    # a = -1 (index 0): canted at every temperature (eta far from 1), order lost across 1 ... 2.5
    assert Oz[0, iT[g["am1_Oz_loss_T_lo"]]] > 0.9 and Oz[0, iT[3.0]] < 0.15
    assert np.all(eta[0] < 0.62) and np.all(eta[0] > 0.45)
    # north_star's checkerboard half-sweeps on the same workload (R11): the same cone angle at every point
    # away from the first-order jump of a = 2, the same peak of M_par for a = 0 (profiles/r01_schedules.md)
    c = section4.run(temps, chains=2, equilibrate=10000, steps=4000, every=50, seed=11, schedule="checkerboard")
    eta_c, Mpar_c = c["mean"][:, :, 3], c["mean"][:, :, 2]
    print("checkerboard eta - stride eta", np.round(eta_c - eta, 3))
    away = np.ones_like(eta, dtype=bool)
    away[2, iT[4.0]] = False
    # measured: 0.012 on this shortened protocol (slow relaxation inside the transition windows), 0.003 on the paper's
    assert np.max(np.abs(eta_c - eta)[away]) < 0.025, np.abs(eta_c - eta).max()
    assert abs(Mpar_c[1, iT[4.5]] - Mpar[1, iT[4.5]]) < 0.03


def _onsager_energy(T):
    """Exact energy per spin of the infinite square-lattice Ising model with J = 1 (Onsager 1944):
    u = -coth(2b) [1 + (2/pi)(2 tanh^2(2b) - 1) K(k)], k = 2 sinh(2b) / cosh^2(2b), b = 1/T."""
    from scipy.special import ellipk
    b = 1.0 / np.asarray(T, dtype=np.float64)
    k = 2.0 * np.sinh(2 * b) / np.cosh(2 * b) ** 2
    return -(1.0 / np.tanh(2 * b)) * (1.0 + (2.0 / np.pi) * (2.0 * np.tanh(2 * b) ** 2 - 1.0) * ellipk(k * k))


@pytest.mark.parametrize("schedule", ["checkerboard", "stride", "single"])
def test_ising_limit_matches_onsager(dsmc_mod, schedule):
    """A pin that owes nothing to the oracle: with g = 0, K = 0 and the reversal move the path is plain Metropolis
    sampling of the nearest-neighbour Ising model (no dipole sum, so simultaneous updates of non-neighbouring sites are
    exact), whose energy per spin is known in closed form.  Temperatures away from T_c = 2.269 so that the finite
    lattice (L = 64) is within 1e-3 of the infinite one.  Checks the acceptance rule, the random numbers, the
    neighbour indexing and the energy observable of all three schedules on the GPU."""
    L, R = 64, 8
    T = np.array([1.2, 1.6, 1.9, 2.0, 2.7, 3.0, 3.5, 5.0], dtype=np.float32)
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=0.0, K2=0.0, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = 1.0
    ctx.set_spins(s)
    flip = dsmc_mod.DSMC_TRIAL_FLIP
    if schedule == "checkerboard":
        ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)

    def advance(first, n):
        if schedule == "checkerboard":
            ctx.run(T, 77, 2 * first, 2 * n, flags=flip)
        else:
            l = 32 if schedule == "stride" else 64
            ctx.sublattice_run(T, 77, first * l * l, n * l * l, l, flags=flip)

    burn, n_rec, every = 1500, 300, 10
    advance(0, burn)
    E = np.empty((n_rec, R))
    for k in range(n_rec):
        advance(burn + k * every, every)
        E[k] = ctx.observables()[:, 0]
        assert np.all(np.abs(ctx.get_spins()[:, 2]) == 1.0) if k == 0 else True
    ctx.close()
    mean = E.mean(axis=0)
    # standard error with a factor 2 for the correlation left between states 10 sweeps apart
    se = 2.0 * E.std(axis=0, ddof=1) / np.sqrt(n_rec)
    exact = _onsager_energy(T)
    print("T        ", T)
    print("E/N GPU  ", np.round(mean, 4))
    print("Onsager  ", np.round(exact, 4))
    print("3 sigma  ", np.round(3 * se, 4))
    assert np.all(np.abs(mean - exact) < 3 * se + 1.5e-3), np.abs(mean - exact)


@pytest.mark.parametrize("cfg_id", [2, 3])
def test_checkerboard_is_unbiased_on_baseline_configs(dsmc_mod, cfg_id):
    """north_star's checkerboard updates N/2 sites against one frozen field, the coarsest use of the paper's
    approximation (R11).  GPU-vs-oracle parity cannot show whether that biases the physics, because the oracle
    restates the same schedule; exact single-spin Metropolis (stride l = L, one site per pass, no approximation;
    resident kernel) can.  BASELINE configs 2 and 3 (g = 0.1): thermal averages of E/N, m_z^2-free quantities M_par and
    eta from 8 independent chains per temperature under each schedule must agree within 4 standard errors."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    L, chains = c["L"], 8
    K2c, K4c = inputs.anisotropy(cfg_id)
    Tc = inputs.temperatures(cfg_id)
    R = c["R"] * chains
    T, K2, K4 = np.repeat(Tc, chains), np.repeat(K2c, chains), np.repeat(K4c, chains)
    sweeps, burn, every = (1500, 700, 10) if cfg_id == 2 else (1200, 600, 10)
    res = {}
    for schedule in ("checkerboard", "single"):
        ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=c["g"], K2=K2, K4=K4)
        ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
        ctx.set_spins(inputs.up_spins(L, R) if c["init"] == "up" else inputs.random_spins(L, R, 5))
        if schedule == "checkerboard":
            ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
        ctx.ensemble_reset()
        for k in range(0, sweeps, every):
            if schedule == "checkerboard":
                ctx.run(T, 21, 2 * k, 2 * every)
            else:
                ctx.sublattice_run(T, 21, k * L * L, every * L * L, L)
            if k >= burn:
                ctx.ensemble_add()
        mean = ctx.ensemble_get()[0].reshape(c["R"], chains, 8)
        ctx.close()
        res[schedule] = (mean.mean(axis=1), mean.std(axis=1, ddof=1) / np.sqrt(chains))
    (mc, sc), (ms, ss) = res["checkerboard"], res["single"]
    for q, name in ((0, "E/N"), (2, "M_par"), (3, "eta")):
        d = np.abs(mc[:, q] - ms[:, q])
        tol = 4.0 * np.sqrt(sc[:, q] ** 2 + ss[:, q] ** 2) + 2e-3
        print(name, "checkerboard", np.round(mc[:, q], 4))
        print(name, "single-spin ", np.round(ms[:, q], 4))
        assert np.all(d < tol), (name, d, tol)


@pytest.mark.parametrize("L,R,l,passes", [(64, 16, 32, 160), (32, 8, 16, 128), (16, 6, 4, 64), (12, 5, 12, 96), (64, 3, 64, 64)])
def test_incremental_run_lockstep(dsmc_mod, oracle, L, R, l, passes):
    """DSMC_INCREMENTAL (eq. 8 in reverse): the field of all sites kept in
    registers and corrected by W(c - t) . delta_c for the accepted moves only.  A run cannot be stopped between passes,
    so the kernel logs the margin dE/T + ln u of every trial; the oracle replays the same passes from the same state
    in fp64 (field from scratch every pass).  Every replica is its own chain: until its first decision inside the
    |margin| < 1e-4 band, margins must agree to the lock-step tolerance plus the drift of the running field, decisions
    must be identical and the final spins equal; at most a few chains may leave the comparison.  Finally the field the
    kernel ends with is compared with the field of its final state computed from scratch."""
    from paper_1211_6234_b200 import inputs
    J, g, K2, K4 = 1.0, 0.25, 0.6, 0.1
    n = (L // l) ** 2
    ctx = dsmc_mod.Dsmc(L, R, J=J, g=g, K2=K2, K4=K4)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    W = oracle.build_tensor_ewald(L)
    s0 = inputs.random_spins(L, R, 57)
    ctx.set_spins(s0)
    T = np.linspace(0.2, 1.6, R).astype(np.float32)
    log = torch.zeros((passes, R, n), dtype=torch.float32, device="cuda")
    ctx.sublattice_run(T, 0xABCD, 3, passes, l, flags=dsmc_mod.DSMC_INCREMENTAL, margin_log=log)
    got = log.cpu().numpy()
    s_gpu = ctx.get_spins()
    h_gpu = ctx.get_field()
    s = s0.astype(np.float64)
    alive = np.ones(R, dtype=bool)
    compared = accepted = 0
    for k in range(passes):
        ref = oracle.sublattice_pass(W, s, T, 0xABCD, 3 + k, l, J, g, K2, K4)
        ox, oy = ref["offset"]
        m_ref = np.stack([ref["margin"][:, oy + l * b, ox + l * a] for b in range(L // l) for a in range(L // l)], axis=1)
        band = np.abs(m_ref) < BAND
        ok = alive[:, None] & ~band
        assert np.all(np.abs(got[k] - m_ref)[ok] <= 4e-5 + 3e-6 * np.abs(m_ref)[ok]), (k, np.abs(got[k] - m_ref)[ok].max())
        assert np.array_equal((got[k] < 0)[ok], (m_ref < 0)[ok]), k
        compared += int(ok.sum())
        accepted += int((m_ref < 0)[ok].sum())
        alive &= ~band.any(axis=1)                              # a chain with an ambiguous decision may have branched off
    assert alive.sum() >= max(1, R - 2), alive
    assert 0 < accepted < compared
    assert np.max(np.abs(s_gpu[alive].astype(np.float64) - s[alive])) <= 1e-6
    # the running field against the field of the final state from scratch (fp64 direct sum)
    h_ref = oracle.dipole_field(W, s_gpu.astype(np.float64))
    d = h_gpu.astype(np.float64) - h_ref
    rel = np.sqrt((d ** 2).sum() / (h_ref ** 2).sum())
    print(f"L={L} l={l}: {compared} trials compared, {accepted} accepted, running field rel L2 {rel:.2e} max abs {np.abs(d).max():.2e}")
    assert rel <= 1e-5 and np.abs(d).max() <= 1e-4
    ctx.close()


def test_incremental_field_drift_and_refresh(dsmc_mod, oracle):
    """A whole refresh period and beyond at the paper's L = 64, l = 32 (4096 + 1000 passes: one refresh inside): the
    field the kernel carries stays within the field tolerances of the field of its own final state."""
    from paper_1211_6234_b200 import inputs
    L, R, l = 64, 8, 32
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2247, K2=1.685, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    ctx.set_spins(inputs.random_spins(L, R, 3))
    T = np.linspace(0.2, 1.6, R).astype(np.float32)
    W = oracle.build_tensor_ewald(L)
    for n_passes in (4096, 5096):
        ctx.sublattice_run(T, 9, 0, n_passes, l, flags=dsmc_mod.DSMC_INCREMENTAL)
        h_ref = oracle.dipole_field(W, ctx.get_spins().astype(np.float64))
        d = ctx.get_field().astype(np.float64) - h_ref
        rel = np.sqrt((d ** 2).sum() / (h_ref ** 2).sum())
        print(f"{n_passes} passes: running field rel L2 {rel:.2e} max abs {np.abs(d).max():.2e}")
        assert rel <= 1e-5 and np.abs(d).max() <= 1e-4
    with pytest.raises(dsmc_mod.DsmcError):                      # L * L > 4096
        big = dsmc_mod.Dsmc(128, 2)
        big.build_tensor()
        big.set_spins(inputs.random_spins(128, 2, 1))
        big.sublattice_run(np.ones(2, np.float32), 1, 0, 4, 64, flags=dsmc_mod.DSMC_INCREMENTAL)
    ctx.close()
