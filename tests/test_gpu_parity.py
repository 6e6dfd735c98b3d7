"""GPU parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
  field: relative L2 <= 1e-5 and max abs <= 1e-4 (h in lattice units, i.e. 1e-4*g on g*h);
  decisions: identical outside |dE/T + ln u| < 1e-4, the ambiguous ones counted, < 1e-4 of trials.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

FIELD_REL_L2 = 1e-5
FIELD_MAX_ABS = 1e-4
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


def make_ctx(m, cfg_id, inputs, R=None):
    c = inputs.CONFIGS[cfg_id]
    K2, K4 = inputs.anisotropy(cfg_id)
    R = R or c["R"]
    ctx = m.Dsmc(c["L"], R, J=1.0, g=c["g"], K2=K2[:R], K4=K4[:R])
    ctx.build_tensor(m.DSMC_W_EWALD)
    return ctx


def field_errors(h_gpu, h_ref, mask=None):
    d = h_gpu.astype(np.float64) - h_ref
    if mask is not None:
        d = d[..., mask]
        h_ref = h_ref[..., mask]
    return np.sqrt((d ** 2).sum() / (h_ref ** 2).sum()), np.abs(d).max()


@pytest.mark.parametrize("L", [4, 8, 32, 64])
@pytest.mark.parametrize("method", ["ewald", "image"])
def test_tensor_parity(dsmc_mod, oracle, L, method):
    ctx = dsmc_mod.Dsmc(L, 1)
    if method == "ewald":
        ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
        ref = oracle.build_tensor_ewald(L)
    else:
        ctx.build_tensor(dsmc_mod.DSMC_W_IMAGE, 64, 1)
        ref = oracle.build_tensor_image(L, 64, 1)
    W = ctx.get_tensor()
    # fp64 on both sides, one rounding to fp32 on the GPU side: half an fp32 ulp of each entry
    assert np.all(np.abs(W.astype(np.float64) - ref) <= 6.1e-8 * np.abs(ref) + 1e-12)
    ctx.close()


def test_tensor_parity_L256(dsmc_mod, oracle):
    ctx = dsmc_mod.Dsmc(256, 1)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    W = ctx.get_tensor()
    ref = oracle.build_tensor_ewald(256)
    assert np.all(np.abs(W.astype(np.float64) - ref) <= 6.1e-8 * np.abs(ref) + 1e-12)
    ctx.close()


@pytest.mark.parametrize("cfg_id", [1, 2, 3, 4])
@pytest.mark.parametrize("generic", [False, True])
def test_field_parity_full(dsmc_mod, oracle, cfg_id, generic):
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    L, R = c["L"], c["R"]
    ctx = make_ctx(dsmc_mod, cfg_id, inputs)
    if generic and ctx.field_kernel_kind() == 0:
        pytest.skip("shape already uses the generic kernel")
    W = oracle.build_tensor_ewald(L)
    x = np.arange(L)
    par = (x[:, None] + x[None, :]) % 2
    if generic:
        ctx.select_field_kernel(0)
        assert ctx.field_kernel_kind() == 0
    states = [inputs.initial_spins(cfg_id), inputs.up_spins(L, R), inputs.random_spins(L, R, 99)]
    for s in states:
        ctx.set_spins(s)
        ref = oracle.dipole_field(W, s.astype(np.float64))
        h = ctx.dipole_field(-1)
        rel, mx = field_errors(h, ref)
        assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (cfg_id, rel, mx)
        for colour in (0, 1):
            hc = np.full((R, 3, L, L), 7.0, dtype=np.float32)
            ctx.dipole_field(colour, out=hc)
            assert np.all(hc[..., par != colour] == 7.0)            # inactive targets untouched
            rel, mx = field_errors(hc, ref, par == colour)
            assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (cfg_id, colour, rel, mx)
    ctx.close()


def test_field_parity_L256_sampled(dsmc_mod, oracle):
    """Config 5 at full size, in the launch configuration bench.py times: sampled targets on all
    replicas by the oracle's direct sum."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[5]
    L, R = c["L"], c["R"]
    ctx = make_ctx(dsmc_mod, 5, inputs)
    W = oracle.build_tensor_ewald(L)
    rng = np.random.default_rng(7)
    targets = rng.choice(L * L, size=48, replace=False).astype(np.int32)
    for s in (inputs.initial_spins(5), inputs.up_spins(L, R)):
        ctx.set_spins(s)
        h = ctx.dipole_field(-1)
        got = h.reshape(R, 3, L * L)[:, :, targets]                      # [R][3][nt]
        ref = np.stack([oracle.dipole_field_sampled(W, s[r].astype(np.float64), targets).T for r in range(R)])
        d = got.astype(np.float64) - ref
        rel = np.sqrt((d ** 2).sum() / (ref ** 2).sum())
        assert rel <= FIELD_REL_L2 and np.abs(d).max() <= FIELD_MAX_ABS, (rel, np.abs(d).max())
    # a property that holds at any size: all +z -> h_z = 4 zeta(3/2) beta(3/2) at every site
    assert np.max(np.abs(h[:, 2] - 9.033621683100950)) < 5e-5 and np.max(np.abs(h[:, :2])) < 5e-5
    ctx.close()


def lockstep(dsmc_mod, oracle, ctx, W, T, K2, K4, J, g, seed, steps, first_step=0):
    """Per half-sweep: copy the GPU state into the oracle, run both with the same (seed, step),
    compare field, decisions and new spins; continue from the GPU's state."""
    L, R = ctx.L, ctx.R
    x = np.arange(L)
    par = (x[:, None] + x[None, :]) % 2
    acc_d = torch.zeros((R, L, L), dtype=torch.uint8, device="cuda")
    mar_d = torch.zeros((R, L, L), dtype=torch.float32, device="cuda")
    ambiguous = trials = 0
    worst_rel = worst_abs = 0.0
    for step in range(first_step, first_step + steps):
        colour = step & 1
        act = par == colour
        s_before = ctx.get_spins()
        s_or = s_before.astype(np.float64)
        out = oracle.halfsweep(W, s_or, T, seed, step, J, g, K2, K4)
        ctx.halfsweep(T, seed, step, accept_out=acc_d, margin_out=mar_d)
        s_after = ctx.get_spins()
        acc = acc_d.cpu().numpy()
        mar = mar_d.cpu().numpy()
        # (1) decisions: identical outside the band
        m_or = out["margin"][:, act]
        a_or = out["accept"][:, act].astype(bool)
        a_gpu = acc[:, act].astype(bool)
        amb = np.abs(m_or) < BAND
        assert np.array_equal(a_gpu[~amb], a_or[~amb]), (step, np.sum(a_gpu[~amb] != a_or[~amb]))
        ambiguous += int(amb.sum())
        trials += amb.size
        # the margin the kernel saw agrees with the oracle's to fp32 accuracy
        dm = np.abs(mar[:, act] - m_or)
        assert np.all(dm <= 2e-5 + 3e-6 * np.abs(m_or)), (step, dm.max())
        # (2) new spins: accepted -> the trial spin, rejected -> bit-unchanged, other colour untouched
        acc_full = np.zeros((R, L, L), dtype=bool)
        acc_full[:, act] = a_gpu
        chg = np.broadcast_to(acc_full[:, None], s_after.shape)
        assert np.array_equal(s_after[~chg], s_before[~chg])
        assert np.max(np.abs(s_after[chg].astype(np.float64) - out["trial"][chg]), initial=0.0) <= 1e-6
        # (3) the frozen field the half-sweep used: recompute it on the state at entry
        h_ref = out["h"]
        worst = _field_of_state(ctx, s_before, colour)
        rel, mx = field_errors(worst, h_ref, act)
        worst_rel, worst_abs = max(worst_rel, rel), max(worst_abs, mx)
        ctx.set_spins(s_after)
    assert worst_rel <= FIELD_REL_L2 and worst_abs <= FIELD_MAX_ABS, (worst_rel, worst_abs)
    assert ambiguous <= max(1, BAND_FRACTION * trials) or ambiguous / trials < BAND_FRACTION, (ambiguous, trials)
    return ambiguous, trials


_scratch = {}


def _field_of_state(ctx, s, colour):
    key = (ctx.L, ctx.R)
    if key not in _scratch:
        import paper_1211_6234_b200 as m
        c2 = m.Dsmc(ctx.L, ctx.R)
        c2.set_tensor(ctx.get_tensor())
        _scratch[key] = c2
    c2 = _scratch[key]
    c2.set_spins(s)
    h = np.zeros((ctx.R, 3, ctx.L, ctx.L), dtype=np.float32)
    return c2.dipole_field(colour, out=h)


def test_lockstep_config1(dsmc_mod, oracle):
    """Config 1 in full: L = 8, R = 1, 100 sweeps, every half-sweep compared (image-sum W, A = 64)."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[1]
    ctx = dsmc_mod.Dsmc(c["L"], c["R"], J=1.0, g=c["g"], K2=c["K2"], K4=c["K4"])
    ctx.build_tensor(dsmc_mod.DSMC_W_IMAGE, 64, 1)
    W = oracle.build_tensor_image(c["L"], 64, 1)
    ctx.set_spins(inputs.initial_spins(1))
    T = inputs.temperatures(1)
    lockstep(dsmc_mod, oracle, ctx, W, T, c["K2"], c["K4"], 1.0, c["g"], seed=inputs.SEED_BASE + 1, steps=200)
    ctx.close()


@pytest.mark.parametrize("cfg_id,steps", [(2, 40), (3, 12), (4, 4)])
def test_lockstep_configs(dsmc_mod, oracle, cfg_id, steps):
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    ctx = make_ctx(dsmc_mod, cfg_id, inputs)
    W = oracle.build_tensor_ewald(c["L"])
    K2, K4 = inputs.anisotropy(cfg_id)
    ctx.set_spins(inputs.initial_spins(cfg_id))
    T = inputs.temperatures(cfg_id)
    amb, tr = lockstep(dsmc_mod, oracle, ctx, W, T, K2, K4, 1.0, c["g"], seed=inputs.SEED_BASE + cfg_id, steps=steps)
    print(f"config {cfg_id}: ambiguous {amb} of {tr} trials")
    ctx.close()


def test_init_spins_parity(dsmc_mod, oracle):
    for (L, R) in ((8, 1), (32, 8)):
        ctx = dsmc_mod.Dsmc(L, R)
        ctx.init_spins(dsmc_mod.DSMC_INIT_RANDOM, seed=4242)
        s = ctx.get_spins()
        ref = oracle.init_spins(L, R, 0, 4242)
        assert np.max(np.abs(s - ref)) <= 1e-6
        assert np.array_equal(s[:, 2].astype(np.float64), ref[:, 2])      # z = 2u - 1 is exact in fp32
        ctx.init_spins(dsmc_mod.DSMC_INIT_UP)
        assert np.array_equal(ctx.get_spins(), oracle.init_spins(L, R, 1, 0).astype(np.float32))
        ctx.close()


@pytest.mark.parametrize("cfg_id", [1, 2, 3])
def test_observables_parity(dsmc_mod, oracle, cfg_id):
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    ctx = make_ctx(dsmc_mod, cfg_id, inputs)
    W = oracle.build_tensor_ewald(c["L"])
    K2, K4 = inputs.anisotropy(cfg_id)
    for s in (inputs.initial_spins(cfg_id), inputs.random_spins(c["L"], c["R"], 5)):
        ctx.set_spins(s)
        got = ctx.observables()
        ref = oracle.observables(W, s.astype(np.float64), 1.0, c["g"], K2.astype(np.float64), K4.astype(np.float64))
        assert np.max(np.abs(got - ref)) <= 2e-6, np.abs(got - ref).max(0)
    ctx.close()


def test_set_get_roundtrip_and_errors(dsmc_mod):
    from paper_1211_6234_b200 import inputs
    ctx = dsmc_mod.Dsmc(12, 5)                                   # ragged: L not a multiple of 8, odd R
    s = inputs.random_spins(12, 5, 3)
    ctx.set_spins(s)
    assert np.array_equal(ctx.get_spins(), s)
    d = torch.from_numpy(s).cuda()
    ctx.set_spins(d)
    out = torch.empty_like(d)
    ctx.get_spins(out)
    assert torch.equal(out, d)
    with pytest.raises(dsmc_mod.DsmcError):                      # tensor not built
        ctx.dipole_field(-1)
    ctx.build_tensor()
    with pytest.raises(dsmc_mod.DsmcError):                      # T must be > 0
        ctx.halfsweep(np.zeros(5, np.float32), 1, 0)
    with pytest.raises(dsmc_mod.DsmcError):                      # bad colour
        ctx.dipole_field(2)
    with pytest.raises(dsmc_mod.DsmcError):                      # odd L
        dsmc_mod.Dsmc(7, 1)
    ctx.close()


def test_ragged_shape_field_and_sweep(dsmc_mod, oracle):
    """L = 12, R = 5: not a multiple of any tile size; full parity through the generic kernel."""
    from paper_1211_6234_b200 import inputs
    L, R, g = 12, 5, 0.3
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=g, K2=0.4, K4=-0.1)
    ctx.build_tensor()
    W = oracle.build_tensor_ewald(L)
    s = inputs.random_spins(L, R, 17)
    ctx.set_spins(s)
    rel, mx = field_errors(ctx.dipole_field(-1), oracle.dipole_field(W, s.astype(np.float64)))
    assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS
    T = np.linspace(0.3, 1.5, R).astype(np.float32)
    lockstep(dsmc_mod, oracle, ctx, W, T, 0.4, -0.1, 1.0, g, seed=77, steps=6)
    ctx.close()


def test_halfsweep_parity_L256_sampled(dsmc_mod, oracle):
    """Config 5 at full size, in the launch configuration bench.py times (tiled field kernel +
    4-replica Metropolis kernel): decisions, margins and new spins at sampled active sites of every
    replica, each recomputed one by one by the oracle (direct-sum field, trial draw, dE)."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[5]
    L, R, g = c["L"], c["R"], c["g"]
    K2, K4 = inputs.anisotropy(5)
    T = inputs.temperatures(5)
    seed = inputs.SEED_BASE + 5
    ctx = make_ctx(dsmc_mod, 5, inputs)
    assert ctx.field_kernel_kind() == 1
    W = oracle.build_tensor_ewald(L)
    ctx.set_spins(inputs.initial_spins(5))
    acc_d = torch.zeros((R, L, L), dtype=torch.uint8, device="cuda")
    mar_d = torch.zeros((R, L, L), dtype=torch.float32, device="cuda")
    rng = np.random.default_rng(11)
    ambiguous = trials = 0
    for step in (0, 1):
        s_before = ctx.get_spins()
        ctx.halfsweep(T, seed, step, accept_out=acc_d, margin_out=mar_d)
        s_after = ctx.get_spins()
        acc = acc_d.cpu().numpy().reshape(R, L * L)
        mar = mar_d.cpu().numpy().reshape(R, L * L)
        xs, ys = rng.integers(0, L, 24), rng.integers(0, L, 24)
        xs = (xs - ((xs + ys) % 2 != step)) % L                      # move onto the active colour
        assert np.all((xs + ys) % 2 == step)
        # include the lattice corners' neighbourhood (periodic wrap of the neighbour fetch)
        targets = np.unique(np.concatenate([ys * L + xs, [step * 1, (L - 1) * L + (L - 1 - (1 - step)) % L]])).astype(np.int32)
        targets = targets[((targets % L) + (targets // L)) % 2 == step]
        for r in range(R):
            s_one = s_before[r].astype(np.float64)
            h = oracle.dipole_field_sampled(W, s_one, targets)
            for k, n in enumerate(targets):
                s_new, u, _ = oracle.trial_draw(seed, int(n), r, step)
                dE = oracle.delta_e(W, s_one, h[k], int(n), s_new, 1.0, g, float(K2[r]), float(K4[r]))
                m_or = dE / float(T[r]) + np.log(u)
                trials += 1
                assert abs(mar[r, n] - m_or) <= 2e-5 + 3e-6 * abs(m_or), (step, r, n, mar[r, n], m_or)
                if abs(m_or) < BAND:
                    ambiguous += 1
                else:
                    assert bool(acc[r, n]) == (m_or < 0), (step, r, n, m_or)
                got = s_after[r, :, n // L, n % L]
                if acc[r, n]:
                    assert np.max(np.abs(got - s_new)) <= 1e-6
                else:
                    assert np.array_equal(got, s_before[r, :, n // L, n % L])
        # the other colour is untouched at any size
        x = np.arange(L)
        par = (x[:, None] + x[None, :]) % 2
        assert np.array_equal(s_after[..., par != step], s_before[..., par != step])
        # every spin is still a unit vector
        assert np.max(np.abs(np.sum(s_after.astype(np.float64) ** 2, axis=1) - 1.0)) < 1e-6
    assert ambiguous <= max(1, BAND_FRACTION * trials), (ambiguous, trials)
    ctx.close()


def test_observables_parity_L256_one_replica(dsmc_mod, oracle):
    """Config 5's lattice size through the tiled kernel: observables of 4 replicas on the GPU, the
    first one recomputed by the oracle (one full direct-sum field at L = 256)."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[5]
    L, g = c["L"], c["g"]
    ctx = dsmc_mod.Dsmc(L, 4, J=1.0, g=g, K2=c["K2"], K4=c["K4"])
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    assert ctx.field_kernel_kind() == 1
    s = inputs.random_spins(L, 4, 21)
    ctx.set_spins(s)
    got = ctx.observables()
    W = oracle.build_tensor_ewald(L)
    ref = oracle.observables(W, s[:1].astype(np.float64), 1.0, g, c["K2"], c["K4"])
    assert np.max(np.abs(got[:1] - ref)) <= 2e-6, np.abs(got[:1] - ref)
    ctx.close()


def _window_means(obs):
    """obs[sweep][R][4] -> mean over the second half of the run, [R][4]"""
    obs = np.asarray(obs)
    return obs[obs.shape[0] // 2:].mean(axis=0)


def _long_run_compare(dsmc_mod, oracle, L, R, g, K2, K4, T, n_sweeps, n_seeds, start):
    """north_star: 'Observables over long runs: agreement within 3 sigma'.  Independent seeds on the
    two sides (so the two sets of chains are statistically independent), the same sweep window,
    sigma from the across-seed scatter (eq. 13)."""
    from paper_1211_6234_b200 import inputs
    W = oracle.build_tensor_ewald(L)
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=g, K2=K2, K4=K4)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    gpu, cpu = [], []
    for k in range(n_seeds):
        seed_g, seed_o = 1000 + k, 2000 + k
        s0 = inputs.up_spins(L, R) if start == "up" else inputs.random_spins(L, R, seed_g)
        ctx.set_spins(s0)
        rec = []
        for sw in range(n_sweeps):
            ctx.halfsweep(T, seed_g, 2 * sw)
            ctx.halfsweep(T, seed_g, 2 * sw + 1)
            rec.append(ctx.observables())
        gpu.append(_window_means(rec))
        s = (inputs.up_spins(L, R) if start == "up" else inputs.random_spins(L, R, seed_o)).astype(np.float64)
        rec = []
        for sw in range(n_sweeps):
            oracle.halfsweep(W, s, T, seed_o, 2 * sw, 1.0, g, K2, K4, want=())
            oracle.halfsweep(W, s, T, seed_o, 2 * sw + 1, 1.0, g, K2, K4, want=())
            rec.append(oracle.observables(W, s, 1.0, g, K2, K4))
        cpu.append(_window_means(rec))
    ctx.close()
    gpu, cpu = np.array(gpu), np.array(cpu)                       # [seed][R][4]
    diff = gpu.mean(0) - cpu.mean(0)
    sigma = np.sqrt(gpu.var(0, ddof=1) / n_seeds + cpu.var(0, ddof=1) / n_seeds)
    # m_z of a symmetric double-well flips sign between chains: compare |m_z| there
    zscore = np.abs(diff) / np.maximum(sigma, 1e-7)
    return zscore, diff, sigma, gpu, cpu


def test_long_run_observables_3sigma(dsmc_mod, oracle):
    """(The configs as written are in tests/test_gpu_longrun.py; this one keeps the oracle's own direct-sum field.)
    A config-2-shaped run shortened to what the fp64 oracle finishes in about a minute:
    L = 16, R = 8, T = 0.2 ... 1.6, g = 0.1, K2 = 0.6, 16 independent seeds per side, 300 sweeps,
    means over sweeps 150-299 of E/N, m_z, M_par, eta per replica."""
    L, R = 16, 8
    T = np.linspace(0.2, 1.6, R).astype(np.float32)
    z, diff, sigma, gpu, cpu = _long_run_compare(dsmc_mod, oracle, L, R, 0.1, 0.6, 0.0, T, 300, 16, "up")
    print("max z-score", z.max(), "at", np.unravel_index(z.argmax(), z.shape))
    assert np.all(z <= 3.0), (z, diff, sigma)
    # and the runs are not trivially frozen: the hottest replica has disordered, the coldest has not
    assert abs(gpu.mean(0)[-1, 1]) < 0.3 and gpu.mean(0)[0, 1] > 0.8


@pytest.mark.parametrize("L,R", [(8, 1), (12, 5), (32, 8), (64, 16), (256, 64)])
def test_wall_observables_parity(dsmc_mod, oracle, L, R):
    """eq. 14-15: integer wall counts bit-exact against the oracle (random, striped and uniform
    states, a state with exact zeros), derived ratios to rounding."""
    from paper_1211_6234_b200 import inputs
    ctx = dsmc_mod.Dsmc(L, R)
    x = np.arange(L)
    stripes = inputs.random_spins(L, R, 8)
    stripes[:, 2] = np.abs(stripes[:, 2]) * np.where((x // 4) % 2 == 0, 1.0, -1.0)[None, None, :]
    zeros = inputs.random_spins(L, R, 9)
    zeros[:, 0, ::3, ::2] = 0.0
    zeros[:, 2, 1::2, :] = -0.0
    for s in (inputs.random_spins(L, R, 7), stripes, inputs.up_spins(L, R), zeros):
        ctx.set_spins(s)
        counts, derived = ctx.wall_observables()
        ref = oracle.wall_counts(s.astype(np.float64))
        assert np.array_equal(counts, ref), (L, R)
        assert np.max(np.abs(derived - oracle.wall_order(L, ref))) <= 1e-15
    ctx.close()


def _fft_field_fp64(W, s):
    """Harness-only third opinion: the circular correlation h_n = sum_m W(m - n) s_m by
    numpy's fp64 FFT.  Checked against the oracle's direct sum before it is trusted (below)."""
    Wh = np.fft.fft2(W, axes=(-2, -1))                      # [4][L][L]
    sh = np.fft.fft2(s, axes=(-2, -1))                      # [R][3][L][L]
    M = np.conj(Wh)                                         # correlation: conj of the kernel's transform
    hx = M[0] * sh[:, 0] + M[1] * sh[:, 1]
    hy = M[1] * sh[:, 0] + M[2] * sh[:, 1]
    hz = M[3] * sh[:, 2]
    return np.real(np.fft.ifft2(np.stack([hx, hy, hz], axis=1), axes=(-2, -1)))


def test_field_parity_L256_every_target(dsmc_mod, oracle):
    """Config 5 at full size, EVERY target of every replica, both direct-sum launch configurations
    (colour 0 and 1 half-sweep fields of the tiled kernel) and the FFT route, against an fp64 FFT
    evaluation in the harness that is first pinned to the oracle's direct sum (L = 32 in full, and
    sampled targets at L = 256)."""
    from paper_1211_6234_b200 import inputs
    W32 = oracle.build_tensor_ewald(32)
    s32 = inputs.random_spins(32, 3, 5).astype(np.float64)
    assert np.max(np.abs(_fft_field_fp64(W32, s32) - oracle.dipole_field(W32, s32))) < 1e-12
    c = inputs.CONFIGS[5]
    L, R = c["L"], c["R"]
    W = oracle.build_tensor_ewald(L)
    s = inputs.initial_spins(5)
    ref = _fft_field_fp64(W, s.astype(np.float64))
    targets = np.random.default_rng(3).choice(L * L, size=16, replace=False).astype(np.int32)
    direct = oracle.dipole_field_sampled(W, s[7].astype(np.float64), targets)
    assert np.max(np.abs(ref[7].reshape(3, L * L)[:, targets].T - direct)) < 1e-11
    ctx = make_ctx(dsmc_mod, 5, inputs)
    ctx.set_spins(s)
    for kind in (dsmc_mod.DSMC_FIELD_TILED, dsmc_mod.DSMC_FIELD_FFT):
        ctx.select_field_kernel(kind)
        h = np.zeros((R, 3, L, L), dtype=np.float32)
        ctx.dipole_field(0, out=h)
        ctx.dipole_field(1, out=h)
        rel, mx = field_errors(h, ref)
        print("kind", kind, "rel L2", rel, "max abs", mx)
        assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (kind, rel, mx)
    ctx.close()


def test_field_parity_z_aligned_every_target(dsmc_mod, oracle):
    """The worst case of fp32 accumulation named by SURVEY.md section 7: the fully z-aligned state (config 3's start),
    where every term of h_z has the same sign.  EVERY target of every replica of config 5's shape (L = 256, R = 64),
    both half-sweep launch configurations of the tiled kernel, against the fp64 FFT harness field (pinned to the
    direct sum in test_field_parity_L256_every_target and tests/test_oracle_harness.py) and against the closed form
    h_z = 4 zeta(3/2) beta(3/2).  The bound asserted is half the north_star tolerance: the headroom the far -> near
    source order of the tiled kernel buys."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[5]
    L, R = c["L"], c["R"]
    W = oracle.build_tensor_ewald(L)
    ctx = make_ctx(dsmc_mod, 5, inputs)
    assert ctx.field_kernel_kind() == 1
    for name, s in (("z-aligned", inputs.up_spins(L, R)), ("random", inputs.initial_spins(5))):
        ref = _fft_field_fp64(W, s.astype(np.float64))
        ctx.set_spins(s)
        h = np.zeros((R, 3, L, L), dtype=np.float32)
        ctx.dipole_field(0, out=h)
        ctx.dipole_field(1, out=h)
        rel, mx = field_errors(h, ref)
        print(name, "tiled kernel, L = 256, R = 64: rel L2", rel, "max abs", mx)
        assert rel <= FIELD_REL_L2 and mx <= 0.5 * FIELD_MAX_ABS, (name, rel, mx)
        if name == "z-aligned":
            assert np.max(np.abs(ref[:, 2] - 9.033621683100950)) < 1e-9       # the reference itself: closed form
            assert np.max(np.abs(h[:, 2] - 9.033621683100950)) <= 0.5 * FIELD_MAX_ABS
    ctx.close()


@pytest.mark.parametrize("L,R", [(512, 4), (1024, 4)])
def test_field_parity_tiled_large_L(dsmc_mod, oracle, L, R):
    """The accuracy the tiled kernel guarantees as a function of L (include/dsmc.h, dsmc_select_field_kernel): every
    target, z-aligned (worst case) and random state, up to the largest lattice the kernel accepts (L = 1024: an
    accumulator then runs over 65 536 sources); beyond it dsmc_select_field_kernel(TILED) refuses."""
    from paper_1211_6234_b200 import inputs
    ctx = dsmc_mod.Dsmc(L, R)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)                               # (the table's own parity: test_tensor_parity*)
    assert ctx.field_kernel_kind() == 1
    Wf = ctx.get_tensor().astype(np.float64)                              # the fp32 table, exactly, on both sides
    for name, s in (("z-aligned", inputs.up_spins(L, R)), ("random", inputs.random_spins(L, R, 12))):
        ref = _fft_field_fp64(Wf, s.astype(np.float64))
        ctx.set_spins(s)
        h = ctx.dipole_field(-1)
        rel, mx = field_errors(h, ref)
        print(name, "tiled kernel, L =", L, ": rel L2", rel, "max abs", mx)
        assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (name, L, rel, mx)
    ctx.close()
    big = dsmc_mod.Dsmc(2048, 4)
    assert big.field_kernel_kind() == 0                                   # automatic choice falls back to the generic kernel
    with pytest.raises(dsmc_mod.DsmcError):
        big.select_field_kernel(dsmc_mod.DSMC_FIELD_TILED)
    big.close()


@pytest.mark.parametrize("L,R", [(256, 64), (32, 8), (64, 16), (32, 16), (512, 16), (64, 48), (64, 128), (32, 64)])
@pytest.mark.parametrize("flip", [False, True])
def test_benchmarked_metropolis_instantiation_is_the_tested_one(dsmc_mod, L, R, flip):
    """The lock-step tests pass accept_out / margin_out, which selects the hooked instantiation of the 4-replica
    Metropolis kernel; bench.py, dsmc_halfsweep and dsmc_run launch the instantiations without hooks (step in the
    kernel parameters, or read from the device counter inside the replayed graph).  From one state, the three must
    leave bit-identical spins, half-sweep by half-sweep and over a run long enough to go through the graph: this
    closes the chain oracle -> hooked kernel -> production kernels (eq. 7).  With the FFT field and
    R % 16 == 0 the production path is the FUSED one (the decision taken inside the field's last pass, field_fft.cu:
    fftc_row_update_kernel), the hooked path field kernels + metropolis4_kernel: the same test ties those together.
    From R = 32 and L = 64 up dsmc_run replays that path as independent chains of launches, one per group (or several
    groups) of 16 replicas, on a block-major copy of the spins (dsmc_api.cu: build_sweep_graph, replay_sweep_graph): 4
    chains at (256, 64), 3 at (64, 48), 8 at (64, 128), one at (32, 64); the plain calls always run as one."""
    from paper_1211_6234_b200 import inputs
    T = np.linspace(0.1, 2.0, R).astype(np.float32)
    flags = dsmc_mod.DSMC_TRIAL_FLIP if flip else 0
    ctxs = []
    for _ in range(3):
        c = dsmc_mod.Dsmc(L, R, J=1.0, g=0.1, K2=0.6, K4=0.1)
        if ctxs:
            c.set_tensor(ctxs[0].get_tensor())
        else:
            c.build_tensor(dsmc_mod.DSMC_W_EWALD)
        c.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)        # the field is not under test: the fast one
        c.set_spins(inputs.random_spins(L, R, 41))
        ctxs.append(c)
    plain, hooked, graph = ctxs
    acc = torch.zeros((R, L, L), dtype=torch.uint8, device="cuda")
    mar = torch.zeros((R, L, L), dtype=torch.float32, device="cuda")
    n_half = 4 + 4 * 8 + 7                                       # odd tail: plain prefix, replayed graph, plain tail
    for k in range(n_half):
        plain.halfsweep(T, 123, k, flags=flags)
        hooked.halfsweep(T, 123, k, flags=flags, accept_out=acc, margin_out=mar)
        if k < 2:
            assert np.array_equal(plain.get_spins(), hooked.get_spins()), k
    graph.run(T, 123, 0, n_half, flags=flags)
    s_plain, s_hooked, s_graph = plain.get_spins(), hooked.get_spins(), graph.get_spins()
    assert np.array_equal(s_plain, s_hooked)
    assert np.array_equal(s_plain, s_graph)
    assert not np.array_equal(s_plain, inputs.random_spins(L, R, 41))
    for c in ctxs:
        c.close()


def test_ensemble_statistics_are_bit_reproducible(dsmc_mod):
    """The observable reductions use no floating-point atomics (warp shuffles, shared memory in index order, per-CTA
    partials summed in CTA order): two runs of dsmc_run_recorded give bit-identical dsmc_ensemble_get, and
    dsmc_observables / dsmc_staggered_magnetisation repeat bit for bit -- on a power-of-two R below the warp size,
    a ragged R, R = 64 at config 5's lattice size, and R above the block size."""
    from paper_1211_6234_b200 import inputs
    for (L, R, fft) in ((32, 8, True), (12, 5, False), (256, 64, True), (8, 300, False)):
        T = np.linspace(0.3, 1.7, R).astype(np.float32)
        got = []
        for rep in range(2):
            ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=0.6, K4=0.1)
            ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
            if fft:
                ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
            ctx.set_spins(inputs.random_spins(L, R, 6))
            ctx.ensemble_reset()
            ctx.run_recorded(T, 5, 0, 12, 2)
            mean, var, se, n = ctx.ensemble_get()
            ob = [ctx.observables() for _ in range(3)]
            st = [ctx.staggered_magnetisation() for _ in range(2)]
            assert np.array_equal(ob[0], ob[1]) and np.array_equal(ob[0], ob[2]) and np.array_equal(st[0], st[1])
            got.append((mean, var, se, ob[0], st[0], ctx.wall_observables()[0]))
            ctx.close()
        for a, b in zip(*got):
            assert np.array_equal(a, b), (L, R)


def test_set_spins_debug_check(dsmc_mod):
    """|s| = 1 is the caller's contract, checked to 1e-5 when debugging is on -> DSMC_EINVAL."""
    from paper_1211_6234_b200 import inputs
    L, R = 16, 4
    ctx = dsmc_mod.Dsmc(L, R)
    ctx.build_tensor()
    s = inputs.random_spins(L, R, 1)
    bad = s.copy()
    bad[2, :, 5, 7] *= 1.0 + 5e-5
    ctx.set_spins(bad)                                           # default: not checked, not renormalised
    assert np.array_equal(ctx.get_spins(), bad)
    ctx.set_debug(True)
    ctx.set_spins(s)
    with pytest.raises(dsmc_mod.DsmcError, match="unit vector"):
        ctx.set_spins(bad)
    with pytest.raises(dsmc_mod.DsmcError):                      # the rejected state counts as not set
        ctx.dipole_field(-1)
    nan = s.copy()
    nan[0, 1, 0, 0] = np.nan
    with pytest.raises(dsmc_mod.DsmcError):
        ctx.set_spins(nan)
    ok = s.copy()
    ok[1, :, 3, 3] *= 1.0 + 2e-6                                 # inside the 1e-5 band
    ctx.set_spins(ok)
    ctx.set_debug(False)
    ctx.set_spins(bad)
    ctx.close()


@pytest.mark.parametrize("fft", [False, True])
def test_ensemble_statistics_parity(dsmc_mod, oracle, fft):
    """eq. 13 / eq. 18 accumulated on the device over a run (config 2's shape, 24 recorded states two
    sweeps apart) against the oracle: per-snapshot observables and wall order parameters recomputed by
    the oracle from the recorded states, then its ensemble mean, variance and standard error."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[2]
    L, R, g = c["L"], c["R"], c["g"]
    K2, K4 = inputs.anisotropy(2)
    T = inputs.temperatures(2)
    ctx = make_ctx(dsmc_mod, 2, inputs)
    if fft:
        ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    W = oracle.build_tensor_ewald(L)
    ctx.set_spins(inputs.initial_spins(2))
    ctx.ensemble_reset()
    snaps = []
    for k in range(24):
        ctx.run(T, 77, 4 * k, 4)
        ctx.ensemble_add()
        s = ctx.get_spins().astype(np.float64)
        ob = oracle.observables(W, s, 1.0, g, K2.astype(np.float64), K4.astype(np.float64))
        snaps.append(np.concatenate([ob, oracle.wall_order(L, oracle.wall_counts(s))], axis=1))
    mean, var, se, n = ctx.ensemble_get()
    m_ref, v_ref, se_ref = oracle.ensemble(np.array(snaps))
    assert n == 24
    assert np.max(np.abs(mean - m_ref)) <= 2e-6                       # the per-snapshot observable tolerance
    assert np.all(np.abs(var - v_ref) <= 1e-5 * np.sqrt(v_ref) + 1e-10)
    assert np.all(np.abs(se - se_ref) <= 1e-5 + 1e-3 * se_ref)
    assert var[:, 0].max() > 1e-6                                     # the run is not frozen
    ctx.ensemble_reset()
    with pytest.raises(dsmc_mod.DsmcError):
        ctx.ensemble_get()
    ctx.close()


@pytest.mark.parametrize("L,R,kind,flip", [(32, 8, 1, False), (32, 8, 2, False), (12, 5, 0, False), (64, 16, 2, False),
                                           (32, 8, 2, True), (12, 5, 0, True), (64, 32, 2, False), (64, 32, 2, True)])
def test_run_graph_replay_is_bit_identical(dsmc_mod, L, R, kind, flip):
    """dsmc_run / dsmc_run_ex replay a captured CUDA graph of 8 sweeps with the step counter on the device: the
    trajectory must be bit-identical to calling dsmc_halfsweep step by step (odd first step, ragged
    tail, runs too short for the graph, a second run with another seed and after switching the field kernel;
    flip = the reversal move through dsmc_run_ex)."""
    from paper_1211_6234_b200 import inputs
    T = np.linspace(0.3, 1.5, R).astype(np.float32)
    flags = dsmc_mod.DSMC_TRIAL_FLIP if flip else 0
    a = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=0.5, K4=0.1)
    b = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=0.5, K4=0.1)
    a.build_tensor(dsmc_mod.DSMC_W_EWALD)
    b.set_tensor(a.get_tensor())
    for ctx in (a, b):
        ctx.select_field_kernel(kind)
        ctx.set_spins(inputs.random_spins(L, R, 3))
    for (seed, first, n) in ((11, 7, 75), (12, 100, 52), (12, 152, 9), (13, 161, 40)):
        a.run(T, seed, first, n, flags=flags)
        for k in range(n):
            b.halfsweep(T, seed, first + k, flags=flags)
        assert np.array_equal(a.get_spins(), b.get_spins()), (seed, first, n)
    if kind == 2:                                               # the graph is rebuilt when the kernel changes
        for ctx in (a, b):
            ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_AUTO)
        a.run(T, 12, 300, 44, flags=flags)
        for k in range(44):
            b.halfsweep(T, 12, 300 + k, flags=flags)
        assert np.array_equal(a.get_spins(), b.get_spins())
    a.close()
    b.close()


def test_sharded_ladder_is_bit_identical(dsmc_mod):
    """One ladder of 8 replicas run as a whole and as two shards of 4 with dsmc_set_replica_offset (what
    run_config does under torchrun, one shard per GPU): the random streams are those of the whole ladder, and
    with the FFT field (whose arithmetic per replica pair does not depend on R) and shards that use the same
    Metropolis kernel (R % 4 == 0) the trajectories are identical bit for bit -- through dsmc_init_spins and
    through dsmc_run (graph replay)."""
    L, R = 32, 8
    T = np.linspace(0.3, 1.7, R).astype(np.float32)
    K2 = np.linspace(0.4, 0.8, R).astype(np.float32)
    K4 = np.linspace(-0.1, 0.1, R).astype(np.float32)
    whole = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=K2, K4=K4)
    whole.build_tensor(dsmc_mod.DSMC_W_EWALD)
    whole.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    whole.init_spins(dsmc_mod.DSMC_INIT_RANDOM, seed=9)
    s0 = whole.get_spins()
    whole.run(T, 21, 0, 40)
    ref = whole.get_spins()
    for (lo, hi) in ((0, 4), (4, 8)):
        part = dsmc_mod.Dsmc(L, hi - lo, J=1.0, g=0.2, K2=K2[lo:hi], K4=K4[lo:hi])
        part.set_tensor(whole.get_tensor())
        part.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
        part.set_replica_offset(lo)
        part.init_spins(dsmc_mod.DSMC_INIT_RANDOM, seed=9)
        assert np.array_equal(part.get_spins(), s0[lo:hi])
        part.run(T[lo:hi], 21, 0, 40)
        assert np.array_equal(part.get_spins(), ref[lo:hi]), (lo, hi)
        part.close()
    whole.close()


_PDL_AB_SCRIPT = """
import hashlib, sys
import numpy as np
import paper_1211_6234_b200 as m
L, R, graph = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3])
T = np.linspace(0.3, 1.7, R).astype(np.float32)
ctx = m.Dsmc(L, R, J=1.0, g=0.2, K2=np.full(R, 0.6, np.float32), K4=np.full(R, 0.1, np.float32))
ctx.build_tensor(m.DSMC_W_EWALD)
ctx.select_field_kernel(m.DSMC_FIELD_FFT)
ctx.init_spins(m.DSMC_INIT_RANDOM, seed=5)
if graph:
    ctx.run(T, 31, 0, 120)                       # bulk replayed from the captured graph
else:
    for k in range(60):
        ctx.halfsweep(T if k == 0 else None, 31, k)
print(hashlib.sha256(np.ascontiguousarray(ctx.get_spins()).tobytes()).hexdigest())
"""


@pytest.mark.parametrize("L,R,graph", [(32, 8, 0), (32, 8, 1), (64, 16, 1), (128, 4, 1), (256, 8, 0)])
def test_dependent_launch_is_bit_identical(L, R, graph):
    """the kernels of a sweep are chained by programmatic dependent launches; each waits for its
    predecessor before it touches shared state, so nothing but the launch overlaps.  A missing or misplaced wait shows up as a
    race on spins, field, spectrum scratch or step counter: the same run with plain launches (DSMC_NO_PDL=1, read once
    per process, hence the subprocesses) must leave the same spins to the last bit -- launch by launch and through
    the replayed graph, on one-wave and many-wave grids."""
    import os, subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    digest = []
    for no_pdl in ("0", "1"):
        env = dict(os.environ, DSMC_NO_PDL=no_pdl)
        p = subprocess.run([sys.executable, "-c", _PDL_AB_SCRIPT, str(L), str(R), str(graph)], cwd=root, env=env,
                           capture_output=True, text=True, timeout=600)
        assert p.returncode == 0, p.stderr[-2000:]
        digest.append(p.stdout.strip().splitlines()[-1])
    assert len(digest[0]) == 64 and digest[0] == digest[1]


@pytest.mark.parametrize("L,R,every,fft", [(32, 8, 1, True), (32, 8, 3, True), (64, 4, 20, True), (12, 5, 2, False)])
def test_run_recorded_matches_separate_calls(dsmc_mod, L, R, every, fft):
    """dsmc_run_recorded (a state recorded every k steps) = the same dsmc_run / dsmc_ensemble_add calls one by
    one: identical spins (the graph of `every` sweeps + record replays the same kernels with the same Philox counters),
    the same number of snapshots, statistics equal up to the rounding of the fp64 atomic sums."""
    T = np.linspace(0.4, 1.5, R).astype(np.float32)
    n_rec, first = 9, 6
    pair = []
    for _ in range(2):
        ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=0.15, K2=0.6, K4=0.1)
        ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
        if fft:
            ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
        ctx.init_spins(dsmc_mod.DSMC_INIT_RANDOM, seed=3)
        ctx.ensemble_reset()
        pair.append(ctx)
    a, b = pair
    a.run_recorded(T, 17, first, n_rec, every)
    for k in range(n_rec):
        b.run(T if k == 0 else None, 17, first + 2 * every * k, 2 * every)
        b.ensemble_add()
    assert np.array_equal(a.get_spins(), b.get_spins())
    ma, va, sa, na = a.ensemble_get()
    mb, vb, sb, nb = b.ensemble_get()
    assert na == nb == n_rec
    np.testing.assert_allclose(ma, mb, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(va, vb, rtol=1e-9, atol=1e-15)
    # a second call continues the same ensemble and trajectory
    a.run_recorded(None, 17, first + 2 * every * n_rec, 2, every)
    b.run(None, 17, first + 2 * every * n_rec, 4 * every)
    assert np.array_equal(a.get_spins(), b.get_spins())
    assert a.ensemble_get()[3] == n_rec + 2
    with pytest.raises(Exception):
        a.run_recorded(None, 17, 1, 2, every)      # odd first step
    with pytest.raises(Exception):
        a.run_recorded(None, 17, 0, 2, 0)          # every < 1
    a.close()
    b.close()


@pytest.mark.gpu
def test_stream_footprint_leaves_the_state_alone(dsmc_mod):
    """dsmc_stream_footprint (bench.py's measured denominator of the Metropolis roofline) rewrites every spin of the
    colour with the bits it read: the state, and a run continued from it, must not change."""
    from paper_1211_6234_b200 import inputs
    L, R = 64, 16
    T = np.linspace(0.3, 1.5, R).astype(np.float32)
    a = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=0.5, K4=0.1)
    b = dsmc_mod.Dsmc(L, R, J=1.0, g=0.2, K2=0.5, K4=0.1)
    a.build_tensor(dsmc_mod.DSMC_W_EWALD)
    b.set_tensor(a.get_tensor())
    s0 = inputs.random_spins(L, R, 77)
    for c in (a, b):
        c.set_spins(s0)
        c.halfsweep(T, 5, 0)
    for colour in (0, 1, 1, 0):
        a.stream_footprint(colour)
    assert np.array_equal(a.get_spins(), b.get_spins())
    for c in (a, b):
        c.halfsweep(T, 5, 1)
    assert np.array_equal(a.get_spins(), b.get_spins())
    with pytest.raises(dsmc_mod.DsmcError):
        a.stream_footprint(2)
    c5 = dsmc_mod.Dsmc(12, 5)
    c5.set_spins(inputs.random_spins(12, 5, 1))
    with pytest.raises(dsmc_mod.DsmcError):
        c5.stream_footprint(0)                                  # R % 4 != 0
    for c in (a, b, c5):
        c.close()
