"""GPU parity of the FFT route of the dipole field (DSMC_FIELD_FFT) against the fp64 oracle's direct
sum: the same a1 step, the same tolerances as the direct-sum kernels."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

FIELD_REL_L2 = 1e-5
FIELD_MAX_ABS = 1e-4


@pytest.fixture(scope="module")
def dsmc_mod():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1211_6234_b200 as m
    from paper_1211_6234_b200 import build
    build.build()
    return m


def errs(h, ref, mask=None):
    d = h.astype(np.float64) - ref
    if mask is not None:
        d, ref = d[..., mask], ref[..., mask]
    return np.sqrt((d ** 2).sum() / (ref ** 2).sum()), np.abs(d).max()


@pytest.mark.parametrize("L,R", [(32, 8), (64, 16), (128, 4), (32, 2), (64, 6), (32, 64)])
def test_fft_field_parity_full(dsmc_mod, oracle, L, R):
    """Every supported transform length below 256 (N2 = 2, 4, 8), replica counts that give 1, 2, 3, 4, 8
    and 32 pairs per CTA; random, z-aligned and striped states; all colours."""
    from paper_1211_6234_b200 import inputs
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=0.1, K2=0.6, K4=0.0)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    assert ctx.field_kernel_kind() == 2
    W = oracle.build_tensor_ewald(L)
    x = np.arange(L)
    par = (x[:, None] + x[None, :]) % 2
    stripes = np.zeros((R, 3, L, L), dtype=np.float32)
    stripes[:, 2] = np.where((x // 4) % 2 == 0, 1.0, -1.0)[None, None, :]
    for s in (inputs.random_spins(L, R, 99), inputs.up_spins(L, R), stripes):
        ctx.set_spins(s)
        ref = oracle.dipole_field(W, s.astype(np.float64))
        rel, mx = errs(ctx.dipole_field(-1), ref)
        assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (L, R, rel, mx)
        for colour in (0, 1):
            hc = np.full((R, 3, L, L), 7.0, dtype=np.float32)
            ctx.dipole_field(colour, out=hc)
            assert np.all(hc[..., par != colour] == 7.0)
            rel, mx = errs(hc, ref, par == colour)
            assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (L, R, colour, rel, mx)
    ctx.close()


def test_fft_field_general_tensor(dsmc_mod, oracle):
    """A random W with no symmetry at all (not even, xx != yy): pins the direction of the correlation
    (rho = m - n), the component mixing and the complex multiplier."""
    from paper_1211_6234_b200 import inputs
    L, R = 32, 4
    rng = np.random.default_rng(5)
    W = rng.standard_normal((4, L, L)).astype(np.float32)
    ctx = dsmc_mod.Dsmc(L, R)
    ctx.set_tensor(W)
    ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    s = inputs.random_spins(L, R, 3)
    ctx.set_spins(s)
    ref = oracle.dipole_field(W.astype(np.float64), s.astype(np.float64))
    rel, mx = errs(ctx.dipole_field(-1), ref)
    assert rel <= FIELD_REL_L2, (rel, mx)
    ctx.close()


def test_fft_field_L256_sampled(dsmc_mod, oracle):
    """Config 5 at full size (N2 = 16): sampled targets on all replicas by the oracle's direct sum, the
    uniform-state closed form at every site, and agreement with the tiled direct-sum kernel."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[5]
    L, R = c["L"], c["R"]
    ctx = dsmc_mod.Dsmc(L, R, J=1.0, g=c["g"], K2=c["K2"], K4=c["K4"])
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    W = oracle.build_tensor_ewald(L)
    rng = np.random.default_rng(7)
    targets = rng.choice(L * L, size=48, replace=False).astype(np.int32)
    s = inputs.initial_spins(5)
    ctx.set_spins(s)
    h_direct = ctx.dipole_field(-1).copy()
    ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    h = ctx.dipole_field(-1)
    got = h.reshape(R, 3, L * L)[:, :, targets]
    ref = np.stack([oracle.dipole_field_sampled(W, s[r].astype(np.float64), targets).T for r in range(R)])
    d = got.astype(np.float64) - ref
    rel = np.sqrt((d ** 2).sum() / (ref ** 2).sum())
    assert rel <= FIELD_REL_L2 and np.abs(d).max() <= FIELD_MAX_ABS, (rel, np.abs(d).max())
    rel2, mx2 = errs(h, h_direct.astype(np.float64))
    assert rel2 <= 2e-5 and mx2 <= 2e-4, (rel2, mx2)              # two fp32 routes, each within tolerance
    ctx.set_spins(inputs.up_spins(L, R))
    h = ctx.dipole_field(-1)
    assert np.max(np.abs(h[:, 2] - 9.033621683100950)) < 5e-5 and np.max(np.abs(h[:, :2])) < 5e-5
    ctx.close()


def test_fft_lockstep(dsmc_mod, oracle):
    """Half-sweeps driven by the FFT field: decisions, margins and new spins against the oracle."""
    from paper_1211_6234_b200 import inputs
    from test_gpu_parity import lockstep
    c = inputs.CONFIGS[2]
    K2, K4 = inputs.anisotropy(2)
    ctx = dsmc_mod.Dsmc(c["L"], c["R"], J=1.0, g=c["g"], K2=K2, K4=K4)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
    W = oracle.build_tensor_ewald(c["L"])
    ctx.set_spins(inputs.initial_spins(2))
    lockstep(dsmc_mod, oracle, ctx, W, inputs.temperatures(2), K2, K4, 1.0, c["g"], seed=inputs.SEED_BASE + 2, steps=10)
    ctx.close()


def test_fft_unsupported_shapes(dsmc_mod):
    for (L, R) in ((12, 4), (32, 3), (16, 4)):
        ctx = dsmc_mod.Dsmc(L, R)
        with pytest.raises(dsmc_mod.DsmcError):
            ctx.select_field_kernel(dsmc_mod.DSMC_FIELD_FFT)
        ctx.close()


def test_largest_transform_L512(dsmc_mod, oracle):
    """The largest supported lattice of the FFT route (N2 = 32) and the tiled kernel at the same size,
    every target, against the harness fp64 FFT (pinned to the oracle in test_gpu_parity) plus sampled
    targets by the oracle's direct sum."""
    from paper_1211_6234_b200 import inputs
    from test_gpu_parity import _fft_field_fp64
    L, R = 512, 4
    ctx = dsmc_mod.Dsmc(L, R)
    ctx.build_tensor(dsmc_mod.DSMC_W_EWALD)
    W = ctx.get_tensor().astype(np.float64)                   # the table itself is checked at L <= 256
    s = inputs.random_spins(L, R, 2)
    ctx.set_spins(s)
    ref = _fft_field_fp64(W, s.astype(np.float64))
    targets = np.random.default_rng(1).choice(L * L, size=8, replace=False).astype(np.int32)
    direct = oracle.dipole_field_sampled(W, s[1].astype(np.float64), targets)
    assert np.max(np.abs(ref[1].reshape(3, L * L)[:, targets].T - direct)) < 1e-10
    for kind in (dsmc_mod.DSMC_FIELD_FFT, dsmc_mod.DSMC_FIELD_TILED):
        ctx.select_field_kernel(kind)
        rel, mx = errs(ctx.dipole_field(-1), ref)
        assert rel <= FIELD_REL_L2 and mx <= FIELD_MAX_ABS, (kind, rel, mx)
    ctx.close()
