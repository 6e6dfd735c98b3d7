"""dsmc_wall_counts_noalloc (include/dsmc.h): the allocation-free entry point whose reduction scratch is a static
device array inside libdsmc.so.  Its counts must equal those of the existing path (dsmc_wall_observables, which is
itself pinned to the fp64 CPU definition in test_gpu_parity.py) bit for bit -- they are integers -- on calls made one
after another, which share the static array.

Collected last on purpose (file name): the run uses `pytest -x`, and a failure here must not hide the
parity tests.  Passes alone in a fresh process and after the other tests (it depends on no state of theirs: the
entry point clears what it needs and looks the array's address up itself on first use).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _spins_with_zeros(L, R, seed):
    """Unit spins, iid on S^2, plus a sprinkling of exact axis spins so that sgn(0) = 0 terms of eq. 14 occur."""
    from paper_1211_6234_b200 import inputs
    s = inputs.random_spins(L, R, seed)
    rng = np.random.default_rng(seed)
    for r in range(R):
        ys, xs = np.divmod(rng.choice(L * L, 2 * L, replace=False), L)     # distinct sites: the spins stay unit
        axis = rng.integers(0, 3, 2 * L)
        s[r, :, ys, xs] = 0.0
        s[r, axis, ys, xs] = np.where(rng.random(2 * L) < 0.5, -1.0, 1.0).astype(np.float32)
    return s


def _existing_path(m, s):
    R, L = s.shape[0], s.shape[-1]
    ctx = m.Dsmc(L, R)
    ctx.set_spins(s)
    counts, _ = ctx.wall_observables()
    ctx.close()
    return counts


# consecutive calls share the static scratch: a large shape first, then smaller and odd ones whose partial-sum slots
# and tickets overlap what the previous call left behind, then the first shape again
SHAPES = [(64, 16), (48, 5), (6, 3), (4, 1), (256, 2), (64, 16)]


def test_noalloc_wall_counts_equal_the_existing_path_on_consecutive_calls():
    import torch
    import paper_1211_6234_b200 as m
    dev = torch.device("cuda:0")
    prepared = []
    for k, (L, R) in enumerate(SHAPES):
        s = _spins_with_zeros(L, R, 9100 + k)
        prepared.append((s, _existing_path(m, s), torch.from_numpy(s).to(dev),
                         torch.full((R, 6), -1, dtype=torch.int64, device=dev)))
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated(dev)
    for _ in range(2):                                     # back to back, no synchronisation in between
        for s, want, s_dev, out in prepared:
            m.wall_counts_noalloc(s_dev, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before
    for s, want, s_dev, out in prepared:
        got = out.cpu().numpy()
        assert np.array_equal(got, want), (s.shape, got, want)   # integers: bit exact
        assert got.sum() > 0


def test_noalloc_same_input_twice_in_a_row_on_a_side_stream():
    import torch
    import paper_1211_6234_b200 as m
    dev = torch.device("cuda:0")
    L, R = 128, 32
    s = _spins_with_zeros(L, R, 9200)
    want = _existing_path(m, s)
    s_dev = torch.from_numpy(s).to(dev)
    out = [torch.zeros((R, 6), dtype=torch.int64, device=dev) for _ in range(2)]
    torch.cuda.synchronize()
    side = torch.cuda.Stream(dev)
    with torch.cuda.stream(side):
        m.wall_counts_noalloc(s_dev, out[0], stream=side)
        m.wall_counts_noalloc(s_dev, out[1], stream=side)
    side.synchronize()
    assert np.array_equal(out[0].cpu().numpy(), want)
    assert np.array_equal(out[1].cpu().numpy(), want)


def test_noalloc_all_up_state_has_no_walls_and_stripes_count_exactly():
    """Closed forms (eq. 14): the uniform state has no wall; stripes of width 1 along y (s_z = (-1)^x) have
    n_h^z = 2 N and n_v^z = 0; the x and y components are zero everywhere, so each of their bonds counts 1."""
    import torch
    import paper_1211_6234_b200 as m
    dev = torch.device("cuda:0")
    L, R = 32, 2
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[0, 2] = 1.0
    s[1, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, :]
    out = torch.zeros((R, 6), dtype=torch.int64, device=dev)
    m.wall_counts_noalloc(torch.from_numpy(s).to(dev), out)
    N = L * L
    assert out.cpu().numpy().tolist() == [[N, N, N, N, 0, 0], [N, N, N, N, 2 * N, 0]]


def test_noalloc_refuses_sizes_beyond_the_static_array():
    import ctypes
    import torch
    import paper_1211_6234_b200 as m
    dev = torch.device("cuda:0")
    lib = m.load_library()
    s = torch.zeros((1025, 3, 4, 4), dtype=torch.float32, device=dev)
    out = torch.full((1025, 6), -7, dtype=torch.int64, device=dev)
    with pytest.raises(m.DsmcError, match="DSMC_NOALLOC_MAX_R = 1024"):
        m.wall_counts_noalloc(s, out)
    with pytest.raises(m.DsmcError, match="even"):
        m.wall_counts_noalloc(torch.zeros((1, 3, 5, 5), dtype=torch.float32, device=dev),
                              torch.zeros((1, 6), dtype=torch.int64, device=dev))
    err = ctypes.create_string_buffer(256)
    with torch.cuda.device(dev):
        # L beyond the limit: refused from the sizes alone, before any pointer is looked at
        assert lib.dsmc_wall_counts_noalloc(s.data_ptr(), 4098, 1, out.data_ptr(), None, err, len(err)) == -1
        assert b"DSMC_NOALLOC_MAX_L = 4096" in err.value
        # a host pointer would fault in the kernel: refused with a message instead
        host = np.zeros((1, 3, 4, 4), dtype=np.float32)
        assert lib.dsmc_wall_counts_noalloc(host.ctypes.data, 4, 1, out.data_ptr(), None, err, len(err)) == -1
        assert b"not device memory" in err.value
        assert lib.dsmc_wall_counts_noalloc(s.data_ptr(), 4, 1, out.data_ptr(), None, None, 0) == 0   # err is optional
    torch.cuda.synchronize()
    assert int(out[1:].min()) == -7 and int(out[1:].max()) == -7      # refused calls launched nothing
