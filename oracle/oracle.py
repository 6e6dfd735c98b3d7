"""ctypes wrapper around the fp64 CPU oracle (oracle/dsmc_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It shares
nothing with paper_1211_6234_b200 (the CUDA path) and never imports it.

All arrays are numpy float64, C-contiguous, in the layouts of dsmc_oracle.c:
  W[4][L][L] (xx, xy, yy, zz; W[c][rho_y][rho_x]),  s[R][3][L][L],  h[R][3][L][L].
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dsmc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_u8_p = ctypes.POINTER(ctypes.c_uint8)
_c_u32_p = ctypes.POINTER(ctypes.c_uint32)
_c_int_p = ctypes.POINTER(ctypes.c_int)


def build(force=False):
    """Compile liboracle.so with gcc (plain C, -O2, OpenMP on outer loops only)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
    subprocess.check_call(cmd)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_delta_e.restype = ctypes.c_double
        _lib.oracle_num_threads.restype = ctypes.c_int
        _lib.oracle_philox4x32_10.restype = None
        _lib.oracle_trial_draw.restype = None
    return _lib


def _d(a):
    return a.ctypes.data_as(_c_double_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _per_replica(v, R):
    a = np.empty(R, dtype=np.float64)
    a[:] = v
    return a


def num_threads():
    return int(lib().oracle_num_threads())


def build_tensor_image(L, A=64, tail=1):
    W = np.empty((4, L, L), dtype=np.float64)
    rc = lib().oracle_build_tensor_image(int(L), int(A), int(tail), _d(W))
    assert rc == 0, rc
    return W


def build_tensor_ewald(L, alphaL=2.5, nreal=6, nk=12):
    W = np.empty((4, L, L), dtype=np.float64)
    rc = lib().oracle_build_tensor_ewald(int(L), ctypes.c_double(alphaL), int(nreal), int(nk), _d(W))
    assert rc == 0, rc
    return W


def dipole_field(W, s, colour=-1, h=None):
    s = _f64(s)
    R, _, L, _ = s.shape
    W = _f64(W)
    if h is None:
        h = np.zeros_like(s)
    rc = lib().oracle_dipole_field(L, R, _d(W), _d(s), int(colour), _d(h))
    assert rc == 0, rc
    return h


def dipole_field_sampled(W, s_one, targets):
    """Field of ONE replica s_one[3][L][L] at the listed linear site indices."""
    s_one = _f64(s_one)
    L = s_one.shape[-1]
    W = _f64(W)
    t = np.ascontiguousarray(targets, dtype=np.int32)
    out = np.empty((len(t), 3), dtype=np.float64)
    rc = lib().oracle_dipole_field_sampled(L, _d(W), _d(s_one), len(t),
                                           t.ctypes.data_as(_c_int_p), _d(out))
    assert rc == 0, rc
    return out


def energy(W, s, J, g, K2, K4, parts=False):
    s = _f64(s)
    R, _, L, _ = s.shape
    W = _f64(W)
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    E = np.empty(R, dtype=np.float64)
    P = np.empty((R, 3), dtype=np.float64)
    rc = lib().oracle_energy(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4),
                             _d(W), _d(s), _d(E), _d(P))
    assert rc == 0, rc
    return (E, P) if parts else E


def philox4x32_10(ctr, key):
    c = (ctypes.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (ctypes.c_uint32 * 4)()
    lib().oracle_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def trial_draw(seed, site, replica, step, tag=0):
    """-> (s'[3], u, raw[4]) for the counter (site, replica, step, tag) and key seed."""
    out = (ctypes.c_double * 4)()
    raw = (ctypes.c_uint32 * 4)()
    lib().oracle_trial_draw(ctypes.c_uint64(seed), ctypes.c_uint32(site), ctypes.c_uint32(replica),
                            ctypes.c_uint64(step), ctypes.c_uint32(tag), out, raw)
    return np.array(out[:3]), float(out[3]), [int(v) for v in raw]


def init_spins(L, R, mode, seed):
    s = np.empty((R, 3, L, L), dtype=np.float64)
    rc = lib().oracle_init_spins(int(L), int(R), int(mode), ctypes.c_uint64(seed), _d(s))
    assert rc == 0, rc
    return s


def delta_e(W, s_one, h_n, n, s_new, J, g, K2, K4):
    s_one = _f64(s_one)
    L = s_one.shape[-1]
    W = _f64(W)
    h_n = _f64(h_n)
    s_new = _f64(s_new)
    return float(lib().oracle_delta_e(L, ctypes.c_double(J), ctypes.c_double(g), ctypes.c_double(K2),
                                      ctypes.c_double(K4), _d(W), _d(s_one), _d(h_n), int(n),
                                      _d(s_new)))


def halfsweep(W, s, T, seed, step, J, g, K2, K4, want=("h", "accept", "margin", "trial"),
              sequential=False):
    """One checkerboard half-sweep IN PLACE on s (float64 [R][3][L][L]).

    Returns a dict with the requested side outputs (full-lattice arrays; only the
    active colour's entries are meaningful)."""
    assert s.dtype == np.float64 and s.flags.c_contiguous
    R, _, L, _ = s.shape
    W = _f64(W)
    T = _per_replica(T, R)
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    N = L * L
    out = {}
    if sequential:
        acc = np.zeros((R, L, L), dtype=np.uint8)
        mar = np.zeros((R, L, L), dtype=np.float64)
        rc = lib().oracle_halfsweep_sequential(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2),
                                               _d(K4), _d(W), _d(s), _d(T), ctypes.c_uint64(seed),
                                               ctypes.c_uint64(step), acc.ctypes.data_as(_c_u8_p), _d(mar))
        assert rc == 0, rc
        out["accept"] = acc
        out["margin"] = mar
        return out
    h = np.zeros((R, 3, L, L), dtype=np.float64) if "h" in want else None
    acc = np.zeros((R, L, L), dtype=np.uint8) if "accept" in want else None
    mar = np.zeros((R, L, L), dtype=np.float64) if "margin" in want else None
    tri = np.zeros((R, 3, L, L), dtype=np.float64) if "trial" in want else None
    rc = lib().oracle_halfsweep(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4), _d(W),
                                _d(s), _d(T), ctypes.c_uint64(seed), ctypes.c_uint64(step),
                                _d(h) if h is not None else None,
                                acc.ctypes.data_as(_c_u8_p) if acc is not None else None,
                                _d(mar) if mar is not None else None,
                                _d(tri) if tri is not None else None)
    assert rc == 0, rc
    if h is not None:
        out["h"] = h
    if acc is not None:
        out["accept"] = acc
    if mar is not None:
        out["margin"] = mar
    if tri is not None:
        out["trial"] = tri
    return out


def halfsweep_given_field(W, s, h, T, seed, step, J, g, K2, K4, want=()):
    """Step (ii) of the half-sweep IN PLACE on s with the frozen field h[R][3][L][L] of the state at entry
    handed in (halfsweep() is "h <- dipole_field(W, s, colour), then this"); W supplies W(0) only."""
    assert s.dtype == np.float64 and s.flags.c_contiguous
    R, _, L, _ = s.shape
    W = _f64(W)
    h = _f64(h)
    assert h.shape == s.shape
    T = _per_replica(T, R)
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    acc = np.zeros((R, L, L), dtype=np.uint8) if "accept" in want else None
    mar = np.zeros((R, L, L), dtype=np.float64) if "margin" in want else None
    tri = np.zeros((R, 3, L, L), dtype=np.float64) if "trial" in want else None
    rc = lib().oracle_halfsweep_given_field(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4), _d(W),
                                            _d(s), _d(T), ctypes.c_uint64(seed), ctypes.c_uint64(step), _d(h), None,
                                            acc.ctypes.data_as(_c_u8_p) if acc is not None else None,
                                            _d(mar) if mar is not None else None,
                                            _d(tri) if tri is not None else None)
    assert rc == 0, rc
    out = {}
    if acc is not None:
        out["accept"] = acc
    if mar is not None:
        out["margin"] = mar
    if tri is not None:
        out["trial"] = tri
    return out


def observables_given_field(s, h, J, g, K2, K4):
    """observables() with the full-lattice field h = dipole_field(W, s) handed in."""
    s = _f64(s)
    h = _f64(h)
    R, _, L, _ = s.shape
    assert h.shape == s.shape
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    out = np.empty((R, 4), dtype=np.float64)
    rc = lib().oracle_observables_given_field(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4),
                                              _d(s), _d(h), _d(out))
    assert rc == 0, rc
    return out


def observables(W, s, J, g, K2, K4):
    s = _f64(s)
    R, _, L, _ = s.shape
    W = _f64(W)
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    out = np.empty((R, 4), dtype=np.float64)
    rc = lib().oracle_observables(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4),
                                  _d(W), _d(s), _d(out))
    assert rc == 0, rc
    return out


def wall_counts(s):
    """eq. 14 per replica: int64 [R][6] = n_h^x, n_v^x, n_h^y, n_v^y, n_h^z, n_v^z."""
    s = _f64(s)
    R, _, L, _ = s.shape
    out = np.zeros((R, 6), dtype=np.int64)
    rc = lib().oracle_wall_counts(L, R, _d(s), out.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)))
    assert rc == 0, rc
    return out


def wall_order(L, counts):
    """[R][4] = wall density, O_x, O_y, O_z (eq. 15, per snapshot)."""
    counts = np.ascontiguousarray(counts, dtype=np.int64)
    R = counts.shape[0]
    out = np.zeros((R, 4), dtype=np.float64)
    rc = lib().oracle_wall_order(L, R, counts.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), _d(out))
    assert rc == 0, rc
    return out


def sublattice_offset(seed, pass_index, l):
    off = (ctypes.c_int * 2)()
    lib().oracle_sublattice_offset.restype = None
    lib().oracle_sublattice_offset(ctypes.c_uint64(seed), ctypes.c_uint64(pass_index), int(l), off)
    return int(off[0]), int(off[1])


def sublattice_pass(W, s, T, seed, pass_index, l, J, g, K2, K4, flip=False, sequential=False):
    """One pass of the paper's stride-l schedule (App. A) IN PLACE on s.
    -> dict(offset, accept[R][L][L], margin[R][L][L], trial[R][3][L][L]); update sites only."""
    assert s.dtype == np.float64 and s.flags.c_contiguous
    R, _, L, _ = s.shape
    W = _f64(W)
    T = _per_replica(T, R)
    K2 = _per_replica(K2, R)
    K4 = _per_replica(K4, R)
    off = (ctypes.c_int * 2)()
    acc = np.zeros((R, L, L), dtype=np.uint8)
    mar = np.zeros((R, L, L), dtype=np.float64)
    tri = np.zeros((R, 3, L, L), dtype=np.float64)
    rc = lib().oracle_sublattice_pass(L, R, ctypes.c_double(J), ctypes.c_double(g), _d(K2), _d(K4), _d(W),
                                      _d(s), _d(T), ctypes.c_uint64(seed), ctypes.c_uint64(pass_index),
                                      int(l), int(bool(flip)), int(bool(sequential)), off,
                                      acc.ctypes.data_as(_c_u8_p), _d(mar), _d(tri))
    assert rc == 0, rc
    return {"offset": (int(off[0]), int(off[1])), "accept": acc, "margin": mar, "trial": tri}


def staggered(s):
    """App. B's staggered magnetisation per replica: [R][3] = m_h, m_v, m_st."""
    s = _f64(s)
    R, _, L, _ = s.shape
    out = np.zeros((R, 3), dtype=np.float64)
    rc = lib().oracle_staggered(L, R, _d(s), _d(out))
    assert rc == 0, rc
    return out


def ensemble(x):
    """x[n snapshots][...] -> (mean, var, se) over the first axis: eq. 13 and eq. 18."""
    x = _f64(x)
    n = x.shape[0]
    K = int(np.prod(x.shape[1:])) if x.ndim > 1 else 1
    mean, var, se = np.zeros(K), np.zeros(K), np.zeros(K)
    rc = lib().oracle_ensemble(int(n), K, _d(x.reshape(n, K)), _d(mean), _d(var), _d(se))
    assert rc == 0, rc
    shp = x.shape[1:]
    return mean.reshape(shp), var.reshape(shp), se.reshape(shp)
