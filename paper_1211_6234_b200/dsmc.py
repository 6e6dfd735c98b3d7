"""Thin Python binding of the C ABI in include/dsmc.h (argument marshalling only).

PyTorch supplies device memory (one workspace tensor) and the CUDA stream; all arithmetic of the
path runs inside libdsmc.so.  There is no CPU fallback: a missing library or GPU raises.
"""
import ctypes
import os

import numpy as np

DSMC_HOST, DSMC_DEVICE = 0, 1
DSMC_W_IMAGE, DSMC_W_EWALD = 0, 1
DSMC_REUSE_FIELD = 1
DSMC_TRIAL_FLIP = 2
DSMC_NO_RESIDENT = 4
DSMC_INCREMENTAL = 8
DSMC_INIT_RANDOM, DSMC_INIT_UP = 0, 1
DSMC_FIELD_AUTO, DSMC_FIELD_GENERIC, DSMC_FIELD_TILED, DSMC_FIELD_FFT = -1, 0, 1, 2

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdsmc.so")
_lib = None

# every symbol include/dsmc.h declares: (name, restype, argtypes)
_vp, _i, _f, _u64, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_uint64, ctypes.c_size_t
ABI = [
    ("dsmc_create", _i, [ctypes.POINTER(_vp), _i, _i, _f, _f, _f, _f]),
    ("dsmc_set_replica_offset", _i, [_vp, ctypes.c_uint32]),
    ("dsmc_set_anisotropy", _i, [_vp, _vp, _vp]),
    ("dsmc_workspace_bytes", _sz, [_i, _i]),
    ("dsmc_bind", _i, [_vp, _vp, _sz, _vp]),
    ("dsmc_build_tensor", _i, [_vp, _i, _i, _i]),
    ("dsmc_get_tensor", _i, [_vp, _vp, _i]),
    ("dsmc_set_tensor", _i, [_vp, _vp, _i]),
    ("dsmc_set_spins", _i, [_vp, _vp, _i]),
    ("dsmc_get_spins", _i, [_vp, _vp, _i]),
    ("dsmc_init_spins", _i, [_vp, _i, _u64]),
    ("dsmc_dipole_field", _i, [_vp, _i, _vp, _i]),
    ("dsmc_get_field", _i, [_vp, _vp, _i]),
    ("dsmc_halfsweep", _i, [_vp, _vp, _u64, _u64]),
    ("dsmc_halfsweep_ex", _i, [_vp, _vp, _u64, _u64, _i, _vp, _vp]),
    ("dsmc_run", _i, [_vp, _vp, _u64, _u64, _u64]),
    ("dsmc_run_ex", _i, [_vp, _vp, _u64, _u64, _u64, _i]),
    ("dsmc_run_recorded", _i, [_vp, _vp, _u64, _u64, _u64, _i, _i]),
    ("dsmc_sublattice_pass", _i, [_vp, _vp, _u64, _u64, _i, _i, _vp, _vp, _vp]),
    ("dsmc_sublattice_run", _i, [_vp, _vp, _u64, _u64, _u64, _i, _i]),
    ("dsmc_sublattice_run_ex", _i, [_vp, _vp, _u64, _u64, _u64, _i, _i, _vp]),
    ("dsmc_observables", _i, [_vp, _vp]),
    ("dsmc_wall_observables", _i, [_vp, _vp, _vp]),
    ("dsmc_staggered_magnetisation", _i, [_vp, _vp]),
    ("dsmc_ensemble_reset", _i, [_vp]),
    ("dsmc_ensemble_add", _i, [_vp]),
    ("dsmc_ensemble_get", _i, [_vp, _vp, _vp, _vp, _vp]),
    ("dsmc_set_debug", _i, [_vp, _i]),
    ("dsmc_set_timing", _i, [_vp, _i]),
    ("dsmc_last_timing", _i, [_vp, _vp]),
    ("dsmc_launch_count", _u64, [_vp]),
    ("dsmc_field_kernel_kind", _i, [_vp]),
    ("dsmc_select_field_kernel", _i, [_vp, _i]),
    ("dsmc_field_kernel_supported", _i, [_vp, _i]),
    ("dsmc_fp32_fma_peak", _i, [_vp, _vp]),
    ("dsmc_stream_footprint", _i, [_vp, _i]),
    ("dsmc_wall_counts_noalloc", _i, [_vp, _i, _i, _vp, _vp, ctypes.c_char_p, _sz]),
    ("dsmc_destroy", _i, [_vp]),
    ("dsmc_last_error", ctypes.c_char_p, [_vp]),
    ("dsmc_version", ctypes.c_char_p, []),
]


class DsmcError(RuntimeError):
    pass


def load_library(path=None):
    """dlopen libdsmc.so and set the prototypes; raises if it has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _LIB_PATH
    if not os.path.exists(p):
        raise DsmcError(f"{p} not found: build it with `python -m paper_1211_6234_b200.build` "
                        "(there is no CPU fallback)")
    lib = ctypes.CDLL(p)
    for name, res, args in ABI:
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    if path is None:
        _lib = lib
    return lib


def _np_f32(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def wall_counts_noalloc(s, counts, stream=None):
    """dsmc_wall_counts_noalloc: eq. 14 wall counts of s (torch CUDA float32 [R][3][L][L]) into counts (torch CUDA
    int64 [R][6]) with no device allocation anywhere in the call (scratch = a static device array in the library;
    limits DSMC_NOALLOC_MAX_R / _L in include/dsmc.h).  Asynchronous on `stream` (default: torch's current stream);
    calls that overlap on one GPU race."""
    import torch
    lib = load_library()
    if not (isinstance(s, torch.Tensor) and s.is_cuda and s.is_contiguous() and s.dtype == torch.float32 and s.dim() == 4
            and s.shape[1] == 3 and s.shape[2] == s.shape[3]):
        raise TypeError("s: expected a contiguous CUDA float32 tensor [R][3][L][L]")
    R, L = int(s.shape[0]), int(s.shape[2])
    if not (isinstance(counts, torch.Tensor) and counts.is_cuda and counts.is_contiguous() and counts.dtype == torch.int64
            and tuple(counts.shape) == (R, 6) and counts.device == s.device):
        raise TypeError(f"counts: expected a contiguous CUDA int64 tensor [{R}][6] on {s.device}")
    err = ctypes.create_string_buffer(256)
    with torch.cuda.device(s.device):
        st = stream if stream is not None else torch.cuda.current_stream(s.device)
        rc = lib.dsmc_wall_counts_noalloc(s.data_ptr(), L, R, counts.data_ptr(), st.cuda_stream, err, len(err))
    if rc != 0:
        raise DsmcError(f"dsmc error {rc}: {err.value.decode()}")


class Dsmc:
    """One simulation context: L x L lattice, R replicas.  Mirrors the dsmc_* calls one to one."""

    def __init__(self, L, R, J=1.0, g=0.1, K2=0.6, K4=0.0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise DsmcError("no CUDA device: the dsmc path has no CPU fallback")
        self._torch = torch
        self.lib = load_library()
        self.L, self.R = int(L), int(R)
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self._h = _vp()
        rc = self.lib.dsmc_create(ctypes.byref(self._h), self.L, self.R, J, g,
                                  float(np.atleast_1d(K2)[0]), float(np.atleast_1d(K4)[0]))
        if rc != 0:
            raise DsmcError(f"dsmc_create({L}, {R}) failed: {rc}")
        nbytes = self.lib.dsmc_workspace_bytes(self.L, self.R)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._check(self.lib.dsmc_bind(self._h, self._ws_ptr, nbytes, self.stream.cuda_stream))
        if np.ndim(K2) > 0 or np.ndim(K4) > 0:
            self.set_anisotropy(K2, K4)

    # -- helpers -------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            raise DsmcError(f"dsmc error {rc}: {self.lib.dsmc_last_error(self._h).decode()}")

    def _ptr(self, a, dtype="float32"):
        """(pointer, where) for a numpy array (host) or torch CUDA tensor (device) of the ABI's element type."""
        torch = self._torch
        if isinstance(a, torch.Tensor):
            if not a.is_contiguous() or str(a.dtype) != "torch." + dtype:
                raise TypeError(f"expected a contiguous {dtype} tensor, got {a.dtype}")
            if a.is_cuda and a.device != self.device:
                raise ValueError(f"tensor on {a.device}, context on {self.device}")
            return a.data_ptr(), (DSMC_DEVICE if a.is_cuda else DSMC_HOST)
        if not (isinstance(a, np.ndarray) and a.flags.c_contiguous and a.dtype == np.dtype(dtype)):
            raise TypeError(f"expected a C-contiguous {dtype} array")
        return a.ctypes.data, DSMC_HOST

    def close(self):
        if self._h:
            self._torch.cuda.synchronize(self.device)
            self.lib.dsmc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the calls of include/dsmc.h -----------------------------------------------------------
    def set_anisotropy(self, K2, K4):
        k2 = np.empty(self.R, dtype=np.float32)
        k4 = np.empty(self.R, dtype=np.float32)
        k2[:] = K2
        k4[:] = K4
        self._check(self.lib.dsmc_set_anisotropy(self._h, k2.ctypes.data, k4.ctypes.data))

    def build_tensor(self, method=DSMC_W_EWALD, cutoff_A=64, tail=1):
        self._check(self.lib.dsmc_build_tensor(self._h, method, cutoff_A, tail))

    def get_tensor(self):
        W = np.empty((4, self.L, self.L), dtype=np.float32)
        self._check(self.lib.dsmc_get_tensor(self._h, W.ctypes.data, DSMC_HOST))
        return W

    def set_tensor(self, W):
        W = _np_f32(W, (4, self.L, self.L))
        self._check(self.lib.dsmc_set_tensor(self._h, W.ctypes.data, DSMC_HOST))

    def set_spins(self, s):
        if isinstance(s, np.ndarray):
            s = _np_f32(s, (self.R, 3, self.L, self.L))
        p, where = self._ptr(s)
        self._check(self.lib.dsmc_set_spins(self._h, p, where))

    def get_spins(self, out=None):
        if out is None:
            out = np.empty((self.R, 3, self.L, self.L), dtype=np.float32)
        p, where = self._ptr(out)
        self._check(self.lib.dsmc_get_spins(self._h, p, where))
        return out

    def init_spins(self, mode=DSMC_INIT_RANDOM, seed=0):
        self._check(self.lib.dsmc_init_spins(self._h, mode, seed))

    def dipole_field(self, colour=-1, out=None, want_output=True):
        if not want_output:
            self._check(self.lib.dsmc_dipole_field(self._h, colour, None, DSMC_HOST))
            return None
        if out is None:
            out = np.zeros((self.R, 3, self.L, self.L), dtype=np.float32)
        p, where = self._ptr(out)
        self._check(self.lib.dsmc_dipole_field(self._h, colour, p, where))
        return out

    def get_field(self, out=None):
        """The field array as kept in the context (no recomputation), canonical [R][3][L][L]."""
        if out is None:
            out = np.zeros((self.R, 3, self.L, self.L), dtype=np.float32)
        p, where = self._ptr(out)
        self._check(self.lib.dsmc_get_field(self._h, p, where))
        return out

    def _T(self, T):
        if T is None:
            return None, None
        t = np.empty(self.R, dtype=np.float32)
        t[:] = T
        return t, t.ctypes.data

    def halfsweep(self, T, seed, step, flags=0, accept_out=None, margin_out=None):
        t, tp = self._T(T)
        if flags == 0 and accept_out is None and margin_out is None:
            self._check(self.lib.dsmc_halfsweep(self._h, tp, seed, step))
            return
        ap = self._ptr(accept_out, "uint8")[0] if accept_out is not None else None
        mp = self._ptr(margin_out)[0] if margin_out is not None else None
        self._check(self.lib.dsmc_halfsweep_ex(self._h, tp, seed, step, flags, ap, mp))

    def run(self, T, seed, first_step, n_half, flags=0):
        t, tp = self._T(T)
        if flags == 0:
            self._check(self.lib.dsmc_run(self._h, tp, seed, first_step, n_half))
        else:
            self._check(self.lib.dsmc_run_ex(self._h, tp, seed, first_step, n_half, flags))

    def run_recorded(self, T, seed, first_step, n_records, every, flags=0):
        """n_records x [every sweeps, ensemble_add], one native call."""
        t, tp = self._T(T)
        self._check(self.lib.dsmc_run_recorded(self._h, tp, seed, first_step, n_records, every, flags))

    def sublattice_pass(self, T, seed, pass_index, l, flags=0, accept_out=None, margin_out=None):
        """One pass of the paper's stride-l schedule -> the offset (S_1, S_2)."""
        t, tp = self._T(T)
        ap = self._ptr(accept_out, "uint8")[0] if accept_out is not None else None
        mp = self._ptr(margin_out)[0] if margin_out is not None else None
        off = (ctypes.c_int * 2)()
        self._check(self.lib.dsmc_sublattice_pass(self._h, tp, seed, pass_index, l, flags, ap, mp, off))
        return int(off[0]), int(off[1])

    def sublattice_run(self, T, seed, first_pass, n_passes, l, flags=0, margin_log=None):
        t, tp = self._T(T)
        if margin_log is None:
            self._check(self.lib.dsmc_sublattice_run(self._h, tp, seed, first_pass, n_passes, l, flags))
        else:
            self._check(self.lib.dsmc_sublattice_run_ex(self._h, tp, seed, first_pass, n_passes, l, flags,
                                                        self._ptr(margin_log)[0]))

    def observables(self):
        out = np.empty((self.R, 4), dtype=np.float64)
        self._check(self.lib.dsmc_observables(self._h, out.ctypes.data))
        return out

    def wall_observables(self):
        """-> (counts int64 [R][6] = n_h^x, n_v^x, n_h^y, n_v^y, n_h^z, n_v^z; derived float64 [R][4] =
        wall density, O_x, O_y, O_z)  (eq. 14-15)"""
        counts = np.empty((self.R, 6), dtype=np.int64)
        derived = np.empty((self.R, 4), dtype=np.float64)
        self._check(self.lib.dsmc_wall_observables(self._h, counts.ctypes.data, derived.ctypes.data))
        return counts, derived

    def staggered_magnetisation(self):
        """-> float64 [R][3] = m_h, m_v, m_st of App. B"""
        out = np.empty((self.R, 3), dtype=np.float64)
        self._check(self.lib.dsmc_staggered_magnetisation(self._h, out.ctypes.data))
        return out

    def ensemble_reset(self):
        self._check(self.lib.dsmc_ensemble_reset(self._h))

    def ensemble_add(self):
        """Accumulate the current state's E/N, m_z, M_par, eta, wall density, O_x, O_y, O_z (asynchronous)."""
        self._check(self.lib.dsmc_ensemble_add(self._h))

    def ensemble_get(self):
        """-> (mean, var, se, n): [R][8] each; eq. 13 and eq. 18"""
        mean, var, se = (np.empty((self.R, 8), dtype=np.float64) for _ in range(3))
        n = ctypes.c_uint64(0)
        self._check(self.lib.dsmc_ensemble_get(self._h, mean.ctypes.data, var.ctypes.data, se.ctypes.data,
                                               ctypes.byref(n)))
        return mean, var, se, int(n.value)

    def set_debug(self, on=True):
        """Debug checks: set_spins verifies |s| = 1 to 1e-5 (DsmcError otherwise)."""
        self._check(self.lib.dsmc_set_debug(self._h, int(on)))

    def set_timing(self, on=True):
        self._check(self.lib.dsmc_set_timing(self._h, int(on)))

    def last_timing(self):
        out = np.empty(3, dtype=np.float32)
        self._check(self.lib.dsmc_last_timing(self._h, out.ctypes.data))
        return out

    def launch_count(self):
        return int(self.lib.dsmc_launch_count(self._h))

    def field_kernel_kind(self):
        return int(self.lib.dsmc_field_kernel_kind(self._h))

    def fp32_fma_peak(self):
        out = ctypes.c_double(0.0)
        self._check(self.lib.dsmc_fp32_fma_peak(self._h, ctypes.addressof(out)))
        return float(out.value)

    def stream_footprint(self, colour):
        """One launch that moves a Metropolis half-sweep's bytes without its arithmetic (roofline denominator)."""
        self._check(self.lib.dsmc_stream_footprint(self._h, int(colour)))

    def set_replica_offset(self, first_replica):
        """This context holds replicas first_replica ... of a larger ladder (bit-reproducible sharding)."""
        self._check(self.lib.dsmc_set_replica_offset(self._h, int(first_replica)))

    def fft_supported(self):
        return bool(self.lib.dsmc_field_kernel_supported(self._h, DSMC_FIELD_FFT))

    def select_field_kernel(self, kind):
        self._check(self.lib.dsmc_select_field_kernel(self._h, kind))
