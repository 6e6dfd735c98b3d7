"""Harness of the long-run 3-sigma tests (north_star: "Observables over long runs: agreement within 3 sigma";
SURVEY.md 8c parity protocol: means over the same sweep window from >= 8 independent seeds a side, sigma from
the across-seed scatter, eq. 13).

The oracle side of a long run is the oracle's own half-sweep and observables (oracle_halfsweep_given_field,
oracle_observables_given_field: Philox, trial move, dE, acceptance, eq. 11/16/17 are the oracle's) fed with a dipole
field this harness evaluates by fp64 FFT -- SURVEY.md 8c-O2 allows exactly that "to make long oracle runs
affordable"; the direct sum stays the definition, and tests/test_oracle_harness.py pins this FFT field to it.
Chains of different seeds are independent, so they run as child processes (one OpenMP thread each).

Test infrastructure only; nothing here is imported by the product.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

OBS_NAMES = ("E/N", "m_z", "M_par", "eta")


def spectral_table(W):
    """conj of the 2-D transform of W[4][L][L] (real input, half spectrum): h = W correlated with s."""
    import scipy.fft as sfft
    return np.conj(sfft.rfft2(np.asarray(W, dtype=np.float64), axes=(-2, -1)))


def fft_field_fp64(Mh, s):
    """h_n = sum_m W(m - n) s_m for s[R][3][L][L] (fp64) by FFT: x and y components mix through W^xy."""
    import scipy.fft as sfft
    sh = sfft.rfft2(s, axes=(-2, -1))
    hx = Mh[0] * sh[:, 0] + Mh[1] * sh[:, 1]
    hy = Mh[1] * sh[:, 0] + Mh[2] * sh[:, 1]
    hz = Mh[3] * sh[:, 2]
    return sfft.irfft2(np.stack([hx, hy, hz], axis=1), s=s.shape[-2:], axes=(-2, -1))


def oracle_chain(job):
    """One oracle chain of a BASELINE config as written: -> per-sweep observables [n_sweeps][R][4].
    job = (cfg_id, seed, n_sweeps)."""
    cfg_id, seed, n_sweeps = job
    from oracle import oracle as o
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    L, R, g = c["L"], c["R"], c["g"]
    K2, K4 = (a.astype(np.float64) for a in inputs.anisotropy(cfg_id))
    T = inputs.temperatures(cfg_id).astype(np.float64)
    W = o.build_tensor_ewald(L)
    Mh = spectral_table(W)
    s = initial_state(cfg_id, seed).astype(np.float64)
    rec = np.empty((n_sweeps, R, 4))
    h = fft_field_fp64(Mh, s)
    for sw in range(n_sweeps):
        o.halfsweep_given_field(W, s, h, T, seed, 2 * sw, 1.0, g, K2, K4)
        h = fft_field_fp64(Mh, s)
        o.halfsweep_given_field(W, s, h, T, seed, 2 * sw + 1, 1.0, g, K2, K4)
        h = fft_field_fp64(Mh, s)                 # serves the record and the next sweep's first half
        rec[sw] = o.observables_given_field(s, h, 1.0, g, K2, K4)
    return rec


def initial_state(cfg_id, seed):
    """The config's initial state: all +z (config 3), else iid uniform on S^2 drawn per seed."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    if c["init"] == "up":
        return inputs.up_spins(c["L"], c["R"])
    return inputs.random_spins(c["L"], c["R"], inputs.SEED_BASE + 7919 * cfg_id + seed)


class _Chains:
    """Oracle chains as child processes (`python longrun_harness.py cfg seed n out.npy`, one OpenMP thread each),
    at most `workers` at a time; get(job) waits for that chain and returns its record."""

    def __init__(self, jobs, workers):
        import concurrent.futures as cf
        import tempfile
        self.dir = tempfile.mkdtemp(prefix="dsmc_longrun_")
        self.procs = []
        self.stopped = False
        self.pool = cf.ThreadPoolExecutor(max_workers=workers)
        self.futures = {job: self.pool.submit(self._run, job) for job in jobs}

    def _run(self, job):
        import subprocess
        if self.stopped:
            return None
        cfg_id, seed, n_sweeps = job
        out = os.path.join(self.dir, f"c{cfg_id}_s{seed}_n{n_sweeps}.npy")
        env = dict(os.environ, OMP_NUM_THREADS="1")
        p = subprocess.Popen([sys.executable, os.path.abspath(__file__), str(cfg_id), str(seed), str(n_sweeps), out],
                             env=env, cwd=ROOT, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
        self.procs.append(p)
        log, _ = p.communicate()
        if p.returncode != 0:
            raise RuntimeError(f"oracle chain {job} failed ({p.returncode}): {log[-2000:]}")
        return np.load(out)

    def get(self, job, timeout=3000):
        return self.futures[job].result(timeout=timeout)

    def close(self):
        import shutil
        self.stopped = True
        for f in self.futures.values():
            f.cancel()
        for p in self.procs:
            if p.poll() is None:
                p.kill()                       # the exact children this object started
        self.pool.shutdown(wait=True)
        shutil.rmtree(self.dir, ignore_errors=True)


def start_oracle_chains(jobs, workers=None):
    """Start the chains in the background; -> object with get((cfg_id, seed, n_sweeps)) and close()."""
    n = workers or max(1, min(len(jobs), (os.cpu_count() or 2) - 1))
    return _Chains(list(jobs), n)


def gpu_chain(m, cfg_id, seed, n_sweeps, field_kind=None):
    """The CUDA path on the same config: dsmc_run sweep by sweep, dsmc_observables after every sweep."""
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[cfg_id]
    K2, K4 = inputs.anisotropy(cfg_id)
    T = inputs.temperatures(cfg_id)
    ctx = m.Dsmc(c["L"], c["R"], J=1.0, g=c["g"], K2=K2, K4=K4)
    ctx.build_tensor(m.DSMC_W_EWALD)
    if field_kind is not None:
        ctx.select_field_kernel(field_kind)
    ctx.set_spins(initial_state(cfg_id, seed))
    rec = np.empty((n_sweeps, c["R"], 4))
    for sw in range(n_sweeps):
        ctx.run(T if sw == 0 else None, seed, 2 * sw, 2)
        rec[sw] = ctx.observables()
    ctx.close()
    return rec


def window_mean(rec):
    """Mean over the second half of the run (the same sweep window on both sides)."""
    rec = np.asarray(rec)
    return rec[rec.shape[0] // 2:].mean(axis=0)


def z_scores(a, b):
    """a, b: [seed][R][4] window means of the two sides.  -> (z, diff, sigma): |difference of the across-seed
    means| in units of its standard error (eq. 13 with the across-seed scatter)."""
    a, b = np.asarray(a), np.asarray(b)
    diff = a.mean(0) - b.mean(0)
    sigma = np.sqrt(a.var(0, ddof=1) / a.shape[0] + b.var(0, ddof=1) / b.shape[0])
    # fp32 path against fp64 oracle: per-snapshot observables agree to 2e-6 (test_observables_parity), so a scatter
    # below that is not resolvable and must not blow z up
    return np.abs(diff) / np.maximum(sigma, 2e-6), diff, sigma


if __name__ == "__main__":
    cfg, seed, n, out = int(sys.argv[1]), int(sys.argv[2]), int(sys.argv[3]), sys.argv[4]
    np.save(out, oracle_chain((cfg, seed, n)))
