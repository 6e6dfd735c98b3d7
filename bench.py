#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on BASELINE.json's config 5 (L=256, R=64) on B200.

  python bench.py --gpus N --steps K --warmup W            # the CUDA path (one JSON line, rank 0)
  python bench.py --impl reference --steps K --warmup W     # the fp64 CPU oracle on host cores

One "step" = one Monte Carlo sweep of the whole hot path: for colour 0 then 1, dipole field
(a1) + fused Metropolis half-sweep (a2), on all R replicas.  value = spin updates per second
(N*R updates per step).  Multi-GPU: the path shards by replica with no exchange ("replicas only",
DESIGN.md section 7): every rank runs the full config-5 workload, weak scaling.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

CFG_ID = 5
WORKLOAD = ("config5 L=256 R=64 J=1 g=0.1 K2=0.6 K4=0.1 T=0.1..2.0, 1 step = 1 sweep "
            "(2 x [dipole field + Metropolis half-sweep])")
FLOP_PER_PAIR = 10.0           # 5 FMA per (target, source, replica): SURVEY.md section 8(d)
BYTES_PER_UPDATE = 48.0        # own spin 12 + neighbours 12 (amortised) + h 12 + write 12
# dram__bytes_read.sum + dram__bytes_write.sum per launch and gpu__time_duration from the committed `ncu --set full`
# captures of THIS round's kernels (profiles/r02_*.md name the commands).  They are constants of those captures, not
# quantities of this run: each is reported under a key that says so, next to the live CUDA-event figures.
NCU = {
    "field_tiled_kernel": {"profile": "profiles/r02_field_kernel.md", "dram_bytes": 329.7e6, "time_us": 22650.0},
    "metropolis4_kernel": {"profile": "profiles/r02_metropolis_kernel.md", "dram_bytes": 78.4e6, "time_us": 20.01},
    "fft_field_group": {"profile": "profiles/r02_fft_field_kernels.md", "dram_bytes": 105.2e6, "time_us": 52.1},
}
# fp32 FMA peak: 148 SMs x 128 lanes x 2 flop x 1.965 GHz
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [t.strip() for t in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(steps, warmup, n_rep):
    """The oracle, as it stands, on a bounded sample of config 5: one half-sweep (field for the active
    colour + Metropolis decisions) restricted to n_rep of the 64 replicas.  -> (updates/s, seconds/step)"""
    from oracle import oracle as o
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[CFG_ID]
    L = c["L"]
    K2, K4 = inputs.anisotropy(CFG_ID)
    T = inputs.temperatures(CFG_ID)
    W = o.build_tensor_ewald(L)
    s = inputs.initial_spins(CFG_ID)[:n_rep].astype(np.float64)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        o.halfsweep(W, s, T[:n_rep].astype(np.float64), inputs.SEED_BASE + CFG_ID, it, 1.0, c["g"],
                    K2[:n_rep].astype(np.float64), K4[:n_rep].astype(np.float64), want=())
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    sec = float(np.mean(times))
    updates = (L * L // 2) * n_rep
    return updates / sec, sec, o.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1211_6234_b200 import inputs
    c = inputs.CONFIGS[CFG_ID]
    n_rep = 2
    ups, sec, cores = oracle_sample(args.steps, min(args.warmup, 1), n_rep)
    sample = (f"one checkerboard half-sweep (field of the active colour + Metropolis) of config 5 restricted to "
              f"{n_rep} of {c['R']} replicas per step (work is linear in R)")
    line = {
        "impl": "reference", "metric": "spin_updates_per_s", "value": ups, "unit": "updates/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "L": c["L"], "R": c["R"], "parallelism": "host cores, rank 0 only",
                   "sample": f"each step = one half-sweep on {n_rep} of {c['R']} replicas"},
        "cpu_baseline": {"value": ups, "unit": "updates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": ups, "unit": "updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def metropolis_roofline(nbytes, in_sweep_ms, b2b_ms, n_b2b, hbm_peak, hbm_kind, updates, stream_ms):
    """The Metropolis kernel against HBM bandwidth by every timing there is: `frac` is the
    conservative one -- algorithmic bytes over the CUDA-event time of the launch where it really runs, inside a sweep,
    which includes the exposed launch latency (the event between the field kernel and this launch rules out the
    dependent-launch overlap the production path has)."""
    ncu = NCU["metropolis4_kernel"]

    def both(gbs):
        return {"GB/s": gbs, "of_measured_hbm": gbs / hbm_peak, "of_8TBs": gbs / 8000.0}
    in_sweep = nbytes / (in_sweep_ms * 1e-3) / 1e9
    b2b = nbytes / (b2b_ms * 1e-3) / 1e9
    return {"kernel": "metropolis4_kernel", "bound": "hbm", "achieved": in_sweep, "peak": hbm_peak, "unit": "GB/s",
            "frac": in_sweep / hbm_peak, "peak_kind": hbm_kind, "frac_of_8TBs": in_sweep / 8000.0,
            "timing": "algorithmic bytes / mean CUDA-event time of the launch inside a direct-sum sweep",
            "ms_per_launch_in_sweep": in_sweep_ms, "bytes_per_launch": nbytes,
            "back_to_back": dict(both(b2b), ms_per_launch=b2b_ms, launches_timed=n_b2b,
                                 what="24 dependent launches over 3 contexts (300 MB: every launch finds its data "
                                      "evicted from L2), one event pair around the batch"),
            "stream_same_footprint": dict(both(nbytes / (stream_ms * 1e-3) / 1e9), ms_per_launch=stream_ms,
                                          metropolis_over_stream=stream_ms / b2b_ms,
                                          what="dsmc_stream_footprint in the same rotation: the Metropolis kernel's grid, "
                                               "loads and addresses, every thread's spins written back, no arithmetic -- "
                                               "what the memory system delivers for this footprint"),
            "ncu": dict(algorithmic_bytes_over_ncu_time=both(nbytes / (ncu["time_us"] * 1e-6) / 1e9),
                        dram_bytes_over_ncu_time=both(ncu["dram_bytes"] / (ncu["time_us"] * 1e-6) / 1e9),
                        gpu__time_duration_us=ncu["time_us"], dram_bytes=ncu["dram_bytes"], profile=ncu["profile"],
                        what="constants of the committed capture (cold L2, serialised launch), not of this run"),
            "updates_per_s_in_sweep": updates / (in_sweep_ms * 1e-3), "updates_per_s_back_to_back": updates / (b2b_ms * 1e-3),
            "traffic": ncu["dram_bytes"], "traffic_from": ncu["profile"]}


def paper_schedule(m, inputs, dev):
    """The paper's own update schedule at its own size (L = 64, l = 32, J/C_D = 8.9, K/C_D = 15,
    a = 0 -> J = 1, g = 2/8.9 = 0.2247, K2 = 1.685, R7): stride-l passes of n = 4 simultaneous sites, one MC
    step = l*l = 1024 passes.  Timed through dsmc_sublattice_run with the lattice resident in shared memory (one CTA
    per replica pair, one kernel for the whole run) and, for comparison, through the two-launches-per-pass path."""
    import torch
    L, out = 64, {}
    # T = 0.2 ... 1.6 is the ladder of the BASELINE configs; "cold" = script-T 0.2 ... 2 of the paper's production run
    # (T = script-T g / 2, R7), where few moves are accepted and the incremental field update pays
    for name, R, l, flags, Trange in (("resident", 16, 32, 0, (0.2, 1.6)), ("resident_R296", 296, 32, 0, (0.2, 1.6)),
                                      ("resident_l16_R296", 296, 16, 0, (0.2, 1.6)),
                                      ("resident_cold", 16, 32, 0, (0.022, 0.22)),
                                      ("incremental", 16, 32, m.DSMC_INCREMENTAL, (0.2, 1.6)),
                                      ("incremental_cold", 16, 32, m.DSMC_INCREMENTAL, (0.022, 0.22)),
                                      ("incremental_cold_R296", 296, 32, m.DSMC_INCREMENTAL, (0.022, 0.22)),
                                      ("two_launch_graph", 16, 32, m.DSMC_NO_RESIDENT, (0.2, 1.6))):
        npass = l * l
        ctx = m.Dsmc(L, R, J=1.0, g=0.2247, K2=1.685, K4=0.0, device=dev)
        ctx.build_tensor(m.DSMC_W_EWALD)
        ctx.set_spins(inputs.random_spins(L, R, 1))
        T = np.linspace(Trange[0], Trange[1], R).astype(np.float32)
        # equilibrate first (the acceptance rate of the quench from a random state is not the ladder's)
        ctx.sublattice_run(T, 1, 0, 40 * npass, l, flags=flags & ~m.DSMC_INCREMENTAL)
        ctx.sublattice_run(T, 1, 40 * npass, npass, l, flags=flags)
        torch.cuda.synchronize(dev)
        reps = 4
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.sublattice_run(None, 1, 41 * npass, reps * npass, l, flags=flags)
        e1.record()
        torch.cuda.synchronize(dev)
        ms = e0.elapsed_time(e1) / reps
        out[name] = {"R": R, "l": l, "T": list(Trange), "us_per_pass": ms * 1e3 / npass, "ms_per_mc_step": ms,
                     "updates_per_s": L * L * R / (ms * 1e-3)}
        if flags & m.DSMC_INCREMENTAL:                            # the acceptance rate the timing goes with
            log = torch.zeros((npass, R, (L // l) ** 2), dtype=torch.float32, device=dev)
            ctx.sublattice_run(None, 1, 45 * npass, npass, l, flags=flags, margin_log=log)
            acc = (log < 0).float().mean(dim=(0, 2)).cpu().numpy()
            out[name]["acceptance_coldest_hottest"] = [float(acc[0]), float(acc[-1])]
        ctx.close()
    # resident kernel: one CTA = one SM sums 4 targets x 4096 sources x 5 FMA x 2 replicas per pass
    fma_clk = 4 * L * L * 5 * 2 / 128.0
    out["workload"] = "L=64 l=32 (n=4 sites per pass, 1024 passes per MC step), J=1 g=0.2247 K2=1.685 K4=0, T=0.2..1.6"
    out["resident_fma_bound_us_per_pass"] = fma_clk / 1965.0
    out["resident_frac_of_sm_fma_peak"] = (fma_clk / 1965.0) / out["resident"]["us_per_pass"]
    return out


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_1211_6234_b200 import multirank
    rank, world, local = multirank.env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the dsmc path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    import paper_1211_6234_b200 as m
    from paper_1211_6234_b200 import build, inputs
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()

    c = inputs.CONFIGS[CFG_ID]
    L, R = c["L"], c["R"]
    N = L * L
    K2, K4 = inputs.anisotropy(CFG_ID)
    T = inputs.temperatures(CFG_ID)
    seed = inputs.SEED_BASE + CFG_ID                  # one seed for the job; the ranks' chains differ in the replica index
    ctx = m.Dsmc(L, R, J=1.0, g=c["g"], K2=K2, K4=K4, device=dev)
    ctx.set_replica_offset(multirank.rank_replica_offset(R, rank))
    ctx.build_tensor(m.DSMC_W_EWALD)
    s_host = torch.from_numpy(inputs.random_spins(L, R, seed + rank)).pin_memory()
    ctx.set_spins(s_host.numpy())
    out_host = torch.empty_like(s_host).pin_memory()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def sweep(k):
        ctx.halfsweep(T, seed, 2 * k)
        ctx.halfsweep(None, seed, 2 * k + 1)

    # ---- whole-path throughput, inputs resident in HBM ---------------------------------------------
    for k in range(args.warmup):
        sweep(k)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(args.steps):
        sweep(args.warmup + k)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0

    # ---- per-kernel device times on the launching stream (CUDA events inside the library) ----------
    ctx.set_timing(True)
    f_ms, m_ms = [], []
    for k in range(max(args.steps, 3)):
        for h in (0, 1):
            ctx.halfsweep(None, seed, 2 * (args.warmup + args.steps + k) + h)
            t = ctx.last_timing()
            f_ms.append(float(t[0]))
            m_ms.append(float(t[1]))
    ctx.set_timing(False)
    clocks = sampler.stop() if sampler else None

    # ---- the same sweep with the FFT route of the field, reported beside ------
    fft = None
    if ctx.fft_supported():
        ctx.select_field_kernel(m.DSMC_FIELD_FFT)
        base = 4 * (args.warmup + 2 * args.steps + 8)
        for k in range(args.warmup):
            sweep(base + k)
        torch.cuda.synchronize(dev)
        n_fft = max(50, args.steps)
        l0f = ctx.launch_count()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctx.dipole_field(0, want_output=False)            # the host gets ahead of the GPU (short kernels)
        f0.record()
        for k in range(n_fft):
            sweep(base + args.warmup + k)
        f1.record()
        torch.cuda.synchronize(dev)
        fft_ms = f0.elapsed_time(f1) / n_fft
        fft_launches = (ctx.launch_count() - l0f - 3) / n_fft
        # the same sweeps through dsmc_run, the call a user makes for a long run: replayed CUDA graphs, the groups of
        # 16 replicas as independent chains of launches
        n_run = max(200, args.steps)
        first = 2 * (base + args.warmup + n_fft)
        ctx.run(None, seed, first, 2 * n_run)                 # captures the graphs
        first += 2 * n_run
        torch.cuda.synchronize(dev)
        l0r = ctx.launch_count()
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        ctx.run(None, seed, first, 2 * n_run)
        r1.record()
        torch.cuda.synchronize(dev)
        run_ms = r0.elapsed_time(r1) / n_run
        run_launches = (ctx.launch_count() - l0r) / n_run
        ctx.set_timing(True)
        ff, fm = [], []
        for k in range(20):
            ctx.halfsweep(None, seed, 2 * (base + args.warmup + n_fft) + k)
            tt = ctx.last_timing()
            ff.append(float(tt[0]))
            fm.append(float(tt[1]))
        ctx.set_timing(False)
        # end to end with HOST buffers, as the e2e key of the main line
        def fft_e2e_step(k):
            ctx.set_spins(s_host.numpy())
            sweep(k)
            ctx.get_spins(out_host.numpy())
        fft_e2e_step(0)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for k in range(5):
            fft_e2e_step(k)
        torch.cuda.synchronize(dev)
        fft_e2e_s = (time.perf_counter() - t0) / 5
        ctx.select_field_kernel(m.DSMC_FIELD_AUTO)
        fft = {"e2e_s": fft_e2e_s, "ms_per_step": fft_ms, "field_ms_per_launch_group": float(np.mean(ff)),
               "metropolis_ms_in_sweep": float(np.mean(fm)), "launches_per_step": fft_launches,
               "run_ms_per_step": run_ms, "run_launches_per_step": run_launches, "run_steps": n_run}

    # Metropolis kernel alone with a working set larger than L2: three independent contexts are
    # updated in rotation, so the ~100 MB a launch touches were evicted by the ~200 MB the two
    # launches in between touched.  One event pair brackets the whole batch (no per-launch gaps).
    others = []
    Wdev = ctx.get_tensor()
    for j in range(2):
        cj = m.Dsmc(L, R, J=1.0, g=c["g"], K2=K2, K4=K4, device=dev)
        cj.set_replica_offset(multirank.rank_replica_offset(R, rank))
        cj.set_tensor(Wdev)
        cj.set_spins(inputs.random_spins(L, R, seed + 17 + j))
        others.append(cj)
    ring = [ctx] + others
    for cj in ring:
        cj.dipole_field(-1, want_output=False)
        cj.halfsweep(T, seed, 20_000, flags=m.DSMC_REUSE_FIELD)
        cj.halfsweep(None, seed, 20_001, flags=m.DSMC_REUSE_FIELD)
    torch.cuda.synchronize(dev)
    rounds = 8
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # a 22 ms field launch goes first so that the host has enqueued every Metropolis launch before
    # the first one starts: the batch is then paced by the GPU, not by the host's launch rate
    ring[0].dipole_field(1, want_output=False)
    m0.record()
    for k in range(rounds):
        for cj in ring:
            cj.halfsweep(None, seed, 30_000 + k, flags=m.DSMC_REUSE_FIELD)
    m1.record()
    torch.cuda.synchronize(dev)
    metro_cold_ms = m0.elapsed_time(m1) / (rounds * len(ring))
    launches_metro = rounds * len(ring)
    # the same rotation with the kernel that moves a half-sweep's bytes without its arithmetic (dsmc_stream_footprint):
    # what the memory system delivers for this footprint, grid and access pattern -- the measured denominator
    ring[0].dipole_field(1, want_output=False)
    m0.record()
    for k in range(rounds):
        for cj in ring:
            cj.stream_footprint(1)
    m1.record()
    torch.cuda.synchronize(dev)
    stream_ms = m0.elapsed_time(m1) / (rounds * len(ring))
    for cj in others:
        cj.close()
    del others, ring

    # ---- end to end through the public API with HOST buffers ----------------------------------------
    def e2e_step(k):
        ctx.set_spins(s_host.numpy())                 # H2D from pinned memory
        sweep(k)
        ctx.get_spins(out_host.numpy())               # D2H of the step's result (synchronises)
    e2e_step(0)
    barrier()
    t0 = time.perf_counter()
    n_e2e = max(2, min(args.steps, 5))
    for k in range(n_e2e):
        e2e_step(k)
    barrier()
    e2e_serial_s = (time.perf_counter() - t0) / n_e2e

    # The same steps double-buffered over two contexts on two streams (two independent batches in flight): every step
    # still uploads its inputs from pinned host memory and downloads its result through the C ABI, but one context's
    # copies run under the other's sweep.  Steps per timed iteration: 2.
    sa, sb = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    pair = []
    for st in (sa, sb):
        cj = m.Dsmc(L, R, J=1.0, g=c["g"], K2=K2, K4=K4, device=dev, stream=st)
        cj.set_replica_offset(multirank.rank_replica_offset(R, rank))
        cj.set_tensor(Wdev)
        pair.append((cj, torch.empty_like(s_host).pin_memory()))

    def launch_step(cj, k):
        cj.set_spins(s_host.numpy())                  # H2D from pinned memory (asynchronous on the context's stream)
        cj.halfsweep(T, seed, 2 * k)
        cj.halfsweep(None, seed, 2 * k + 1)

    (ca, outa), (cb, outb) = pair
    launch_step(ca, 0)
    launch_step(cb, 0)
    ca.get_spins(outa.numpy())
    cb.get_spins(outb.numpy())                        # warm: both contexts configured, buffers touched
    barrier()
    t0 = time.perf_counter()
    launch_step(ca, 0)
    n_pairs = max(4, n_e2e // 2)
    for k in range(n_pairs):
        launch_step(cb, 2 * k + 1)
        ca.get_spins(outa.numpy())                    # D2H of step 2k (waits for it only)
        if k + 1 < n_pairs:
            launch_step(ca, 2 * k + 2)
        cb.get_spins(outb.numpy())
    barrier()
    e2e_s = (time.perf_counter() - t0) / (2 * n_pairs)
    e2e_step(2 * (n_pairs - 1))                       # the same step through the serial route: identical result
    pipelined_matches = bool(torch.equal(outa, out_host))
    for cj, _ in pair:
        cj.close()
    del pair

    # ---- max over ranks ----------------------------------------------------------------------------
    ms, e2e_s, e2e_serial_s = multirank.max_over_ranks([ms, e2e_s, e2e_serial_s], device=dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    updates_per_step = N * R
    ms_per_step = ms / args.steps
    value = multirank.whole_job_rate(updates_per_step, world, ms_per_step * 1e-3)
    field_ms = float(np.mean(f_ms))
    metro_ms = float(np.mean(m_ms))
    flop_per_field = FLOP_PER_PAIR * (N // 2) * N * R
    field_tflops = flop_per_field / (field_ms * 1e-3) / 1e12
    hbm_peak, hbm_kind = measured_peaks()
    ffma_peak = ctx.fp32_fma_peak()            # dependency-free FFMA chains, same process, same clocks
    metro_bytes = BYTES_PER_UPDATE * (N // 2) * R
    metro_gbs = metro_bytes / (metro_cold_ms * 1e-3) / 1e9

    line = {
        "metric": "spin_updates_per_s", "value": value, "unit": "updates/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "L": L, "R": R, "parallelism": f"replicas only x{world}",
                   "l2": "working set per step (spins 50 MB + h 25 MB + split-K partials 201 MB) exceeds the 126 MB L2; "
                         "the Metropolis-only figure rotates over 3 contexts (300 MB) so every launch starts with its data evicted from L2",
                   "field_kernel": "tiled" if ctx.field_kernel_kind() == 1 else "generic"},
        "clocks": clocks,
        "e2e": {"value": world * updates_per_step / e2e_s, "unit": "updates/s",
                "h2d_bytes_per_step": int(s_host.numel() * 4), "d2h_bytes_per_step": int(out_host.numel() * 4),
                "mode": "double-buffered: two contexts on two streams, a step's copies (dsmc_set_spins / dsmc_get_spins with "
                        "HOST pointers, pinned memory) run under the other context's sweep",
                "equals_serial_result": pipelined_matches,
                "serial": {"value": world * updates_per_step / e2e_serial_s, "unit": "updates/s",
                           "what": "one context: upload, sweep, download, one after the other"}},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "field_tiled_kernel (+ reduce_partials)", "bound": "alu", "achieved": field_tflops,
                     "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": field_tflops / FP32_PEAK_TFLOPS,
                     "peak_kind": "derived: 148 SM x 128 fp32 lanes x 2 x 1.965 GHz (DESIGN.md section 6)",
                     "measured_ffma_peak": ffma_peak, "frac_of_measured_ffma_peak": field_tflops / ffma_peak,
                     "traffic": NCU["field_tiled_kernel"]["dram_bytes"], "traffic_from": NCU["field_tiled_kernel"]["profile"],
                     "ms_per_launch": field_ms, "flop_per_launch": flop_per_field},
        "dipole_field_gflops": field_tflops * 1e3,
        "roofline_metropolis": metropolis_roofline(metro_bytes, metro_ms, metro_cold_ms, launches_metro, hbm_peak, hbm_kind,
                                                   (N // 2) * R, stream_ms),
    }
    if fft is not None:
        # algorithmic HBM bytes of one half-sweep field by FFT: read every spin (12 B per site and replica),
        # write h of the active colour (12 B per active site and replica); the spectrum scratch is overhead
        fft_bytes = 12.0 * N * R + 12.0 * (N // 2) * R
        gbs = fft_bytes / (fft["field_ms_per_launch_group"] * 1e-3) / 1e9
        line["fft_path"] = {
            "what": "the same sweep with dsmc_select_field_kernel(DSMC_FIELD_FFT): the field as a batched 2-D FFT "
                    "convolution over replica pairs on checkerboard half-spectra (3 half-size kernels, the unchanged "
                    "colour's spectrum cached), same parity tolerances; not the path 'value' times",
            "metropolis_ms_in_sweep": fft["metropolis_ms_in_sweep"],
            "value": world * updates_per_step / (fft["run_ms_per_step"] * 1e-3), "unit": "updates/s",
            "ms_per_step": fft["run_ms_per_step"], "gpu_launches_per_step": fft["run_launches_per_step"],
            "timed": f"one dsmc_run call of {fft['run_steps']} sweeps (replayed graphs; the groups of 16 replicas as "
                     "independent chains of launches on a block-major copy of the spins, the copies in and out included)",
            "halfsweep_calls": {"ms_per_step": fft["ms_per_step"], "gpu_launches_per_step": fft["launches_per_step"],
                                "what": "the same sweeps as two dsmc_halfsweep calls each (one chain, no graph)"},
            "speedup_vs_direct_sum": ms_per_step / fft["run_ms_per_step"],
            "e2e": {"value": world * updates_per_step / fft["e2e_s"], "unit": "updates/s",
                    "h2d_bytes_per_step": int(s_host.numel() * 4), "d2h_bytes_per_step": int(out_host.numel() * 4)},
            "sweep_roofline": {
                "what": "the whole sweep of this path (field and decision fused) against the bytes a sweep must move: per "
                        "half-sweep read every spin (12 B x N x R) and write the updated colour (12 B x N/2 x R)",
                "bound": "hbm", "bytes_per_step": 2 * fft_bytes, "unit": "GB/s", "peak": hbm_peak, "peak_kind": hbm_kind,
                "achieved": 2 * fft_bytes / (fft["run_ms_per_step"] * 1e-3) / 1e9,
                "frac": 2 * fft_bytes / (fft["run_ms_per_step"] * 1e-3) / 1e9 / hbm_peak},
            "roofline": {"kernel": "fftc_x_forward + fftc_y + fftc_x_inverse", "bound": "hbm", "achieved": gbs,
                         "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "peak_kind": hbm_kind,
                         "ms_per_launch_group": fft["field_ms_per_launch_group"], "bytes_per_launch_group": fft_bytes,
                         "traffic": NCU["fft_field_group"]["dram_bytes"], "traffic_from": NCU["fft_field_group"]["profile"]}}
    line["paper_schedule"] = paper_schedule(m, inputs, dev)
    if world == 1 and not args.no_cpu_baseline:
        ups, sec, cores = oracle_sample(1, 0, 24)
        line["cpu_baseline"] = {"value": ups, "unit": "updates/s", "cores": cores, "kind": "oracle",
                                "sample": "one checkerboard half-sweep of config 5 on 24 of 64 replicas "
                                          f"({sec:.1f} s; work is linear in R)"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
