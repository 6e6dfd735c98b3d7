"""App. B of the paper on the GPU: the dipolar Ising model on L = 64 under the stride-l schedule.

  python -m paper_1211_6234_b200.appendix_b                       # l = 32 (the paper's choice) and l = 64
  python -m paper_1211_6234_b200.appendix_b --steps 20000 --l 32

PAPER.md:364-402: spins (0, 0, +-1), trial = complete reversal (DSMC_TRIAL_FLIP), eq. 19 with J / C_D = 1.7
(0.85 per bond in the build's convention, R22), order parameter m_st = <(m_h^2 + m_v^2)^(1/2)>
of the four sub-lattices (R23), chi_st = (L^2 / k_B T)(<m_st^2> - <m_st>^2), T_c from the peak of chi_st.
l = 32 updates n = 4 sites per pass with the simultaneous-flip approximation of section 3.2; l = L = 64
updates one random site per pass, i.e. conventional single-spin Metropolis with no approximation: the
pair of runs is the comparison of the paper's Table 1 (T_c = .85 "GPU algorithm" against .82
"conventional MC" from its ref. [66]).  Smaller strides (--l 16 8 4 2) make the approximation coarser
("the error will be increased for decreasing l"); --l 0 is the checkerboard half-sweep of
north_star (n = N/2 simultaneous sites, the coarsest use of the approximation).

Every pass, the sub-lattice sums of m_st included, runs in libdsmc.so (dsmc_sublattice_run with the lattice
resident in shared memory, dsmc_staggered_magnetisation); this script marshals arguments and averages the
per-snapshot m_st over the recorded states.  Temperatures are in units of C_D (g = 1).  Replica r has
temperature T[r // chains]: `chains` independent chains per temperature give the error bars.
"""
import argparse
import json
import time

import numpy as np


def scan(l, temps, chains, equilibrate, steps, seed, device="cuda"):
    """-> dict of arrays over temperatures: m_st, chi_st and their standard errors over the chains."""
    import torch
    from . import Dsmc, DSMC_W_EWALD, DSMC_TRIAL_FLIP, DSMC_FIELD_FFT
    L, g, J = 64, 1.0, 0.85
    nT = len(temps)
    R = nT * chains
    T = np.repeat(np.asarray(temps, dtype=np.float32) * g, chains)
    ctx = Dsmc(L, R, J=J, g=g, K2=0.0, K4=0.0, device=device)
    ctx.build_tensor(DSMC_W_EWALD)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, :, None]      # h = 1 stripes: the ground state
    ctx.set_spins(s)
    per_step = l * l if l else 2                                           # passes (half-sweeps) per MC step
    if l == 0:
        ctx.select_field_kernel(DSMC_FIELD_FFT)

    def advance(first_step, n_steps, Targ):
        if l:                                                              # stride-l passes (l = L: single-spin Metropolis)
            ctx.sublattice_run(Targ, seed, first_step * per_step, n_steps * per_step, l, flags=DSMC_TRIAL_FLIP)
        else:                                                              # checkerboard half-sweeps (north_star's schedule)
            ctx.run(Targ, seed, 2 * first_step, 2 * n_steps, flags=DSMC_TRIAL_FLIP)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    advance(0, equilibrate, T)
    s1 = np.zeros(R)
    s2 = np.zeros(R)
    for k in range(steps):
        advance(equilibrate + k, 1, None)
        m = ctx.staggered_magnetisation()[:, 2]
        s1 += m
        s2 += m * m
    wall = time.perf_counter() - t0
    ctx.close()
    mean = (s1 / steps).reshape(nT, chains)
    var = (s2 / steps).reshape(nT, chains) - mean ** 2
    chi = (L * L) * var / (np.asarray(temps, dtype=np.float64)[:, None] * g)
    se = lambda a: a.std(axis=1, ddof=1) / np.sqrt(chains) if chains > 1 else np.zeros(nT)
    return {"l": l, "T": np.asarray(temps, dtype=np.float64), "m_st": mean.mean(axis=1), "m_st_se": se(mean),
            "chi_st": chi.mean(axis=1), "chi_st_se": se(chi), "seconds": wall,
            "passes_per_s": (equilibrate + steps) * per_step / wall}


def energy_histograms(temps, chains, equilibrate, steps, seed, l=32, bins=60, device="cuda"):
    """Fig. 19: distribution of the energy per spin over the recorded states at a few temperatures
    near the transition.  -> (bin centres [nT][bins], normalised counts [nT][bins])."""
    import torch
    from . import Dsmc, DSMC_W_EWALD, DSMC_TRIAL_FLIP
    L, g, J = 64, 1.0, 0.85
    nT = len(temps)
    R = nT * chains
    T = np.repeat(np.asarray(temps, dtype=np.float32) * g, chains)
    ctx = Dsmc(L, R, J=J, g=g, K2=0.0, K4=0.0, device=device)
    ctx.build_tensor(DSMC_W_EWALD)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = np.where(np.arange(L) % 2 == 0, 1.0, -1.0)[None, :, None]
    ctx.set_spins(s)
    per_step = l * l
    ctx.sublattice_run(T, seed, 0, equilibrate * per_step, l, flags=DSMC_TRIAL_FLIP)
    E = np.empty((steps, R))
    for k in range(steps):
        ctx.sublattice_run(None, seed, (equilibrate + k) * per_step, per_step, l, flags=DSMC_TRIAL_FLIP)
        E[k] = ctx.observables()[:, 0]
    ctx.close()
    E = E.reshape(steps, nT, chains).transpose(1, 0, 2).reshape(nT, -1)
    centres, counts = np.empty((nT, bins)), np.empty((nT, bins))
    for i in range(nT):
        h, edges = np.histogram(E[i], bins=bins)
        centres[i], counts[i] = 0.5 * (edges[1:] + edges[:-1]), h / h.sum()
    return centres, counts


def count_modes(counts, smooth=5, floor=0.25):
    """Number of local maxima of a histogram after a moving average, ignoring bumps below `floor` of the highest."""
    c = np.convolve(counts, np.ones(smooth) / smooth, mode="same")
    peaks = [i for i in range(1, len(c) - 1) if c[i] > c[i - 1] and c[i] >= c[i + 1] and c[i] > floor * c.max()]
    return len(peaks)


def peak_temperature(T, chi):
    """Location of the maximum of chi_st: vertex of the parabola through the largest sample and its neighbours."""
    i = int(np.argmax(chi))
    if i == 0 or i == len(T) - 1:
        return float(T[i])
    x, y = T[i - 1:i + 2], chi[i - 1:i + 2]
    a, b, _ = np.polyfit(x, y, 2)
    return float(-b / (2.0 * a))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--l", type=int, nargs="*", default=[32, 64],
                    help="stride(s): 32 = the paper's, 64 = single-spin, any divisor of 64 >= 2; 0 = checkerboard half-sweeps")
    ap.add_argument("--tmin", type=float, default=0.50)
    ap.add_argument("--tmax", type=float, default=1.22)
    ap.add_argument("--nt", type=int, default=37)
    ap.add_argument("--chains", type=int, default=8)
    ap.add_argument("--equilibrate", type=int, default=2000, help="MC steps before recording")
    ap.add_argument("--steps", type=int, default=8000, help="recorded MC steps (one state per step)")
    ap.add_argument("--seed", type=int, default=0x1211B)
    ap.add_argument("--json", action="store_true")
    ap.add_argument("--energy-histograms", action="store_true",
                    help="Fig. 19 instead of the scan: energy distributions at script-T = .833, .85, .867, .884")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("appendix_b: no CUDA device (there is no CPU fallback)")
    if args.energy_histograms:
        script_T = np.array([0.833, 0.85, 0.867, 0.884])                 # PAPER.md:384 (Fig. 19); T / g = script-T / 2
        centres, counts = energy_histograms(script_T / 2.0, 74, args.equilibrate, args.steps, args.seed)
        for i, t in enumerate(script_T):
            print(f"script-T = {t:.3f}: <E/N> = {np.sum(centres[i] * counts[i]):.4f}, modes = {count_modes(counts[i])}")
            print("   E/N    " + " ".join(f"{x:7.3f}" for x in centres[i][::4]))
            print("   P      " + " ".join(f"{x:7.4f}" for x in counts[i][::4]))
        return
    temps = np.linspace(args.tmin, args.tmax, args.nt)
    results = [scan(l, temps, args.chains, args.equilibrate, args.steps, args.seed) for l in args.l]
    if args.json:
        print(json.dumps([{k: (v.tolist() if isinstance(v, np.ndarray) else v) for k, v in r.items()} for r in results]))
        return
    for r in results:
        n = (64 // r["l"]) ** 2 if r["l"] else 2048
        print(f"l = {r['l']} (n = {n} simultaneous sites): {args.equilibrate} + {args.steps} MC steps, {args.nt} temperatures x "
              f"{args.chains} chains in {r['seconds']:.1f} s ({r['passes_per_s']:.3e} passes/s); "
              f"T_c (peak of chi_st) = {peak_temperature(r['T'], r['chi_st']):.3f} C_D")
    print("   T/C_D " + "".join(f"   m_st(l={r['l']})      chi_st(l={r['l']})    " for r in results))
    for i, t in enumerate(temps):
        print(f"{t:8.3f} " + "".join(f"{r['m_st'][i]:8.4f}+-{r['m_st_se'][i]:6.4f} {r['chi_st'][i]:9.3f}+-{r['chi_st_se'][i]:7.3f}  "
                                      for r in results))


if __name__ == "__main__":
    main()
