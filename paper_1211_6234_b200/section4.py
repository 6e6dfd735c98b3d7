"""Section 4 of the paper on the GPU: the Heisenberg production run with second and fourth order anisotropy.

  python -m paper_1211_6234_b200.section4                                  # shortened protocol, about a minute
  python -m paper_1211_6234_b200.section4 --equilibrate 100000 --steps 50000   # the paper's protocol

PAPER.md:173-175: L = 64, l = 32 (n = 4 simultaneous sites per pass, 1024 passes per MC step), script-J = J / C_D = 8.9
(stripe width 8), script-K = 15, a in {-1, 0, 2} (eq. 12), perpendicular striped start, 10^5 MC steps of
equilibration, then 5 x 10^4 steps with the state recorded every 50 (n = 1000), script-T = k_B T / C_D from 0.2 to 10.
Map to the build (R7; the paper's C_D is g / 2): J = 1, g = 2 / 8.9, K2 = 7.5 g (1 - a), K4 = 7.5 g a,
T = script-T g / 2.  Reported per (a, script-T): wall density (n_h + n_v) / 4N (eq. 14, Fig. 10), O_z (eq. 15,
Fig. 11), eta (eq. 17, Fig. 12), M_par (eq. 16, Fig. 13) and their variances (eq. 18, Figs. 14-16), each the mean
over `chains` independent chains.

All replicas (3 anisotropies x temperatures x chains) run side by side: the passes in
sublattice_resident_kernel (one CTA per replica pair), the recorded states reduced on the device by
dsmc_ensemble_add.  This script marshals arguments and formats the result.
"""
import argparse
import json
import time

import numpy as np

A_VALUES = (-1.0, 0.0, 2.0)
NAMES = ["E/N", "m_z", "M_par", "eta", "wall_density", "O_x", "O_y", "O_z"]


def run(temps, chains, equilibrate, steps, every, seed, device="cuda", schedule="stride", stride=32):
    """schedule: "stride" = stride-l passes (l = `stride`; the paper's l = 32 has n = 4 simultaneous sites), "single" = l = L = 64 (one site per
    pass, no approximation), "checkerboard" = north_star's half-sweeps (n = N/2 simultaneous sites, FFT field)."""
    import torch
    from . import Dsmc, DSMC_W_EWALD, DSMC_FIELD_FFT
    L, l = 64, stride
    g = 2.0 / 8.9
    K = 7.5 * g
    nT = len(temps)
    R = len(A_VALUES) * nT * chains
    a = np.repeat(np.asarray(A_VALUES), nT * chains)
    T = np.tile(np.repeat(np.asarray(temps, dtype=np.float64) * g / 2.0, chains), len(A_VALUES)).astype(np.float32)
    ctx = Dsmc(L, R, J=1.0, g=g, K2=(K * (1.0 - a)).astype(np.float32), K4=(K * a).astype(np.float32), device=device)
    ctx.build_tensor(DSMC_W_EWALD)
    s = np.zeros((R, 3, L, L), dtype=np.float32)
    s[:, 2] = np.where((np.arange(L) // 8) % 2 == 0, 1.0, -1.0)[None, None, :]     # perpendicular stripes of width 8
    ctx.set_spins(s)
    if schedule == "single":
        l = L
    per_step = l * l
    if schedule == "checkerboard":
        ctx.select_field_kernel(DSMC_FIELD_FFT)

    def advance(first_step, n_steps, Targ):
        if schedule == "checkerboard":
            ctx.run(Targ, seed, 2 * first_step, 2 * n_steps)
        else:
            ctx.sublattice_run(Targ, seed, first_step * per_step, n_steps * per_step, l)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    advance(0, equilibrate, T)
    ctx.ensemble_reset()
    done = 0
    while done < steps:
        k = min(every, steps - done)
        advance(equilibrate + done, k, None)
        done += k
        ctx.ensemble_add()
    mean, var, se, n = ctx.ensemble_get()
    wall = time.perf_counter() - t0
    ctx.close()
    shape = (len(A_VALUES), nT, chains, 8)
    return {"T": np.asarray(temps, dtype=np.float64), "mean": mean.reshape(shape).mean(axis=2),
            "variance": var.reshape(shape).mean(axis=2), "standard_error": se.reshape(shape).mean(axis=2),
            "recorded": n, "seconds": wall, "replicas": R, "mc_steps": equilibrate + steps}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--tmin", type=float, default=0.25)
    ap.add_argument("--tmax", type=float, default=10.0)
    ap.add_argument("--nt", type=int, default=40)
    ap.add_argument("--chains", type=int, default=2)
    ap.add_argument("--equilibrate", type=int, default=20000, help="MC steps before recording (paper: 100000)")
    ap.add_argument("--steps", type=int, default=10000, help="MC steps of the recorded part (paper: 50000)")
    ap.add_argument("--every", type=int, default=50, help="record a state every this many MC steps (paper: 50)")
    ap.add_argument("--seed", type=int, default=0x5EC4)
    ap.add_argument("--schedule", choices=["stride", "single", "checkerboard"], default="stride")
    ap.add_argument("--stride", type=int, default=32, help="l of the stride schedule (divides 64; the paper: 32)")
    ap.add_argument("--json", action="store_true")
    args = ap.parse_args()
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("section4: no CUDA device (there is no CPU fallback)")
    temps = np.linspace(args.tmin, args.tmax, args.nt)
    r = run(temps, args.chains, args.equilibrate, args.steps, args.every, args.seed, schedule=args.schedule, stride=args.stride)
    if args.json:
        print(json.dumps({k: (v.tolist() if isinstance(v, np.ndarray) else v) for k, v in r.items()}))
        return
    print(f"L=64 schedule={args.schedule}{args.stride if args.schedule == 'stride' else ''} script-J=8.9 script-K=15: {r['replicas']} replicas (3 a x {args.nt} script-T x {args.chains} chains), "
          f"{args.equilibrate} + {args.steps} MC steps, {r['recorded']} states recorded, {r['seconds']:.1f} s "
          f"({r['mc_steps'] / r['seconds']:.3e} MC steps/s)")
    cols = [4, 7, 3, 2]                                                   # wall density, O_z, eta, M_par
    for ia, a in enumerate(A_VALUES):
        print(f"\na = {a:+.0f}   script-T   wall_density      O_z              eta              M_par          "
              f"var(M_par)   var(eta)     var(O_z)")
        for it, t in enumerate(temps):
            cells = "".join(f"{r['mean'][ia, it, k]:9.4f}+-{r['standard_error'][ia, it, k]:6.4f}" for k in cols)
            v = r["variance"][ia, it]
            print(f"        {t:8.3f} {cells}   {v[2]:10.3e} {v[3]:10.3e} {v[7]:10.3e}")


if __name__ == "__main__":
    main()
