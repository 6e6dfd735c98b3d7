"""Run one of BASELINE.json's five configurations on the GPU and print the ensemble statistics.

  python -m paper_1211_6234_b200.run_config 3 --field fft
  python -m paper_1211_6234_b200.run_config 2 --sweeps 2000 --record-every 1 --equilibrate 0
  python -m torch.distributed.run --nproc-per-node 8 --master-addr 127.0.0.1 -m paper_1211_6234_b200.run_config 5

Under torchrun the temperature ladder is split over the ranks (one GPU each, contiguous blocks of
replicas, no exchange inside the run: the chains are independent); rank 0 gathers the R x 8 results.

Everything runs in libdsmc.so (dsmc_run for the sweeps, dsmc_ensemble_add for the recorded states: no
host round trip inside the loop); this script only marshals arguments and formats the result.
The protocol is the paper's: equilibrate, then record a state every k sweeps and
report <X>, the standard error of eq. 13 and the variance of eq. 18 for each replica.
"""
import argparse
import json
import time

import numpy as np

NAMES = ["E/N", "m_z", "M_par", "eta", "wall_density", "O_x", "O_y", "O_z"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", type=int, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--field", choices=["auto", "fft", "direct"], default="auto",
                    help="auto = FFT when the shape allows it, else the direct sum")
    ap.add_argument("--sweeps", type=int, default=None, help="total sweeps (default: the configuration's)")
    ap.add_argument("--equilibrate", type=int, default=None, help="sweeps before recording (default: half)")
    ap.add_argument("--record-every", type=int, default=1)
    ap.add_argument("--json", action="store_true")
    args = ap.parse_args()

    import torch
    import torch.distributed as dist
    from . import Dsmc, DSMC_W_EWALD, DSMC_W_IMAGE, DSMC_FIELD_FFT, DSMC_FIELD_AUTO, DSMC_INIT_UP, inputs, multirank
    if not torch.cuda.is_available():
        raise SystemExit("run_config: no CUDA device (there is no CPU fallback)")
    rank, world, local = multirank.env()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = inputs.CONFIGS[args.config]
    L, R_all = c["L"], c["R"]
    lo, hi = multirank.replica_shard(R_all, world, rank)       # this rank's block of the ladder
    if hi == lo:
        raise SystemExit(f"run_config: {world} ranks for {R_all} replicas leaves rank {rank} without work")
    R = hi - lo
    K2, K4 = (a[lo:hi] for a in inputs.anisotropy(args.config))
    T = inputs.temperatures(args.config)[lo:hi]
    seed = inputs.SEED_BASE + args.config
    ctx = Dsmc(L, R, J=1.0, g=c["g"], K2=K2, K4=K4, device=torch.device("cuda", local))
    ctx.set_replica_offset(lo)                                 # same random streams as the unsharded ladder
    if args.config == 1:
        ctx.build_tensor(DSMC_W_IMAGE, 64, 1)               # BASELINE config 1: image cutoff |a|,|b| <= 64
    else:
        ctx.build_tensor(DSMC_W_EWALD)
    use_fft = args.field == "fft" or (args.field == "auto" and ctx.fft_supported())
    ctx.select_field_kernel(DSMC_FIELD_FFT if use_fft else DSMC_FIELD_AUTO)
    if c["init"] == "up":
        ctx.init_spins(DSMC_INIT_UP)
    else:
        ctx.set_spins(inputs.initial_spins(args.config)[lo:hi])
    sweeps = args.sweeps if args.sweeps is not None else c["sweeps"]
    burn = args.equilibrate if args.equilibrate is not None else sweeps // 2
    every = max(1, args.record_every)

    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ctx.run(T, seed, 0, 2 * burn)
    ctx.ensemble_reset()
    n_rec = (sweeps - burn) // every
    ctx.run_recorded(None, seed, 2 * burn, n_rec, every)       # n_rec x [every sweeps, record], one native call
    done = burn + n_rec * every
    if done < sweeps:                                          # a last, shorter interval
        ctx.run(None, seed, 2 * done, 2 * (sweeps - done))
        ctx.ensemble_add()
    mean, var, se, n = ctx.ensemble_get()                   # synchronises
    wall = time.perf_counter() - t0
    kind = ["generic", "tiled", "fft"][ctx.field_kernel_kind()]
    ctx.close()
    if world > 1:
        dev = torch.device("cuda", local)
        wall = multirank.max_over_ranks([wall], device=dev)[0]
        mean, var, se = (multirank.gather_replica_rows(a, R_all, device=dev) for a in (mean, var, se))
        T = multirank.gather_replica_rows(T.astype(np.float64), R_all, device=dev)
        K4 = multirank.gather_replica_rows(K4.astype(np.float64), R_all, device=dev)
        dist.destroy_process_group()
        if rank != 0:
            return
    R = R_all
    result = {
        "config": args.config, "L": L, "R": R, "n_gpus": world, "field_kernel": kind,
        "sweeps": sweeps, "equilibrate": burn, "recorded": n, "seconds": wall,
        "sweeps_per_s": sweeps / wall, "updates_per_s": sweeps * L * L * R / wall,
        "T": [float(t) for t in T], "K4": [float(k) for k in K4], "quantities": NAMES,
        "mean": mean.tolist(), "standard_error": se.tolist(), "variance": var.tolist(),
    }
    if args.json:
        print(json.dumps(result))
        return
    print(f"config {args.config}: L={L} R={R} field={result['field_kernel']} sweeps={sweeps} (recorded {n}) "
          f"in {wall:.2f} s = {result['sweeps_per_s']:.1f} sweeps/s = {result['updates_per_s']:.3e} updates/s")
    print("   T     K4   " + "".join(f"{q:>22s}" for q in NAMES[:5] + NAMES[7:]))
    for r in range(R):
        cols = [0, 1, 2, 3, 4, 7]
        cells = "".join(f"{mean[r, k]:13.5f} +-{se[r, k]:7.5f}" for k in cols)
        print(f"{T[r]:6.3f} {K4[r]:6.2f} {cells}")


if __name__ == "__main__":
    main()
