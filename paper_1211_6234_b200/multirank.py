"""Host-side bookkeeping of the multi-GPU run ("replicas only").

The path shards by replica with no data-path collective: every rank runs its own chains (one seed for the job,
disjoint replica indices in the Philox counter: dsmc_set_replica_offset),
and the only exchange is one MAX all-reduce of the ranks' device timings, so that the reported time is
the slowest rank's.  torch.distributed is plumbing here (NCCL on GPUs, gloo in the CPU tests)."""
import os


def env():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def rank_seed(seed, rank):
    """A Philox key per rank that cannot collide with another rank's for any pair of base seeds below 2^32: the
    rank goes in the high word of the 64-bit seed (key word 1), the base seed stays in the low word.  (The
    library's own mechanism for one job is dsmc_set_replica_offset -- one seed, disjoint replica indices in the
    counter -- which is what bench.py and run_config use; this is for jobs that want distinct keys.)"""
    return (int(seed) & 0xFFFFFFFF) | ((int(rank) + 1) << 32)


def rank_replica_offset(R_per_rank, rank):
    """First global replica index of `rank` when every rank runs R_per_rank replicas of one job under one seed."""
    return int(rank) * int(R_per_rank)


def replica_shard(R, world, rank):
    """Contiguous block of the R replicas owned by `rank` when ONE ladder is split over the ranks
    (strong scaling); blocks differ by at most one replica."""
    base, extra = divmod(int(R), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(values, device="cpu"):
    """Element-wise maximum of a list of floats over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_rate(units_per_rank_step, world, seconds_per_step):
    """Aggregate throughput of `world` ranks that each process units_per_rank_step per step (weak
    scaling) in seconds_per_step (the max over ranks)."""
    return world * units_per_rank_step / seconds_per_step


def gather_replica_rows(local, R, device="cpu"):
    """Concatenate per-rank blocks of per-replica rows (the blocks of replica_shard) on every rank:
    local is a float64 array [R_local, ...]; returns [R, ...].  The one collective of a sharded run:
    R x 8 numbers at the end, never inside the sweep loop."""
    import numpy as np
    import torch
    import torch.distributed as dist
    local = np.ascontiguousarray(local, dtype=np.float64)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    tail = local.shape[1:]
    width = int(np.prod(tail)) if tail else 1
    out = torch.zeros((R, width), dtype=torch.float64, device=device)
    lo, hi = replica_shard(R, world, rank)
    assert hi - lo == local.shape[0], (lo, hi, local.shape)
    out[lo:hi] = torch.from_numpy(local.reshape(hi - lo, width)).to(device)
    dist.all_reduce(out, op=dist.ReduceOp.SUM)              # disjoint blocks: the sum is the concatenation
    return out.cpu().numpy().reshape((R,) + tail)
