"""The N > 1 host logic of bench.py on CPU: two gloo ranks at 127.0.0.1."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

from paper_1211_6234_b200 import multirank  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert multirank.env() == (rank, world, rank)
    # every rank times its own work; the job's time is the slowest rank's
    mine = [10.0 + 5.0 * rank, 3.0 - rank]
    got = multirank.max_over_ranks(mine)
    # a ladder of 5 replicas split over the ranks: every rank ends with all rows, in replica order
    import numpy as np
    lo, hi = multirank.replica_shard(5, world, rank)
    rows = np.arange(lo, hi, dtype=np.float64)[:, None] * np.ones((1, 8)) + 0.25
    allrows = multirank.gather_replica_rows(rows, 5)
    assert allrows.shape == (5, 8) and np.array_equal(allrows[:, 0], np.arange(5) + 0.25)
    dist.barrier()
    out.put((rank, got, multirank.rank_seed(0x12116234, rank), multirank.rank_replica_offset(64, rank)))
    dist.destroy_process_group()


def test_two_ranks_max_and_seeds():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1] == [15.0, 3.0]                 # max over ranks, identical everywhere
    assert res[0][2] != res[1][2]                                # independent chains per rank
    assert (res[0][2] & 0xFFFFFFFF) == (res[1][2] & 0xFFFFFFFF) == 0x12116234   # ... that differ in the high word only
    assert multirank.rank_seed(1000, 1) != multirank.rank_seed(2000, 0)          # no collision between base seeds
    assert [res[0][3], res[1][3]] == [0, 64]                     # bench.py: one seed, disjoint replica indices
    # weak scaling: value = world x per-rank units / max time
    assert multirank.whole_job_rate(4_194_304, world, 0.015) == 2 * 4_194_304 / 0.015


def test_single_process_identity():
    assert multirank.env()[1] >= 1
    assert multirank.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]


def test_replica_shards_partition_the_ladder():
    for R in (64, 16, 5, 1):
        for world in (1, 2, 3, 8):
            blocks = [multirank.replica_shard(R, world, r) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == R
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
