"""The path does not shard (replicas only), so the multi-rank logic is host-side only: every rank
runs an independent replica, times are reduced with MAX over ranks, the value is the whole job's.  Covered here
with two gloo ranks on the CPU (no GPU needed)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    mine = [10.0 + 5.0 * rank, 30.0 - 7.0 * rank]            # rank 0: (10, 30); rank 1: (15, 23)
    ms, e2e = bench.max_over_ranks(dist, mine, "cpu")
    out[rank] = (ms, e2e, bench.whole_job_value(1000, 4, world, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_two_gloo_ranks():
    world, port = 2, 29541
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]                                      # every rank sees the same reduced numbers
    ms, e2e, value = res[0]
    assert (ms, e2e) == (15.0, 30.0)                             # slowest rank in each column
    assert abs(value - 2 * 1000 * 4 / 15e-3) < 1e-6             # all ranks' units / max time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(None, [3.0, 4.0], "cpu") == [3.0, 4.0]
    assert bench.whole_job_value(10, 2, 1, 1000.0) == 20.0
