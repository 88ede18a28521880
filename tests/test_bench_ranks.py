"""The N > 1 path of bench.py (replicas only): the timed region of the job is the slowest rank's,
the value counts the units of all ranks. World size 2 over gloo on the CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 100.0 + 50.0 * rank                      # rank 1 is the slow replica
    ms = bench.max_over_ranks(ms_local, world)
    out[rank] = (ms, bench.replicas_value(32768, world, ms * 1e-3))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_max_time_and_whole_job_value():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29611, out), nprocs=world, join=True)
    for rank in range(world):
        ms, value = out[rank]
        assert ms == 150.0                               # the maximum over ranks, on every rank
        assert abs(value - 2 * 32768 / 0.150) < 1e-6     # units of all ranks / the slowest rank's time


def test_single_rank_is_a_no_op():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, 1) == 12.5
    assert bench.replicas_value(100, 1, 0.5) == 200.0
