"""World-size-2 gloo test (CPU) of bench.py's multi-GPU host logic: replicas only, the job's time is the
max over ranks and `value` is the whole-job figure.  No data-path collective exists."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    us = [10.0 + 5.0 * rank, 100.0 - 7.0 * rank]          # rank 0: (10, 100); rank 1: (15, 93)
    got = bench.max_over_ranks(us, dist, "cpu")
    dist.barrier()
    out[rank] = (got, bench.whole_job_us_per_call(got[0], world))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo_world2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29517 + os.getpid() % 1000, out), nprocs=2, join=True)
    for rank in (0, 1):
        got, value = out[rank]
        assert got == [15.0, 100.0]
        assert value == 7.5                                  # two replicas -> two calls per 15 us


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0], None, "cpu") == [3.0, 4.0]
    assert bench.whole_job_us_per_call(8.0, 1) == 8.0
