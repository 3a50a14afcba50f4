"""The N > 1 path of bench.py is "replicas only" (Multi-GPU): no data-path collective, whole-job value =
all ranks' units over the slowest rank's time.  This covers that host logic with two gloo ranks on the CPU."""
import os
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = 2.0 if rank == 0 else 5.0            # rank 1 is the slow replica
    out[rank] = (bench.max_over_ranks(ms, world), bench.aggregate_throughput(100, ms, world))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation():
    world = 2
    port = 29500 + os.getpid() % 1000
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    for rank in range(world):
        t, v = out[rank]
        assert t == 5.0                       # every rank sees the slowest rank's time
        assert abs(v - world * 100 / 5e-3) < 1e-6


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert abs(bench.aggregate_throughput(10, 2.0, 1) - 5000.0) < 1e-9
