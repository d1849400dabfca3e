"""N > 1 path on CPU (gloo, world_size 2): the path does not shard (replicas only), so the only multi-rank
logic is bench.py's accounting -- max over ranks of the timed region, whole-job value = ranks x steps / that time."""
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
    ms_local = 100.0 * (rank + 1)                  # rank 1 is the slow replica
    ms_total, value = bench.aggregate_replicas(ms_local, steps=10, world=world, dist=dist, device="cpu")
    dist.barrier()
    out[rank] = (ms_total, value)
    dist.destroy_process_group()


def test_replica_accounting_world_size_2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29517, out), nprocs=2, join=True)
    for r in (0, 1):
        ms_total, value = out[r]
        assert ms_total == 200.0                                   # max over ranks
        assert abs(value - 2 * 10 / 0.2) < 1e-9                    # whole-job steps/s


def test_single_rank_accounting():
    sys.path.insert(0, ROOT)
    import bench
    ms_total, value = bench.aggregate_replicas(50.0, steps=5, world=1, dist=None)
    assert ms_total == 50.0 and abs(value - 100.0) < 1e-9
