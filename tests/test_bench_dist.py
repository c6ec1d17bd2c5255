"""N > 1 host logic of bench.py on CPU (gloo, world_size 2): the path does not shard ("replicas only",
DESIGN.md section 5), so the only cross-rank step is the max-over-ranks of the device-timed totals."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local_ms = 100.0 + 50.0 * rank            # rank 1 is the slower replica
    total = bench.max_over_ranks(local_ms, dist)
    out[rank] = (total, bench.replica_value_s(total / 2, world))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_metric_world2():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29531, out), nprocs=world, join=True)
    assert out[0][0] == out[1][0] == 150.0                 # every rank sees the slowest replica's time
    assert abs(out[0][1] - 150.0 / 2 / 1e3 / 2) < 1e-15    # 2 steps, 2 replicas -> seconds per eigensolve


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, None) == 12.5
    assert bench.replica_value_s(2000.0, 1) == 2.0
