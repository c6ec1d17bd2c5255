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


def test_nev_rule_is_deterministic_and_shared_by_both_arms():
    """bench.choose_nev: config 4 runs all eigenpairs when W + K full solves fit the budget and the nev = N/2 run of
    BASELINE.json otherwise; both arms build `config` from the same function, so their dicts are equal."""
    sys.path.insert(0, ROOT)
    import bench
    N = 49152
    nev, rule = bench.choose_nev(4, N, (N, N // 2), 3, 2, 1500.0)
    assert nev == N and "fits" in rule
    nev, rule = bench.choose_nev(4, N, (N, N // 2), 5, 20, 1500.0)           # the driver's call
    assert nev == N // 2 and "exceed" in rule
    assert bench.choose_nev(4, N, (N, N // 2), 5, 20, 1500.0, nev_arg=100) == (100, "--nev given")
    assert bench.choose_nev(3, 27648, (27648, 13824), 5, 20, 1500.0)[0] == 27648
    assert bench.choose_nev(1, 4096, (4096,), 500, 2000, 1.0)[0] == 4096      # a config with a single run never switches

    from types import SimpleNamespace
    W = SimpleNamespace(name="cfg4_x", N=N)
    assert bench.config_dict(W, nev, rule) == bench.config_dict(W, nev, rule)
    assert set(bench.config_dict(W, nev, rule)) >= {"workload", "N", "nev", "nev_rule", "band_width"}


def test_credited_work_matches_the_closed_forms():
    sys.path.insert(0, ROOT)
    import bench
    cw = bench.credited_work(1024, 512, 64)
    assert cw["p1_flops"] == 16.0 / 3.0 * 1024 ** 3
    assert cw["p4a_flops"] == cw["p4b_flops"] == 8.0 * 1024 * 1024 * 512
    # chase steps: sum over sweeps j of ceil((N - 1 - j) / b)
    assert cw["p2_steps"] == sum(-(-(1023 - j) // 64) for j in range(1023))
    assert cw["p2_bytes"] == cw["p2_steps"] * (2 * (2048 + 4096) * 16 + 1024)
