"""N > 1 host logic of the column-sharded back-transformation (SURVEY.md 8(f)3 first slice) on CPU with
gloo, world_size 2: the shard plan covers every column once, is slab-aligned and balanced, and applying a unitary to the
shards and gathering equals applying it to the whole (column independence -- what makes S4a / S4b shardable)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_column_shards_cover_and_balance():
    sys.path.insert(0, ROOT)
    from paper_2310_03341_b200 import shard
    for nev, world in [(49152, 8), (24576, 8), (1000, 3), (64, 4), (1, 2), (0, 2), (130, 2), (24576, 7)]:
        sh = shard.column_shards(nev, world)
        assert len(sh) == world and sh[0][0] == 0 and sh[-1][1] == nev
        for (b0, e0), (b1, e1) in zip(sh, sh[1:]):
            assert e0 == b1 and b0 <= e0
        for b, e in sh:
            assert b % shard.SLAB == 0 or b == nev
        sizes = [e - b for b, e in sh]
        assert max(sizes) - min(sizes) < 2 * shard.SLAB        # one slab + the partial tail slab


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2310_03341_b200 import shard
    N, nev = 96, 200 - 63                       # ragged: 137 columns -> slabs 64 + 64 + 9
    rng = np.random.default_rng(7)              # same seed on every rank: replicated S1-S3 give identical inputs
    Q, _ = np.linalg.qr(rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N)))
    Z = rng.standard_normal((N, nev)) + 1j * rng.standard_normal((N, nev))
    b, e = shard.column_shards(nev, world)[rank]
    mine = torch.from_numpy(np.ascontiguousarray((Q @ Z[:, b:e]).T))            # this rank's back-transformed columns
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([e - b]))
    mx = max(int(s.item()) for s in sizes)                    # all_gather wants equal shapes: pad to the widest shard
    padded = torch.zeros((mx, N), dtype=torch.complex128)
    padded[: e - b] = mine
    parts = [torch.zeros((mx, N), dtype=torch.complex128) for _ in sizes]
    dist.all_gather(parts, padded)
    full = torch.cat([p[: int(s.item())] for p, s in zip(parts, sizes)], 0).numpy().T
    out[rank] = (float(np.abs(full - Q @ Z).max()), [int(s.item()) for s in sizes])
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_backtransform_gathers_to_the_full_result_world2():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29547, out), nprocs=world, join=True)
    for r in range(world):
        err, sizes = out[r]
        assert err <= 1e-13
        assert sizes == [128, 9]
