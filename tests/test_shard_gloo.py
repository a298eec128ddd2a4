"""world_size-2 CPU test (gloo) of the multi-rank host logic: domain blocks are disjoint and cover all
domains, every rank generates the inputs of its own domains, and the only cross-rank traffic of the
bench (MAX of the step time, SUM of electrons) reduces as expected.  No data-path collective exists."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, ndom_total, out):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import workloads as W
    from paper_2509_00966_b200.shard import domain_block
    lo, hi = domain_block(ndom_total, rank, world)
    c = W.get_config(0)
    occ_sum = sum(float(W.generate_domain(c, d)["occ"].sum()) for d in range(lo, hi))
    owned = torch.zeros(ndom_total, dtype=torch.int64)
    owned[lo:hi] = 1
    dist.all_reduce(owned)
    t = torch.tensor([0.010 * (rank + 1)], dtype=torch.float64)     # pretend step times
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e = torch.tensor([occ_sum], dtype=torch.float64)
    dist.all_reduce(e)
    if rank == 0:
        np.save(out, np.array([owned.min().item(), owned.max().item(), t.item(), e.item()]))
    dist.destroy_process_group()


def test_two_ranks_shard_domains(tmp_path):
    out = str(tmp_path / "r.npy")
    mp.spawn(_worker, args=(2, 29533, 5, out), nprocs=2, join=True)
    lo, hi, tmax, electrons = np.load(out)
    assert lo == 1 and hi == 1                 # every domain owned exactly once
    assert abs(tmax - 0.020) < 1e-12           # max over ranks
    assert electrons == 5 * 16.0               # config 0: 8 orbitals x f = 2 per domain


def test_domain_block_properties():
    sys.path.insert(0, ROOT)
    from paper_2509_00966_b200.shard import domain_block, weak_scaling_block
    for n in (0, 1, 7, 64):
        for w in (1, 2, 3, 8):
            blocks = [domain_block(n, r, w) for r in range(w)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(w - 1))
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
    assert weak_scaling_block(64, 3) == (192, 256)
