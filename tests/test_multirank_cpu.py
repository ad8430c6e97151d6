"""The N > 1 path of bench.py on CPU: 2 gloo ranks (no GPU).  The path shards over right-hand-side columns with no data-path
collective (the columns are independent given the surface), so what there is to check on the host side is the
rank -> column assignment of bench.rank_case and the max-over-ranks reduction of the timing."""
from __future__ import annotations

import os
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    nrhs = 16
    c = bench.rank_case(rank, nrhs)
    # the wavenumber perturbed by each column of this rank
    ks = []
    for i in range(nrhs // 2):
        col = c.deta[2 * i]
        spec = np.abs(np.fft.rfft(col))
        ks.append(int(spec.argmax()))
        assert np.array_equal(c.dphi[2 * i + 1], col) and not c.dphi[2 * i].any() and not c.deta[2 * i + 1].any()
    mine = torch.tensor(ks, dtype=torch.int64)
    gathered = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)
    eta_sum = torch.tensor([float(np.abs(c.eta).sum())], dtype=torch.float64)
    etas = [torch.empty_like(eta_sum) for _ in range(world)]
    dist.all_gather(etas, eta_sum)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)   # bench.py reduces its per-rank time with MAX
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        q.put(([g.tolist() for g in gathered], [float(e) for e in etas], float(t)))
    dist.destroy_process_group()


def test_rank_case_shards_columns_over_two_gloo_ranks():
    world, port = 2, 29000 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    ks, etas, tmax = q.get()
    assert etas[0] == etas[1]                       # every rank works on the same surface
    assert ks[0] == list(range(1, 9))               # rank 0: k = 1..8
    assert ks[1] == list(range(9, 17))              # rank 1: the next 8 wavenumbers -- disjoint column sets
    assert tmax == 2.0
