"""Host-side multi-rank logic on CPU (gloo, world_size 2): disjoint ray ranges, per-rank seeds, max-over-ranks timing.
The ray path itself has no collective."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2508_15967_b200 import inputs, sharding


def test_ray_ranges_partition_the_ensemble():
    for n, world in ((0, 1), (1, 4), (10, 3), (2**20, 8), (1000003, 7)):
        spans = [sharding.ray_range(n, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        sizes = [e - b for b, e in spans]
        assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.ray_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n = 1001
        b, e = sharding.ray_range(n, rank, world)
        w = inputs.config(1, n_rays=n)                       # every rank draws the same ensemble, keeps its own range
        mine = w.x0[:, b:e]
        counts = torch.tensor([e - b], dtype=torch.int64)
        dist.all_reduce(counts)                              # bookkeeping only
        t_max = sharding.max_over_ranks(0.1 * (rank + 1), dist)
        total = sharding.sum_over_ranks(float(mine[1].sum()), dist)
        seeds = sharding.rank_seed(1004, rank)
        import bench                                          # bench.py's own per-rank plan, both scaling modes
        strong, weak = bench.rank_plan("strong", 4, 1001, rank, world), bench.rank_plan("weak", 4, 1001, rank, world)
        covered = torch.tensor([strong[1][1] - strong[1][0]], dtype=torch.int64)
        dist.all_reduce(covered)
        assert int(covered.item()) == 1001 and strong[0] == 1004 and strong[1] == (b, e)
        assert weak == (seeds, None)
        dist.barrier()
        q.put((rank, int(counts.item()), t_max, total, seeds, float(w.x0[1].sum())))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_cover_all_rays_and_take_the_max_time():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [1001, 1001]                 # the two ranges cover the ensemble
    assert [r[2] for r in res] == [pytest.approx(0.2)] * 2      # max over ranks of the timed interval
    assert res[0][3] == pytest.approx(res[0][5], rel=1e-12)     # shard sums add up to the whole ensemble's
    assert res[0][4] != res[1][4]                              # weak-scaling batches differ per rank
    assert sharding.max_over_ranks(3.0) == 3.0                 # no process group: identity
