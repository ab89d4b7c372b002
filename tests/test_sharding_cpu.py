"""N > 1 host logic on CPU with two gloo ranks: contiguous shards cover the batch exactly once,
per-rank oracle results concatenate to the whole-batch result, and the timing reduction is a max."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2009_06635_b200 import sharding, workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    oracle.set_threads(1)
    grid = W.grid_config1()
    x, q2 = W.queries_in_range(grid, n, 1)
    a, b = sharding.shard_range(n, rank, world)
    part = oracle.OraclePdfGrid.from_spec(grid).xfxq2(grid.pids, x[a:b], q2[a:b])
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([b - a]))
    ms = sharding.reduce_max_ms(10.0 + 5.0 * rank, dist)
    full = torch.zeros((len(grid.pids), n), dtype=torch.float64)
    full[:, a:b] = torch.from_numpy(part)
    dist.all_reduce(full)  # test-only gather: disjoint shards sum to the whole
    if rank == 0:
        ret["sizes"] = [int(s) for s in sizes]
        ret["ms"] = ms
        ret["full"] = full.numpy()
    dist.destroy_process_group()


def test_two_rank_sharding_gloo():
    n, world = 1001, 2
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(world, _free_port(), n, ret), nprocs=world, join=True)
    assert sum(ret["sizes"]) == n and max(ret["sizes"]) - min(ret["sizes"]) <= 1
    assert ret["ms"] == 15.0
    import oracle
    grid = W.grid_config1()
    x, q2 = W.queries_in_range(grid, n, 1)
    whole = oracle.OraclePdfGrid.from_spec(grid).xfxq2(grid.pids, x, q2)
    assert np.array_equal(ret["full"], whole)
    assert sharding.aggregate_throughput([500 * 3, 501 * 3], [10.0, 15.0]) == (1001 * 3) / 15e-3


def test_shard_range_properties():
    for n in (0, 1, 7, 100, 1001):
        for world in (1, 2, 3, 8):
            edges = [sharding.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
