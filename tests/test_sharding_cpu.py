"""N > 1 host logic on CPU with two gloo ranks: contiguous shards cover the batch exactly once,
per-rank oracle results concatenate to the whole-batch result, and the timing reduction is a max.
These are the functions bench.py runs under torchrun (per-rank batch seed, end-to-end split,
max-over-ranks of the timings, whole-job throughput) -- bench.py holds no copy of its own."""
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
    several = sharding.reduce_max([1.0 + rank, 7.0 - rank, 3.0], dist)   # bench.py: total, mean, median, best in one go
    n_e, n_e_all = sharding.e2e_split(n, rank, world, cap=n)              # bench.py's end-to-end leg
    e_sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(e_sizes, torch.tensor([n_e]))
    xr, _ = W.queries_in_range(grid, 16, sharding.rank_seed(3, rank))     # the batch this rank draws for itself
    heads = [torch.zeros(16, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(heads, torch.from_numpy(xr))
    full = torch.zeros((len(grid.pids), n), dtype=torch.float64)
    full[:, a:b] = torch.from_numpy(part)
    dist.all_reduce(full)  # test-only gather: disjoint shards sum to the whole
    if rank == 0:
        ret["sizes"] = [int(s) for s in sizes]
        ret["ms"] = ms
        ret["several"] = several
        ret["e2e"] = ([int(v) for v in e_sizes], n_e_all)
        ret["heads"] = [h.numpy() for h in heads]
        ret["full"] = full.numpy()
    dist.destroy_process_group()


def test_two_rank_sharding_gloo():
    n, world = 1001, 2
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(world, _free_port(), n, ret), nprocs=world, join=True)
    assert sum(ret["sizes"]) == n and max(ret["sizes"]) - min(ret["sizes"]) <= 1
    assert ret["ms"] == 15.0
    assert ret["several"] == [2.0, 7.0, 3.0]
    assert sum(ret["e2e"][0]) == ret["e2e"][1] == n
    assert not np.array_equal(ret["heads"][0], ret["heads"][1])          # the ranks' batches differ ...
    assert np.array_equal(ret["heads"][0], W.queries_in_range(W.grid_config1(), 16, 3)[0])  # ... rank 0's is the 1-GPU one
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


def test_bench_uses_these_functions():
    """bench.py takes its per-rank seed, its end-to-end split, its max over ranks and its whole-job
    throughput from sharding.py and reduces nothing on its own."""
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "bench.py")).read()
    for name in ("sharding.rank_seed(", "sharding.e2e_split(", "sharding.reduce_max(", "sharding.reduce_max_ms(",
                 "sharding.aggregate_throughput("):
        assert name in src, name
    assert "all_reduce" not in src


def test_e2e_split_properties():
    for total in (1, 5, 1000, 10**8):
        for world in (1, 2, 3, 8):
            sizes = [sharding.e2e_split(total, r, world, cap=10**8)[0] for r in range(world)]
            alls = {sharding.e2e_split(total, r, world, cap=10**8)[1] for r in range(world)}
            assert alls == {sum(sizes)} and sum(sizes) == max(total, world) and max(sizes) - min(sizes) <= 1
    assert sharding.e2e_split(10**8, 0, 2, cap=10**6) == (10**6, 2 * 10**6)   # never more than the rank's device batch
    assert sharding.rank_seed(3, 0) == 3 and len({sharding.rank_seed(3, r) for r in range(8)}) == 8
