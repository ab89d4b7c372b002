"""Host logic of the multi-GPU path: points are independent, so a batch is cut
into contiguous per-rank ranges, the grid is replicated at load, and no collective touches the
data path.  The only exchange is the max-over-ranks of the device time for reporting."""
from __future__ import annotations


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [begin, end) of `rank`; sizes differ by at most one point."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank/world/n_total")
    base, rem = divmod(n_total, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def aggregate_throughput(units_per_rank, ms_per_rank) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    return sum(units_per_rank) / (max(ms_per_rank) * 1e-3)


def reduce_max(values, dist=None, device=None) -> list:
    """Element-wise max over ranks of a list of times (identity without a process group)."""
    values = [float(v) for v in values]
    if dist is None or not dist.is_initialized():
        return values
    import torch
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def reduce_max_ms(ms: float, dist=None, device=None) -> float:
    """Max over ranks of a device time (identity without a process group)."""
    return reduce_max([ms], dist, device)[0]


def rank_seed(config: int, rank: int) -> int:
    """Seed of the batch `rank` draws for itself in a weak-scaling run: every rank evaluates its own
    full-size batch (no point is shared, nothing is exchanged); rank 0's is the single-GPU batch."""
    if rank < 0:
        raise ValueError("bad rank")
    return config + 100 * rank


def e2e_split(total_points: int, rank: int, world: int, cap: int) -> tuple[int, int]:
    """End-to-end leg: `total_points` host-resident points are cut over the ranks by shard_range, each
    rank taking at most `cap` (its device batch) and at least one.  -> (this rank's points, all ranks')."""
    sizes = []
    for r in range(world):
        a, b = shard_range(max(total_points, world), r, world)
        sizes.append(max(1, min(cap, b - a)))
    return sizes[rank], sum(sizes)
