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


def reduce_max_ms(ms: float, dist=None, device=None) -> float:
    """Max over ranks of a device time (identity without a process group)."""
    if dist is None or not dist.is_initialized():
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])
