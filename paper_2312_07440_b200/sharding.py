"""Event sharding for N GPUs.  Events are independent (event-level parallelism), so a
rank owns a contiguous event range of every SoA plane and no data-path collective exists."""
from __future__ import annotations


def shard_bounds(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [lo, hi) of `rank`; sizes differ by at most one; covers [0, n_events) exactly."""
    if world < 1 or not (0 <= rank < world) or n_events < 0:
        raise ValueError((n_events, rank, world))
    base, rem = divmod(n_events, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def aggregate_throughput(events_per_rank: list[int], steps: int, max_seconds: float) -> float:
    """Whole-job events/s: all ranks' events over the slowest rank's time (bench.py contract)."""
    return sum(events_per_rank) * steps / max_seconds
