"""Host-side logic of the N>1 path: independent replicas, walkers sharded by rank, no data-path
collective.  The only communication is the timing reduction."""
from __future__ import annotations


def shard_walkers(total_walkers: int, rank: int, world: int):
    """Contiguous, balanced [start, stop) walker range of `rank` (first `total % world` ranks get one more)."""
    if world < 1 or not (0 <= rank < world) or total_walkers < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(total_walkers, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def max_over_ranks(value_ms: float, device=None) -> float:
    """MAX all-reduce of a timing (any backend); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value_ms)
    t = torch.tensor([value_ms], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def aggregate_throughput(walkers_per_rank: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job walker-steps/s: all ranks' walkers over the slowest rank's time."""
    return walkers_per_rank * world * steps / (max_ms * 1e-3)
