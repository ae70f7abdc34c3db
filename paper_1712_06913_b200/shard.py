"""Host-side sharding for N > 1 GPUs (one process per GPU, torch.distributed).

The path shards by independent grids/frames: every rank images a disjoint, contiguous
block of frames with its own imager; there is NO data-path collective.  torch.distributed is used only for the timing
protocol (barrier, max over ranks).  Nothing here touches the device or the method's arithmetic.
"""
from __future__ import annotations


def shard_range(n_items: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous balanced split of range(n_items): the first n_items % world ranks get one item more."""
    if not (0 <= rank < world) or n_items < 0:
        raise ValueError("need 0 <= rank < world and n_items >= 0")
    base, extra = divmod(n_items, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def frame_seeds(rank: int, frames_per_rank: int) -> range:
    """Weak scaling: rank r draws frames_per_rank frames of its own (distinct noise seeds), so per-GPU work is fixed."""
    return range(rank * frames_per_rank, (rank + 1) * frames_per_rank)


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a scalar (the device time of the slowest rank); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: int, world: int, max_ms: float) -> float:
    """Whole-job throughput: units all ranks processed divided by the slowest rank's time."""
    return units_per_rank * world / (max_ms * 1e-3)
