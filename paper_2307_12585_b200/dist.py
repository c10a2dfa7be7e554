"""Multi-GPU plumbing: the path shards with no exchange step.

One process per GPU (torch.distributed; NCCL on GPUs, gloo in the CPU tests).  Waveforms (batch items) are
independent, so the only communication is the barrier around a timed region and the max over ranks of the
device time.  Nothing here touches the data path.
"""
from __future__ import annotations

import os


def env_world():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def shard_range(n_items: int, world: int, rank: int) -> range:
    """Contiguous, balanced slice of n_items batch items owned by `rank`: sizes differ by at most one and the
    slices of ranks 0..world-1 partition range(n_items) in order."""
    if world < 1 or not (0 <= rank < world) or n_items < 0:
        raise ValueError("shard_range: bad arguments")
    base, extra = divmod(n_items, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (a device time in ms) over all ranks; identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """Sum of a per-rank scalar (units processed) over all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()
