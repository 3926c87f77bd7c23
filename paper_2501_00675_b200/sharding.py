"""Host-side multi-GPU plumbing: configurations are independent units (PAPER.md P:87,
"evaluation of a single graph is managed by a single block ... many blocks in the grid evaluate a large
number of graphs simultaneously"; "each of which can be running independent calculations"), so the
batch is split into contiguous slices, one per rank, with NO data-path collective.  torch.distributed is
used only for the barrier and the max-over-ranks of the device time."""
from __future__ import annotations

import os


def shard_range(batch: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice [lo, hi) of `batch` units owned by `rank`; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or batch < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(batch, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def env_rank_world() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of a scalar (the only collective of the whole job); identity when not distributed."""
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None, device=None) -> float:
    if dist is None or not dist.is_available() or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
