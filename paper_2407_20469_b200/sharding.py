"""Host-side multi-GPU plumbing: tiles are independent, so N GPUs each take a
contiguous range of the tile list and there is no collective on the data path.  Only the timing
(max over ranks) and the gathering of per-rank counters use torch.distributed."""
from __future__ import annotations


def shard_tiles(n_tiles: int, rank: int, world: int) -> range:
    """Contiguous, balanced partition of range(n_tiles): the first n_tiles % world ranks get one
    extra tile; neighbouring tiles stay on one GPU (scan-row locality for a later stitcher)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, extra = divmod(n_tiles, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """max over all ranks of a per-rank scalar (elapsed device time); identity without a group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None, device="cpu") -> float:
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
