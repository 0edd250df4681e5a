"""Batch sharding for multi-GPU runs: envs are independent, so rank r simply owns a contiguous
slice of the batch and no collective touches the data path.  The only communication is the max-over-ranks of a timing."""


def shard_range(batch: int, rank: int, world: int):
    """contiguous [lo, hi) slice of `batch` envs owned by `rank`; sizes differ by at most one"""
    if not (0 <= rank < world) or batch < 0:
        raise ValueError("bad rank/world/batch")
    base, extra = divmod(batch, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar (e.g. a CUDA-event time) over the process group; identity without one"""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
