"""Multi-GPU plumbing: the path shards with no exchange, so this module only
splits independent units (images of a batch, swap proposals) across ranks and reduces TIMES and unit
counts for reporting.  One process per GPU; `torch.distributed` (NCCL on GPUs, gloo in the CPU tests).
No data-path collective exists or is needed (the paper's own dual-GPU plan distributes
segments the same way)."""
from __future__ import annotations


def shard_range(n_units: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous [begin, end) slice of n_units independent units for `rank`; sizes differ by at most 1
    and the slices of all ranks partition range(n_units)."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard request")
    q, r = divmod(int(n_units), int(world))
    begin = rank * q + min(rank, r)
    return begin, begin + q + (1 if rank < r else 0)


def rank_seed_offset(rank: int) -> int:
    """Weak scaling: rank r evaluates its own images, seeds offset by 100000 r (bench.py)."""
    return 100000 * int(rank)


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX over all ranks of a list of floats (device times are reported as the slowest
    rank's).  Without an initialised process group the values are returned unchanged."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def sum_over_ranks(value: int, device="cpu") -> int:
    """Exact integer SUM over ranks (units processed by the whole job)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([int(value)], dtype=torch.int64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.cpu()[0])
