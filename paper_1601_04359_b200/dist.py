"""Multi-GPU plumbing.  The evaluation itself shards with no exchange: images of a batch (and
swap proposals) are independent units, which is also the paper's own dual-GPU plan ("uniformly distribute the generated
segments, so that each device holds only a certain amount of them").  This module splits
the units across ranks (`shard_range`), reduces times and unit counts for reporting, and -- for the strong-scaling
split of one batch -- gathers the per-rank count slices into the whole array (`gather_shards`: the ONE collective of
the split path, an all-gather).  One process per GPU; `torch.distributed` (NCCL on GPUs, gloo in the CPU tests)."""
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


def gather_buffer(local, n_units: int, world: int):
    """Receive buffer of `gather_shards`: [world * ceil(n_units / world), ...] like `local` (slices are padded to the
    largest shard so that one all-gather moves them)."""
    import torch
    per = -(-int(n_units) // int(world))
    return torch.empty((world * per,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)


def gather_shards(local, buf, n_units: int, rank: int, world: int):
    """All-gathers the per-rank result slices of a batch that was split with `shard_range`: `local` holds the results
    of units [begin, end) of this rank; returns a view/tensor [n_units, ...] in unit order, the same on every rank.
    `buf` comes from `gather_buffer`.  Without an initialised process group (one rank) `local` is returned."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized() and world > 1):
        return local
    per = buf.shape[0] // world
    b, e = shard_range(n_units, rank, world)
    if e - b == per:
        send = local
    else:                                                 # a short last shard: pad to the common slice size
        send = torch.zeros((per,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
        send[: e - b] = local
    dist.all_gather_into_tensor(buf, send.contiguous())
    if n_units % world == 0:
        return buf[:n_units]
    parts = []
    for r in range(world):
        rb, re = shard_range(n_units, r, world)
        parts.append(buf[r * per: r * per + (re - rb)])
    return torch.cat(parts, dim=0)
