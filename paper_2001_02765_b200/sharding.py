"""Multi-GPU sharding helpers: targets are independent, so rank r owns the
contiguous target slice ``shard_range(N, r, world)``, sums over ALL sources, and no data-path collective is
needed.  ``all_gather_slices`` is the optional exchange a time-stepping caller uses when every rank wants the
whole force field afterwards; it is outside sg_force and outside bench.py's timed region.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int):
    """Contiguous target slice [first, first+count) of rank ``rank`` out of ``world`` (sizes differ by <= 1)."""
    base, rem = divmod(int(n), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def all_gather_slices(local, n: int, group=None):
    """Assemble the length-``n`` array whose rank-r slice ``shard_range(n, r, world)`` is ``local`` on rank r.

    ``local`` is a 1-D tensor (CPU with gloo, CUDA with nccl).  Slices may differ in length by one, so every
    rank pads to the longest slice before ``all_gather_into_tensor``.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    first, count = shard_range(n, rank, world)
    if local.numel() != count:
        raise ValueError(f"rank {rank}: local slice has {local.numel()} elements, expected {count}")
    longest = shard_range(n, 0, world)[1]
    padded = torch.zeros(longest, dtype=local.dtype, device=local.device)
    padded[:count] = local
    out = torch.empty(world * longest, dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(out, padded, group=group)
    pieces = []
    for r in range(world):
        _, c = shard_range(n, r, world)
        pieces.append(out[r * longest:r * longest + c])
    return torch.cat(pieces)
