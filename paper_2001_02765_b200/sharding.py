"""Multi-GPU sharding helpers: targets are independent, so rank r owns a contiguous
target slice, sums over ALL sources, and no data-path collective is needed.

``shard_range`` splits by count (right for the direct kernels, whose cost per target is uniform).  In lattice mode the
cost of a target depends on its level: a target patch of level l meets every source patch, by an offset table if the
two are at most two levels apart (2 FMA per pair) and directly otherwise (~21 FP64 instructions per pair), and the
lattice kernels work on whole 16 x 16 patches.  ``shard_range_by_cost`` therefore cuts the library cell order at
patch boundaries so that every rank gets the same share of the estimated cost (``lattice_patch_costs``).

``all_gather_slices`` is the optional exchange a time-stepping caller uses when every rank wants the whole force
field afterwards; it is outside sg_force and outside bench.py's timed region.
"""
from __future__ import annotations


def shard_range(n: int, rank: int, world: int):
    """Contiguous target slice [first, first+count) of rank ``rank`` out of ``world`` (sizes differ by <= 1)."""
    base, rem = divmod(int(n), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def lattice_patch_costs(patch_levels, far_weight: float = 10.5, near_levels: int = 2):
    """Estimated cost of every target patch in lattice mode, in units of one table-driven patch pair.

    ``patch_levels``: level of every leaf patch, in library patch order.  A pair at most ``near_levels`` levels apart
    costs 1, a farther pair ``far_weight`` (21 FP64 instructions per pair against 2)."""
    levels = [int(l) for l in patch_levels]
    n_levels = max(levels) + 1
    per_level = [0] * n_levels
    for l in levels:
        per_level[l] += 1
    cost_of_level = [sum(per_level[m] * (1.0 if abs(l - m) <= near_levels else far_weight) for m in range(n_levels))
                     for l in range(n_levels)]
    return [cost_of_level[l] for l in levels]


def shard_range_by_cost(patch_costs, cells_per_patch: int, rank: int, world: int):
    """Contiguous target slice [first, first+count) of rank ``rank``, cut at patch boundaries so that the cumulative
    cost is split as evenly as whole patches allow.  The slices of ranks 0..world-1 partition [0, N)."""
    n = len(patch_costs)
    total = float(sum(patch_costs))
    cuts = [0]
    acc, p = 0.0, 0
    for r in range(1, world):
        want = total * r / world
        while p < n and acc + 0.5 * patch_costs[p] <= want:
            acc += patch_costs[p]
            p += 1
        cuts.append(p)
    cuts.append(n)
    first, last = cuts[rank], cuts[rank + 1]
    return first * cells_per_patch, (last - first) * cells_per_patch


def all_gather_slices(local, n: int, group=None, ranges=None):
    """Assemble the length-``n`` array whose rank-r slice is ``local`` on rank r.  ``ranges`` lists (first, count) of
    every rank (default: ``shard_range``).

    ``local`` is a 1-D tensor (CPU with gloo, CUDA with nccl).  Slices may differ in length, so every rank pads to
    the longest slice before ``all_gather_into_tensor``.
    """
    import torch
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    if ranges is None:
        ranges = [shard_range(n, r, world) for r in range(world)]
    first, count = ranges[rank]
    if local.numel() != count:
        raise ValueError(f"rank {rank}: local slice has {local.numel()} elements, expected {count}")
    longest = max(c for _, c in ranges)
    padded = torch.zeros(longest, dtype=local.dtype, device=local.device)
    padded[:count] = local
    out = torch.empty(world * longest, dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(out, padded, group=group)
    pieces = []
    for r in range(world):
        _, c = ranges[r]
        pieces.append(out[r * longest:r * longest + c])
    return torch.cat(pieces)
