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


def regrouped_patch_costs(patches, patch_cells: int, far_weight: float = 10.5, near_levels: int = 2):
    """Estimated lattice-mode cost of every leaf patch of a layout of small patches (1, 2 or 4 cells a side, e.g. the
    paper's zone-wise quadtrees), which the library regroups into padded 16 x 16 blocks: the kernels work on whole
    blocks, holes included, so a block of level l costs sum_m n_blocks(m) * (1 or ``far_weight``) whatever its fill,
    and every patch in it carries an equal share.  A patch of a sparsely filled block (the rim of a refined region)
    is therefore dearer than one of a full block.

    ``patches``: integer array [n, 3] = (level, i0, j0) in library patch order; returns a float array [n] for
    ``shard_range_by_cost``.  (numpy: these layouts have millions of patches.)"""
    import numpy as np
    pa = np.asarray(patches, dtype=np.int64).reshape(-1, 3)
    if patch_cells not in (1, 2, 4):
        raise ValueError("regrouped_patch_costs is for patches of 1, 2 or 4 cells a side")
    # a patch is aligned to its own size, which divides 16: all its cells fall into one block
    key = (pa[:, 0] << 56) | ((pa[:, 2] >> 4) << 28) | (pa[:, 1] >> 4)
    blocks, inverse, per_block = np.unique(key, return_inverse=True, return_counts=True)
    n_levels = int(pa[:, 0].max()) + 1
    blocks_of_level = np.bincount(blocks >> 56, minlength=n_levels).astype(np.float64)
    dist = np.abs(np.arange(n_levels)[:, None] - np.arange(n_levels)[None, :])
    cost_of_level = (np.where(dist <= near_levels, 1.0, far_weight) * blocks_of_level[None, :]).sum(axis=1)
    return cost_of_level[pa[:, 0]] / per_block[inverse]


def shard_range_by_cost(patch_costs, cells_per_patch: int, rank: int, world: int):
    """Contiguous target slice [first, first+count) of rank ``rank``, cut at patch boundaries so that the cumulative
    cost is split as evenly as whole patches allow.  The slices of ranks 0..world-1 partition [0, N)."""
    n = len(patch_costs)
    if n > 100000:                                     # millions of 1-cell patches: the same cuts by prefix sums
        import numpy as np
        c = np.asarray(patch_costs, dtype=np.float64)
        mid = np.cumsum(c) - 0.5 * c                   # patch p goes left of cut r iff its midpoint <= total r / world
        total = float(c.sum())
        cuts = [0] + [int(np.searchsorted(mid, total * r / world, side="right")) for r in range(1, world)] + [n]
        first, last = cuts[rank], cuts[rank + 1]
        return first * cells_per_patch, (last - first) * cells_per_patch
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
