"""N > 1 host path on CPU: two gloo ranks shard the targets of BASELINE.json config 1 with shard_range,
each fills its slice (the oracle stands in for the kernels here: no GPU in this test), and
all_gather_slices reassembles the full field.  Checks the partition, the ragged gather and the
target-range bookkeeping of a (host-only) context per rank."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2001_02765_b200 import SgDisk
from paper_2001_02765_b200.sharding import all_gather_slices, lattice_patch_costs, shard_range, shard_range_by_cost
from workloads import cell_rects, make_config


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_targets, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lay, sigma = make_config(1)
        r = cell_rects(lay)
        first, count = shard_range(n_targets, rank, world)
        with SgDisk.from_layout(lay, device=-1) as d:        # host-only context: bookkeeping only
            d.set_target_range(first, count)
            assert d.launch_counts()[1] == (2 if count else 0)
        idx = np.arange(first, first + count)
        fx, fy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, precision="f64", n_threads=2)
        gx = all_gather_slices(torch.from_numpy(fx), n_targets)
        gy = all_gather_slices(torch.from_numpy(fy), n_targets)
        t = torch.tensor([float(count)])
        dist.all_reduce(t)                                   # every target owned exactly once
        assert int(t.item()) == n_targets
        np.save(os.path.join(out_dir, f"f{rank}.npy"), np.stack([gx.numpy(), gy.numpy()]))
    finally:
        dist.destroy_process_group()


def test_two_rank_target_sharding(tmp_path):
    n_targets = 1001                                         # odd: the two slices differ in length
    port = _free_port()
    mp.spawn(_worker, args=(2, port, n_targets, str(tmp_path)), nprocs=2, join=True)
    a = np.load(tmp_path / "f0.npy")
    b = np.load(tmp_path / "f1.npy")
    assert np.array_equal(a, b)                              # both ranks hold the same assembled field
    lay, sigma = make_config(1)
    r = cell_rects(lay)
    idx = np.arange(n_targets)
    fx, fy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, precision="f64", n_threads=2)
    assert np.array_equal(a[0], fx) and np.array_equal(a[1], fy)


def _worker_cost(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from workloads import nested_layout
        lay = nested_layout(4, 64, 8.0, 16)                  # four levels: coarse patches cost more (far pairs)
        costs = lattice_patch_costs(lay.patches[:, 0])
        ranges = [shard_range_by_cost(costs, lay.P * lay.P, r, world) for r in range(world)]
        first, count = ranges[rank]
        with SgDisk.from_layout(lay, device=-1) as d:        # host-only context: bookkeeping only
            d.set_target_range(first, count)
        local = torch.arange(first, first + count, dtype=torch.float64)      # every target's own index
        full = all_gather_slices(local, lay.n_cells, ranges=ranges)
        assert torch.equal(full, torch.arange(lay.n_cells, dtype=torch.float64))
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([first, count]))
    finally:
        dist.destroy_process_group()


def test_two_rank_cost_based_slices(tmp_path):
    """The lattice-mode partition (whole patches, balanced estimated cost, unequal counts) through the ragged gather."""
    port = _free_port()
    mp.spawn(_worker_cost, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    a, b = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    assert a[0] == 0 and a[0] + a[1] == b[0] and a[1] % 256 == 0 and b[1] % 256 == 0


def test_regrouped_patch_costs_and_large_list_cuts():
    """Cost model of regrouped layouts (1-cell patches packed into padded 16 x 16 blocks): every block of a level costs
    the same whatever its fill, so the patches of a block share its cost; the slices of any world size partition
    [0, N) at patch boundaries, and the prefix-sum path taken for long lists makes the cuts of the plain loop."""
    from paper_2001_02765_b200 import sharding
    from paper_2001_02765_b200.sharding import regrouped_patch_costs
    from workloads import paper_ilr_layout
    lay = paper_ilr_layout(64, 3)
    costs = regrouped_patch_costs(lay.patches, lay.P)
    key = (lay.patches[:, 0].astype(np.int64) << 40) | ((lay.patches[:, 2] >> 4).astype(np.int64) << 20) | (lay.patches[:, 1] >> 4)
    n_blocks = [len(np.unique(key[lay.patches[:, 0] == l])) for l in range(lay.n_levels)]
    for l in range(lay.n_levels):                                  # summed over a level: blocks of the level x all blocks
        assert np.isclose(costs[lay.patches[:, 0] == l].sum(), n_blocks[l] * sum(n_blocks))
    for world in (1, 2, 3, 8):
        cuts = [shard_range_by_cost(costs, lay.P * lay.P, r, world) for r in range(world)]
        assert cuts[0][0] == 0 and sum(c for _, c in cuts) == lay.n_cells
        assert all(cuts[r][0] + cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
        share = [costs[f:f + c].sum() for f, c in cuts]
        assert max(share) - min(share) <= 2.0 * costs.max() + 1e-9 # as even as whole patches allow
    big = np.tile(costs, 100000 // len(costs) + 2)                 # > 100,000 entries: the numpy path
    for world in (2, 5):
        fast = [shard_range_by_cost(big, 1, r, world) for r in range(world)]
        slow = [shard_range_by_cost(list(big[:90000]), 1, r, world) for r in range(world)]
        ref = [sharding.shard_range_by_cost(big[:90000], 1, r, world) for r in range(world)]
        assert slow == ref
        total, acc, p, want_cuts = float(big.sum()), 0.0, 0, [0]
        for r in range(1, world):                                  # the plain loop, restated
            while p < len(big) and acc + 0.5 * big[p] <= total * r / world:
                acc += big[p]; p += 1
            want_cuts.append(p)
        assert [f for f, _ in fast] == want_cuts
