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
from paper_2001_02765_b200.sharding import all_gather_slices, shard_range
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
