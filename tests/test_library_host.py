"""CPU-side tests of the C-ABI library: it loads, exports every symbol include/sg_disk.h declares,
and the host layout builder (S1) validates and flattens patch lists correctly.  No compute calls:
contexts are created with device = -1 (host-only), on which every compute entry must fail loudly."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_2001_02765_b200 as sgd
from paper_2001_02765_b200 import SgDisk, SgError, binding
from workloads import (Layout, make_config, cell_rects, expected_counts, paper_ilr_layout, nested_layout,
                       random_refined_layout)
from workloads.configs import cell_centres, _sorted_patches, uniform_layout

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include")))
                  if f.endswith(".h"))
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sg_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTED_SYMBOLS)
    lib = ctypes.CDLL(binding.lib_path())
    for name in declared:
        assert getattr(lib, name) is not None
    assert "sm_100a" in sgd.version()


def test_no_oracle_in_product_path():
    """The product package must not import, read or link anything under oracle/ (or _work/)."""
    pkg = os.path.join(ROOT, "paper_2001_02765_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.lower(), f"{f} mentions the oracle"
                assert "_work" not in src, f


@pytest.mark.parametrize("cfg,n_v", [(1, 65 * 65), (2, 7361), (3, 53889)])
def test_layout_counts_and_geometry(cfg, n_v):
    lay, _ = make_config(cfg)
    exp = expected_counts(cfg)
    with SgDisk.from_layout(lay, device=-1) as d:
        info = d.layout_info()
        assert info["n_cells"] == exp["n_cells"] == d.num_cells
        assert info["n_vertices"] == n_v == d.num_vertices          # SURVEY.md section 8 size table
        assert info["balanced"] == 1
        xc, yc, h = d.cell_geometry()
    x, y, hh = cell_centres(lay)
    assert np.array_equal(xc, x) and np.array_equal(yc, y) and np.array_equal(h, hh)


def test_vertex_count_matches_bruteforce_dedupe():
    lay = paper_ilr_layout(32, 3)                     # P = 1 quadtree of the paper's kind, with hanging nodes
    r = cell_rects(lay)
    corners = set()
    for a, b in (("kxl", "kyd"), ("kxl", "kyu"), ("kxr", "kyd"), ("kxr", "kyu")):
        corners |= set(zip(r[a].tolist(), r[b].tolist()))
    with SgDisk.from_layout(lay, device=-1) as d:
        assert d.num_vertices == len(corners)
        assert d.num_cells == lay.n_cells


def test_unbalanced_layout_is_accepted_and_flagged():
    # Fig. 1 / Table 10 of the paper: level-3 zones abut a level-1 zone
    l0 = [(0, i, j) for j in range(4) for i in range(4) if (i, j) not in ((1, 1), (2, 2))]
    l1 = [(1, 2, 2), (1, 3, 3)] + [(1, 4 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    l2 = [(2, 4 + di, 6 + dj) for dj in (0, 1) for di in (0, 1)]
    l2 += [(2, 6 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    lay = Layout(3, np.array([0.25, 0.125, 0.0625]), 0.0, 0.0, 1, _sorted_patches(l0 + l1 + l2))
    with SgDisk.from_layout(lay, device=-1) as d:
        assert d.num_cells == 28                       # "28 leaves"
        assert d.layout_info()["balanced"] == 0
        _, _, h = d.cell_geometry()
        assert abs(np.sum(h * h) - 1.0) < 1e-15        # leaves tile [0,1]^2


def test_layout_errors():
    lay, _ = make_config(2)
    mk = lambda **kw: SgDisk(kw.get("nl", lay.n_levels), kw.get("cw", lay.cell_width), -1, -1, kw.get("P", lay.P),
                             kw.get("p", lay.patches), device=-1)
    with pytest.raises(SgError) as e:                  # fine patch inside a coarse leaf
        mk(p=np.vstack([lay.patches, [[1, 0, 0]]]))
    assert e.value.code == binding.SG_ERR_LAYOUT and "overlap" in str(e.value)
    with pytest.raises(SgError) as e:                  # coarse patch over existing fine leaves
        mk(p=np.vstack([lay.patches, [[0, 16, 16]]]))
    assert e.value.code == binding.SG_ERR_LAYOUT
    with pytest.raises(SgError) as e:                  # duplicate
        mk(p=np.vstack([lay.patches, lay.patches[:1]]))
    assert e.value.code == binding.SG_ERR_LAYOUT and "duplicate" in str(e.value)
    with pytest.raises(SgError) as e:                  # off the patch lattice
        mk(p=np.array([[0, 3, 0]], dtype=np.int32))
    assert e.value.code == binding.SG_ERR_LAYOUT
    with pytest.raises(SgError) as e:                  # level out of range
        mk(p=np.array([[2, 0, 0]], dtype=np.int32))
    assert e.value.code == binding.SG_ERR_LAYOUT
    with pytest.raises(SgError) as e:                  # widths not halving
        mk(cw=[1 / 32, 1 / 48])
    assert e.value.code == binding.SG_ERR_ARG
    with pytest.raises(SgError) as e:
        mk(P=0)
    assert e.value.code == binding.SG_ERR_ARG
    with pytest.raises(SgError) as e:                  # empty patch list
        SgDisk(1, [1.0], 0, 0, 16, np.zeros((0, 3), dtype=np.int32), device=-1)
    assert e.value.code == binding.SG_ERR_ARG
    with pytest.raises(SgError) as e:                  # lattice too large for exact FP64 integers
        SgDisk(1, [1.0], 0, 0, 16, np.array([[0, 1 << 25, 0]], dtype=np.int32), device=-1)
    assert e.value.code == binding.SG_ERR_LAYOUT


def test_host_only_context_never_computes():
    """No CPU fallback: compute entry points on a context without a device return SG_ERR_CUDA."""
    lay = uniform_layout(16, 0.0, 0.0, 1.0, 8)
    with SgDisk.from_layout(lay, device=-1) as d:
        lib = binding.load_library()
        dummy = ctypes.c_void_p(16)
        assert lib.sg_set_density(d._ctx, dummy, None) == binding.SG_ERR_CUDA
        assert lib.sg_force(d._ctx, dummy, dummy, None) == binding.SG_ERR_CUDA
        assert b"no CPU fallback" in lib.sg_last_error(d._ctx)
        assert d.launch_counts() == (5, 2)
        d.set_target_range(5, 0)
        assert d.launch_counts() == (5, 0)
        with pytest.raises(SgError):
            d.set_target_range(250, 10)


def test_shard_range_partitions_targets():
    for n in (0, 1, 7, 4096, 1048576, 448768):
        for world in (1, 2, 3, 8):
            pieces = [binding.shard_range(n, r, world) for r in range(world)]
            assert pieces[0][0] == 0 and sum(c for _, c in pieces) == n
            for (f0, c0), (f1, _) in zip(pieces, pieces[1:]):
                assert f0 + c0 == f1
            assert max(c for _, c in pieces) - min(c for _, c in pieces) <= 1


def _near_pair_counts(lay):
    """(target patch, source patch) pairs by level distance: same, source 1 coarser, 1 finer, 2 coarser, 2 finer."""
    cnt = np.bincount(lay.patches[:, 0], minlength=lay.n_levels).astype(np.int64)
    L = lay.n_levels
    return [int(np.sum(cnt * cnt)),
            int(sum(cnt[l] * cnt[l - 1] for l in range(1, L))), int(sum(cnt[l] * cnt[l + 1] for l in range(L - 1))),
            int(sum(cnt[l] * cnt[l - 2] for l in range(2, L))), int(sum(cnt[l] * cnt[l + 2] for l in range(L - 2)))]


@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4", "nest5", "rand1", "rand2", "rand3", "gap", "shuffled"])
def test_lattice_plan_reaches_every_near_patch_pair_exactly_once(name):
    """Host replay of the walk of the offset-table kernels (groups x offsets x warps, the same index arithmetic as
    patch_offset_kernel): every patch pair at most two levels apart is reached exactly once, in the right class."""
    if name.startswith("cfg"):
        lay = make_config(int(name[3:]))[0]
    elif name == "nest5":
        lay = nested_layout(5, 64, 8.0, 16)
    elif name == "gap":                                            # levels 0 and 2 only: level 1 has no leaf patch
        lay = Layout(3, np.array([1.0, 0.5, 0.25]), 0.0, 0.0, 16,
                     _sorted_patches([(0, 16, 0), (0, 0, 16), (0, 16, 16)] +
                                     [(2, 16 * i, 16 * j) for j in range(4) for i in range(4)]))
    elif name == "shuffled":                                       # patch list in random order, levels interleaved
        lay = random_refined_layout(5, 7, 16, 4, 0.35)
        lay = Layout(lay.n_levels, lay.cell_width, lay.x0, lay.y0, lay.P,
                     lay.patches[np.random.default_rng(9).permutation(lay.n_patches)].copy())
    else:
        lay = random_refined_layout(int(name[4:]), 7, 16, 4, 0.35)
    with SgDisk.from_layout(lay, device=-1) as d:
        r = d.lattice_plan_check()
    assert r["available"] and r["duplicates"] == 0 and r["wrong_level"] == 0
    assert r["patches_missing_from_launched_lists"] == 0
    assert r["pairs_per_class"] == _near_pair_counts(lay)
    n_groups0 = sum((c + 7) // 8 for c in np.bincount(lay.patches[:, 0]))
    assert r["groups"][0] == n_groups0


def test_lattice_plan_absent_for_other_patch_sizes():
    lay, _ = make_config(2)                                        # P = 8: generic lattice kernel, no offset plan
    with SgDisk.from_layout(lay, device=-1) as d:
        assert not d.lattice_plan_check()["available"]


def test_shard_range_by_cost_partitions_whole_patches():
    from paper_2001_02765_b200.sharding import lattice_patch_costs, shard_range_by_cost
    lay = nested_layout(5, 64, 8.0, 16)                            # five levels: far pairs make coarse targets dearer
    costs = lattice_patch_costs(lay.patches[:, 0])
    assert len(costs) == lay.n_patches and len(set(costs)) > 1
    PP = lay.P * lay.P
    for world in (1, 2, 3, 8):
        pieces = [shard_range_by_cost(costs, PP, r, world) for r in range(world)]
        assert pieces[0][0] == 0 and sum(c for _, c in pieces) == lay.n_cells
        for (f0, c0), (f1, _) in zip(pieces, pieces[1:]):
            assert f0 + c0 == f1 and f0 % PP == 0 and c0 % PP == 0
        share = [sum(costs[f // PP:(f + c) // PP]) for f, c in pieces]
        assert max(share) - min(share) <= 2 * max(costs)           # balanced to within a patch or two


def test_bench_gpus_n_spawns_n_ranks():
    """`python bench.py --gpus 2` with no torchrun environment re-executes itself under torch.distributed.run with
    two ranks (the driver's N > 1 command must reach an N-rank run); under torchrun it does not."""
    import json
    import subprocess
    import sys
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["SG_BENCH_PRINT_SPAWN"] = "1"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1"],
                         capture_output=True, text=True, env=env, check=True).stdout
    cmd = json.loads(out.strip().splitlines()[-1])["spawn"]
    assert "torch.distributed.run" in cmd and "--nproc-per-node=2" in cmd and "127.0.0.1" in cmd
    assert cmd[-4:] == ["--gpus", "2", "--steps", "1"] and cmd[-5].endswith("bench.py")
    sys.path.insert(0, ROOT)
    import bench
    args = type("A", (), {"impl": "ours", "gpus": 2})()
    os.environ["WORLD_SIZE"] = "2"
    try:
        assert bench.spawn_command(args, []) is None               # already inside a torchrun launch
    finally:
        del os.environ["WORLD_SIZE"]
    assert bench.spawn_command(type("A", (), {"impl": "ours", "gpus": 1})(), []) is None
    assert bench.spawn_command(type("A", (), {"impl": "reference", "gpus": 4})(), []) is None


def test_lattice_plan_fill_of_the_amr_configs():
    """The numbers profiles/r2_captureA quotes for the lock-step fill of the offset walk (host replay): pairs per class
    equal the level-count products, and on cfg 4 only 61 % (same level) / 28-36 % (cross level) of the warp slots of a
    lock-step CTA have work, against 94 % on the uniform cfg 5."""
    lay, _ = make_config(4)
    with SgDisk.from_layout(lay, device=-1) as d:
        fill = d.lattice_plan_fill()
    assert [f["pairs"] for f in fill] == _near_pair_counts(lay)
    frac = [f["pairs"] / (8.0 * f["live_offsets"]) for f in fill]
    assert [round(x, 2) for x in frac] == [0.61, 0.32, 0.36, 0.32, 0.28]
    lay5, _ = make_config(5)
    with SgDisk.from_layout(lay5, device=-1) as d:
        f5 = d.lattice_plan_fill()[0]
    assert f5["pairs"] == 4096 * 4096 and round(f5["pairs"] / (8.0 * f5["live_offsets"]), 2) == 0.94
