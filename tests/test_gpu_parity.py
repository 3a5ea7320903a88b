"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json north_star's: max|dF|/max|F| <= 1e-11 and relative
L2 <= 1e-12 over both components, FP64 (the oracle side is long double)."""
import numpy as np
import pytest

import oracle
from workloads import (Layout, make_config, cell_rects, expected_counts, sample_targets, paper_ilr_layout,
                       nested_layout, d2_sigma, kuzmin_sigma)
from workloads.configs import cell_centres, _sorted_patches, uniform_layout

pytestmark = pytest.mark.gpu

TOL_MAX, TOL_L2 = 1e-11, 1e-12


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


def gpu_force(torch, lay, sigma, G=1.0, target_range=None):
    from paper_2001_02765_b200 import SgDisk
    with SgDisk.from_layout(lay, G=G, device=0) as d:
        s = torch.as_tensor(sigma, dtype=torch.float64).cuda()
        d.set_density(s)
        if target_range is not None:
            d.set_target_range(*target_range)
        Fx, Fy = d.force()
        torch.cuda.synchronize()
        return Fx.cpu().numpy(), Fy.cpu().numpy()


def oracle_force(lay, sigma, idx=None, G=1.0):
    r = cell_rects(lay)
    if idx is None:
        idx = np.arange(lay.n_cells)
    fx, fy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, G=G, precision="f80")
    return fx, fy


def errors(gx, gy, ox, oy):
    scale = max(np.abs(ox).max(), np.abs(oy).max())
    emax = max(np.abs(gx - ox).max(), np.abs(gy - oy).max()) / scale
    l2 = np.sqrt((np.sum((gx - ox) ** 2) + np.sum((gy - oy) ** 2)) / (np.sum(ox ** 2) + np.sum(oy ** 2)))
    return emax, l2


def check(gx, gy, ox, oy):
    assert np.all(np.isfinite(gx)) and np.all(np.isfinite(gy))
    emax, l2 = errors(gx, gy, ox, oy)
    assert emax <= TOL_MAX and l2 <= TOL_L2, (emax, l2)
    return emax, l2


# ------------------------------------------------------------------------------------------
# the five BASELINE.json configs
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2])
def test_small_configs_all_targets(torch_cuda, cfg):
    lay, sigma = make_config(cfg)
    assert lay.n_cells == expected_counts(cfg)["n_cells"]
    gx, gy = gpu_force(torch_cuda, lay, sigma)
    check(gx, gy, *oracle_force(lay, sigma))


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_large_configs_sampled_targets(torch_cuda, large_oracle, cfg):
    """Full-size run in the launch configuration bench.py times; oracle coverage as the configs state it (conftest:
    cfg 3 all 53,248 targets, cfg 4 4,096 stratified by level, cfg 5 4,096 seeded), every oracle value computed one
    by one from all N leaves in long double."""
    lay, sigma, idx, ox, oy = large_oracle(cfg)
    exp = expected_counts(cfg)
    assert lay.n_cells == exp["n_cells"] and lay.n_patches == exp["n_patches"]
    assert idx.size == (lay.n_cells if cfg == 3 else 4096)
    gx, gy = gpu_force(torch_cuda, lay, sigma)
    check(gx[idx], gy[idx], ox, oy)
    # properties that hold at any size: finite everywhere; Newton's third law on the uniform grid
    assert np.all(np.isfinite(gx)) and np.all(np.isfinite(gy))
    if cfg == 5:
        assert abs(np.sum(sigma * gx)) <= 1e-9 * np.sum(np.abs(sigma * gx))
        assert abs(np.sum(sigma * gy)) <= 1e-9 * np.sum(np.abs(sigma * gy))


# ------------------------------------------------------------------------------------------
# edge and degenerate cases
# ------------------------------------------------------------------------------------------
def test_single_cell_has_zero_self_force(torch_cuda):
    lay = Layout(1, np.array([0.5]), 0.0, 0.0, 1, np.array([[0, 3, 2]], dtype=np.int32))
    gx, gy = gpu_force(torch_cuda, lay, np.array([2.5]))
    # P is even in u: [[P]] of the own cell vanishes (to rounding: the four vertex terms cancel)
    assert abs(gx[0]) <= 1e-15 * 2.5 and abs(gy[0]) <= 1e-15 * 2.5


def test_zero_density_gives_zero_force(torch_cuda):
    lay, sigma = make_config(2)
    gx, gy = gpu_force(torch_cuda, lay, np.zeros_like(sigma))
    assert not gx.any() and not gy.any()


def test_fig1_unbalanced_three_level_layout(torch_cuda):
    """The paper's own 28-leaf example (Table 10): P = 1, not 2:1 balanced, coincidences
    between coarse centres and fine grid lines on both axes."""
    l0 = [(0, i, j) for j in range(4) for i in range(4) if (i, j) not in ((1, 1), (2, 2))]
    l1 = [(1, 2, 2), (1, 3, 3)] + [(1, 4 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    l2 = [(2, 4 + di, 6 + dj) for dj in (0, 1) for di in (0, 1)]
    l2 += [(2, 6 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    lay = Layout(3, np.array([0.25, 0.125, 0.0625]), 0.0, 0.0, 1, _sorted_patches(l0 + l1 + l2))
    sigma = np.random.default_rng(5).uniform(0.5, 1.5, lay.n_cells)
    gx, gy = gpu_force(torch_cuda, lay, sigma)
    check(gx, gy, *oracle_force(lay, sigma))


def test_paper_ilr_quadtree_layout(torch_cuda):
    """ILR refinement of PAPER.md:164 (reading A13), zone-wise (P = 1), D2 disk of Eq. 7."""
    lay = paper_ilr_layout(64, 3)
    x, y, _ = cell_centres(lay)
    sigma = d2_sigma(x, y, alpha=0.5)
    gx, gy = gpu_force(torch_cuda, lay, sigma)
    check(gx, gy, *oracle_force(lay, sigma))


def test_nested_levels_ragged_sizes(torch_cuda):
    """Five nested levels with P = 4: vertex count is not a multiple of the 256-vertex tile, target
    count not a multiple of the CTA's target block; many coincident grid lines."""
    lay = nested_layout(5, 32, 8.0, 4)
    x, y, _ = cell_centres(lay)
    sigma = kuzmin_sigma(x, y, a=0.3) * (1 + 0.2 * np.random.default_rng(11).uniform(-1, 1, lay.n_cells))
    gx, gy = gpu_force(torch_cuda, lay, sigma)
    check(gx, gy, *oracle_force(lay, sigma))


def test_target_range_slices_equal_full_result(torch_cuda):
    lay, sigma = make_config(2)
    fx, fy = gpu_force(torch_cuda, lay, sigma)
    n = lay.n_cells
    for first, count in ((0, 1), (1, 1000), (1001, n - 1001), (n - 1, 1), (0, n)):
        gx, gy = gpu_force(torch_cuda, lay, sigma, target_range=(first, count))
        assert gx.shape == (count,)
        # the split of the source list may differ with the range: equal up to summation order
        s = max(np.abs(fx).max(), np.abs(fy).max())
        assert np.abs(gx - fx[first:first + count]).max() <= 1e-13 * s
        assert np.abs(gy - fy[first:first + count]).max() <= 1e-13 * s
    gx, gy = gpu_force(torch_cuda, lay, sigma, target_range=(17, 0))
    assert gx.shape == (0,)


def test_deterministic_and_G_scaling(torch_cuda):
    lay, sigma = make_config(2)
    a = gpu_force(torch_cuda, lay, sigma)
    b = gpu_force(torch_cuda, lay, sigma)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])       # no atomics: bit-identical
    c = gpu_force(torch_cuda, lay, sigma, G=4.0)                              # power of two: exact
    assert np.array_equal(c[0], 4.0 * a[0]) and np.array_equal(c[1], 4.0 * a[1])


def test_patch_order_invariance(torch_cuda):
    """Permuting the patch list permutes the output; values agree to rounding (vertex order changes
    only through the cell indices in the adjacency lists)."""
    lay, sigma = make_config(2)
    PP = lay.P * lay.P
    perm = np.random.default_rng(3).permutation(lay.n_patches)
    lay2 = Layout(lay.n_levels, lay.cell_width, lay.x0, lay.y0, lay.P, lay.patches[perm].copy())
    sig2 = sigma.reshape(-1, PP)[perm].reshape(-1)
    fx, fy = gpu_force(torch_cuda, lay, sigma)
    gx, gy = gpu_force(torch_cuda, lay2, sig2)
    s = max(np.abs(fx).max(), np.abs(fy).max())
    assert np.abs(gx.reshape(-1, PP) - fx.reshape(-1, PP)[perm]).max() <= 1e-13 * s
    assert np.abs(gy.reshape(-1, PP) - fy.reshape(-1, PP)[perm]).max() <= 1e-13 * s


def test_refinement_invariance_on_gpu(torch_cuda):
    """Children inheriting the parent's sigma leave the force at unrefined targets unchanged
    (the sum over a cell's children telescopes)."""
    coarse = uniform_layout(32, -1.0, -1.0, 1 / 16, 8)
    x, y, _ = cell_centres(coarse)
    sig_c = kuzmin_sigma(x, y)
    # refine the central 2x2 patches
    keep = [tuple(p) for p in coarse.patches if not (8 <= p[1] < 24 and 8 <= p[2] < 24)]
    fine = [(1, i, j) for j in range(16, 48, 8) for i in range(16, 48, 8)]
    lay = Layout(2, np.array([1 / 16, 1 / 32]), -1.0, -1.0, 8, _sorted_patches(keep + fine))
    xf, yf, hf = cell_centres(lay)
    # sigma of each leaf = sigma of the coarse cell that contains it
    ci = np.floor((xf + 1.0) * 16).astype(int)
    cj = np.floor((yf + 1.0) * 16).astype(int)
    lut = {}
    rc = cell_rects(coarse)
    for k in range(coarse.n_cells):
        lut[(rc["kxl"][k] // 2, rc["kyd"][k] // 2)] = sig_c[k]
    sig_f = np.array([lut[(a, b)] for a, b in zip(ci, cj)])
    fx, fy = gpu_force(torch_cuda, coarse, sig_c)
    gx, gy = gpu_force(torch_cuda, lay, sig_f)
    coarse_targets = {(a, b): k for k, (a, b) in enumerate(zip(x, y))}
    s = max(np.abs(fx).max(), np.abs(fy).max())
    n_checked = 0
    for k in np.nonzero(hf == 1 / 16)[0]:
        j = coarse_targets[(xf[k], yf[k])]
        assert abs(gx[k] - fx[j]) <= 1e-12 * s and abs(gy[k] - fy[j]) <= 1e-12 * s
        n_checked += 1
    assert n_checked == 32 * 32 - 16 * 16


def test_state_errors(torch_cuda):
    from paper_2001_02765_b200 import SgDisk, SgError, binding
    lay, sigma = make_config(1)
    with SgDisk.from_layout(lay, device=0) as d:
        with pytest.raises(SgError) as e:
            d.force()
        assert e.value.code == binding.SG_ERR_STATE
        with pytest.raises(SgError):
            d.set_density(torch_cuda.zeros(7, dtype=torch_cuda.float64, device="cuda"))


def test_two_live_contexts_of_different_extent(torch_cuda):
    """Two contexts alive at once, the larger lattice (bigger log table, more dynamic shared memory) created FIRST and
    the small one after it: the opt-in shared-memory size of a kernel is a per-function, process-wide setting and must
    not shrink with the last context created.  sg_force calls interleaved, all three modes of use."""
    from paper_2001_02765_b200 import SgDisk
    big = nested_layout(4, 64, 8.0, 16)                 # extent 2048 lattice units
    xb, yb, _ = cell_centres(big)
    sig_b = kuzmin_sigma(xb, yb, a=0.3)
    small = uniform_layout(32, -1.0, -1.0, 1 / 16, 16)  # extent 64
    xs, ys, _ = cell_centres(small)
    sig_s = kuzmin_sigma(xs, ys)
    ref_b = oracle_force(big, sig_b)
    ref_s = oracle_force(small, sig_s)
    with SgDisk.from_layout(big, device=0) as db:
        tb = torch_cuda.as_tensor(sig_b).cuda()
        db.set_density(tb)
        with SgDisk.from_layout(small, device=0) as ds:
            ts = torch_cuda.as_tensor(sig_s).cuda()
            ds.set_density(ts)
            for mode in ("direct", "lattice", "direct"):
                ds.set_interaction_mode(mode)
                db.set_interaction_mode(mode)
                fs = ds.force()
                fb = db.force()
                torch_cuda.cuda.synchronize()
                check(fb[0].cpu().numpy(), fb[1].cpu().numpy(), *ref_b)
                check(fs[0].cpu().numpy(), fs[1].cpu().numpy(), *ref_s)
            # slope path of both (zero slopes: same forces), again large after small
            zs, zb = torch_cuda.zeros_like(ts), torch_cuda.zeros_like(tb)
            ds.set_density_linear(ts, zs, zs)
            db.set_density_linear(tb, zb, zb)
            fs = ds.force()
            fb = db.force()
            torch_cuda.cuda.synchronize()
            check(fb[0].cpu().numpy(), fb[1].cpu().numpy(), *ref_b)
            check(fs[0].cpu().numpy(), fs[1].cpu().numpy(), *ref_s)


def test_current_device_and_reused_context_with_poisoned_partials(torch_cuda):
    """One context, many evaluations with changing target ranges and modes: the partial-sum buffer is NaN-filled before
    every sg_force (SG_POISON_PARTIALS, conftest), so a slot no kernel writes cannot hide behind the previous call's
    value.  The library leaves the caller's current device as it was."""
    from paper_2001_02765_b200 import SgDisk
    lay = nested_layout(5, 64, 8.0, 16)                 # five levels: blocked classes + far pairs (generic kernel)
    x, y, _ = cell_centres(lay)
    sigma = kuzmin_sigma(x, y, a=0.3)
    n = lay.n_cells
    dev_before = torch_cuda.cuda.current_device()
    with SgDisk.from_layout(lay, device=0) as d:
        d.set_density(torch_cuda.as_tensor(sigma).cuda())
        d.set_interaction_mode("direct")
        fx, fy = [t.cpu().numpy() for t in d.force()]
        s = max(np.abs(fx).max(), np.abs(fy).max())
        for mode in ("lattice", "direct", "lattice"):
            d.set_interaction_mode(mode)
            for first, count in ((0, n), (0, 256), (n - 300, 300), (1000, n // 2), (0, n)):
                d.set_target_range(first, count)
                gx, gy = [t.cpu().numpy() for t in d.force()]
                assert np.all(np.isfinite(gx)) and np.all(np.isfinite(gy)), (mode, first, count)
                assert np.abs(gx - fx[first:first + count]).max() <= 1e-12 * s
                assert np.abs(gy - fy[first:first + count]).max() <= 1e-12 * s
    assert torch_cuda.cuda.current_device() == dev_before
