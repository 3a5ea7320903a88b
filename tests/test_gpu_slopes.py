"""GPU tests of the slope-term path (sg_set_density_linear):
parity with the oracle's first-order sum, and the paper's own printed tables reproduced from the GPU output."""
import numpy as np
import pytest

import oracle
from test_oracle_pins import F_D2_xy, _agree_3_digits, _norms
from workloads import (cell_rects, make_config, paper_ilr_layout, paper_vlr_layout, sample_targets, d2_sigma, d2_slopes, d22_sigma,
                       d22_slopes, nested_layout, kuzmin_sigma)
from workloads.configs import cell_centres, uniform_layout

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


def gpu_force_linear(torch, lay, sigma, dx, dy, then_zeroth=False, mode="direct"):
    from paper_2001_02765_b200 import SgDisk
    with SgDisk.from_layout(lay, device=0) as d:
        d.set_interaction_mode(mode)
        t = [torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda() for a in (sigma, dx, dy)]
        d.set_density_linear(*t)
        Fx, Fy = d.force()
        out = [Fx.cpu().numpy(), Fy.cpu().numpy()]
        if then_zeroth:
            d.set_density(t[0])
            Gx, Gy = d.force()
            out += [Gx.cpu().numpy(), Gy.cpu().numpy()]
        torch.cuda.synchronize()
        return out


def kuzmin_slopes(x, y, M=1.0, a=0.2):
    s = kuzmin_sigma(x, y, M, a)
    g = -3.0 * s / (x * x + y * y + a * a)
    return g * x, g * y


def errors(gx, gy, ox, oy):
    scale = max(np.abs(ox).max(), np.abs(oy).max())
    emax = max(np.abs(gx - ox).max(), np.abs(gy - oy).max()) / scale
    l2 = np.sqrt((np.sum((gx - ox) ** 2) + np.sum((gy - oy) ** 2)) / (np.sum(ox ** 2) + np.sum(oy ** 2)))
    return emax, l2


def test_two_level_amr_all_targets_vs_oracle(torch_cuda):
    lay, sigma = make_config(2)
    x, y, _ = cell_centres(lay)
    dx, dy = kuzmin_slopes(x, y)
    gx, gy, zx, zy = gpu_force_linear(torch_cuda, lay, sigma, dx, dy, then_zeroth=True)
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sigma, r["kxc"], r["kyc"], lay.unit, dx=dx, dy=dy)
    emax, l2 = errors(gx, gy, ox, oy)
    assert emax <= 1e-11 and l2 <= 1e-12, (emax, l2)
    # the slope terms matter (otherwise this test would pass without them) ...
    px, py, _ = oracle.force(r, sigma, r["kxc"], r["kyc"], lay.unit)
    assert np.abs(ox - px).max() > 1e-3 * np.abs(ox).max()
    # ... and sg_set_density afterwards switches back to the zeroth-order sum
    emax0, l20 = errors(zx, zy, px, py)
    assert emax0 <= 1e-11 and l20 <= 1e-12, (emax0, l20)


def test_nested_five_levels_vs_oracle(torch_cuda):
    lay = nested_layout(5, 32, 8.0, 4)
    x, y, _ = cell_centres(lay)
    sigma = kuzmin_sigma(x, y, a=0.7)
    dx, dy = kuzmin_slopes(x, y, a=0.7)
    gx, gy = gpu_force_linear(torch_cuda, lay, sigma, dx, dy)
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sigma, r["kxc"], r["kyc"], lay.unit, dx=dx, dy=dy)
    emax, l2 = errors(gx, gy, ox, oy)
    assert emax <= 1e-11 and l2 <= 1e-12, (emax, l2)


@pytest.mark.parametrize("mode", ["direct", "lattice"])
def test_galactic_config_sampled_vs_oracle(torch_cuda, mode):
    """cfg 3 (53,248 leaves, 4 levels, lattice extent 2048) with centred-difference-free analytic slopes of a
    smooth bump; oracle on 1024 sampled targets.  lattice: three-plane function lattices for the pairs <= 2 levels
    apart, direct slope sums for the level 0 <-> level 3 pairs (patch_far_kernel<true>)."""
    lay, _ = make_config(3)
    x, y, _ = cell_centres(lay)
    s2 = 4.0 ** 2
    sigma = np.exp(-(x * x + y * y) / (2 * s2))
    dx, dy = -x / s2 * sigma, -y / s2 * sigma
    gx, gy = gpu_force_linear(torch_cuda, lay, sigma, dx, dy, mode=mode)
    idx = sample_targets(lay, 1024, 77)
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, dx=dx, dy=dy)
    emax, l2 = errors(gx[idx], gy[idx], ox, oy)
    assert emax <= 1e-11 and l2 <= 1e-12, (emax, l2)


# ------------------------------------------------------------------------------------------
# slope path in lattice mode (SURVEY.md 8 f1 x f2): same tolerances as the direct slope kernel
# ------------------------------------------------------------------------------------------
def _lattice_slopes_vs_oracle(torch, lay, sigma, dx, dy, idx=None):
    from paper_2001_02765_b200 import SgDisk
    if idx is None:
        idx = np.arange(lay.n_cells)
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, dx=dx, dy=dy)
    with SgDisk.from_layout(lay, device=0) as d:
        t = [torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda() for a in (sigma, dx, dy)]
        d.set_interaction_mode("lattice")
        d.set_density_linear(*t)
        assert d.kernel_model()["fp64_instr_per_pair"] == 6.0       # the lattice slope path is the one that runs
        Fx, Fy = d.force()
        d.set_interaction_mode("direct")
        Dx, Dy = d.force()
        d.set_interaction_mode("lattice")
        Gx, Gy = d.force()                                           # again, after a mode change: bit-identical
        torch.cuda.synchronize()
        assert torch.equal(Fx, Gx) and torch.equal(Fy, Gy)
    gx, gy = Fx.cpu().numpy(), Fy.cpu().numpy()
    assert np.all(np.isfinite(gx)) and np.all(np.isfinite(gy))
    emax, l2 = errors(gx[idx], gy[idx], ox, oy)
    assert emax <= 1e-11 and l2 <= 1e-12, (emax, l2)
    s = max(np.abs(ox).max(), np.abs(oy).max())
    assert max(np.abs(gx - Dx.cpu().numpy()).max(), np.abs(gy - Dy.cpu().numpy()).max()) <= 1e-11 * s
    return gx, gy


def test_lattice_slopes_two_level_patches_all_targets(torch_cuda):
    """cfg-2-shaped two-level AMR with 16 x 16 patches (coarse ring + refined centre), noisy sigma, Taylor slopes of the
    smooth profile: all 12,288 targets vs the oracle's first-order sum."""
    lay = nested_layout(2, 128, 1.0, 16)
    x, y, _ = cell_centres(lay)
    sigma = kuzmin_sigma(x, y) * (1 + 0.05 * np.random.default_rng(1).uniform(-1, 1, lay.n_cells))
    _lattice_slopes_vs_oracle(torch_cuda, lay, sigma, *kuzmin_slopes(x, y))


def test_lattice_slopes_five_nested_levels_all_targets(torch_cuda):
    """Five nested levels, P = 16: every pair class by function lattices and the pairs three and four levels apart by
    the direct slope sum (patch_far_kernel<true>)."""
    lay = nested_layout(5, 64, 8.0, 16)
    x, y, _ = cell_centres(lay)
    _lattice_slopes_vs_oracle(torch_cuda, lay, kuzmin_sigma(x, y, a=0.7), *kuzmin_slopes(x, y, a=0.7))


def test_lattice_slopes_irregular_hierarchy(torch_cuda):
    """Ragged three-level hierarchy with holes (workloads.random_refined_layout), all targets."""
    from workloads import random_refined_layout
    lay = random_refined_layout(3, 6, 16, 3, 0.3)
    x, y, _ = cell_centres(lay)
    _lattice_slopes_vs_oracle(torch_cuda, lay, kuzmin_sigma(x, y, a=0.4), *kuzmin_slopes(x, y, a=0.4))


def test_lattice_slopes_config4_sampled(torch_cuda):
    """BASELINE.json config 4 (three levels, 448,768 leaves) with the slopes of its own profile taken by centred
    differences of the formula; 512 stratified targets.  The profile's tanh tapers change sigma by its own size over a
    few cells, so the vertex weights a_v, c_v (second differences of the slopes) are large.  The lattice slope path uses
    own-cell (neutral) per-patch weights at every extent, with which it holds the same gates as the direct slope kernel
    (owned 16 x 16 weights measured rel. L2 1.7e-12 here: DESIGN.md 8)."""
    from workloads.configs import _ppd_sigma
    lay, sigma = make_config(4)
    x, y, h = cell_centres(lay)
    e = 1e-4
    dx = (_ppd_sigma(x + e, y) - _ppd_sigma(x - e, y)) / (2 * e)
    dy = (_ppd_sigma(x, y + e) - _ppd_sigma(x, y - e)) / (2 * e)
    _lattice_slopes_vs_oracle(torch_cuda, lay, sigma, dx, dy, idx=sample_targets(lay, 512, 4004))


def test_random_slopes_conditioning(torch_cuda):
    """Uncorrelated random slopes are not a Taylor expansion of any field; the vertex regrouping then cancels
    O(extent/h) leading digits.  Parity still holds to 1e-9."""
    lay, sigma = make_config(2)
    rng = np.random.default_rng(4)
    dx, dy = rng.normal(size=lay.n_cells) * 3.0, rng.normal(size=lay.n_cells) * 3.0
    gx, gy = gpu_force_linear(torch_cuda, lay, sigma, dx, dy)
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sigma, r["kxc"], r["kyc"], lay.unit, dx=dx, dy=dy)
    emax, l2 = errors(gx, gy, ox, oy)
    assert emax <= 1e-9 and l2 <= 1e-9, (emax, l2)


_d2_uniform_cache = {}


def test_paper_table1_row_1024_in_lattice_mode(torch_cuda, golden):
    """PAPER.md:152 (Table 1, N_k = 1024) from the lattice-mode slope path: the paper's full second-order method on its
    own 1024^2 grid in ~0.55 s (171 s on the paper's P100)."""
    row = [r for r in golden("paper_table1_D2_uniform.txt") if int(r[0]) == 1024][0]
    lay = uniform_layout(1024, -1.0, -1.0, 2 / 1024, 16)
    x, y, h = cell_centres(lay)
    Fx, Fy = gpu_force_linear(torch_cuda, lay, d2_sigma(x, y, 0.5), *d2_slopes(x, y, 0.5), mode="lattice")
    ax, ay = F_D2_xy(x, y, 0.5)
    R = np.hypot(x, y)
    eR = (Fx * x + Fy * y) / R - (ax * x + ay * y) / R
    got = list(_norms(Fx - ax, h ** 2)) + list(_norms(eR, h ** 2))
    for g, p in zip(got, row[1:]):
        assert _agree_3_digits(g, p), (got, row)


def d2_uniform_gpu(torch, Nk):
    """The paper's D2 test on the uniform Nk x Nk grid with exact Taylor slopes (R10), slope kernel; the
    Nk = 2048 run (4.2 M cells, 1.8e13 pairs, ~40 s) is shared by the Table 1 row and the oracle parity check."""
    if Nk not in _d2_uniform_cache:
        lay = uniform_layout(Nk, -1.0, -1.0, 2 / Nk, 16)
        x, y, h = cell_centres(lay)
        sig = d2_sigma(x, y, 0.5)
        dx, dy = d2_slopes(x, y, 0.5)
        Fx, Fy = gpu_force_linear(torch, lay, sig, dx, dy)
        _d2_uniform_cache.clear()                              # keep one grid at a time (2048^2: 5 x 34 MB)
        _d2_uniform_cache[Nk] = (lay, x, y, h, sig, dx, dy, Fx, Fy)
    return _d2_uniform_cache[Nk]


def test_slope_kernel_vs_oracle_at_2048_squared(torch_cuda):
    """The slope kernel against the oracle's first-order sum on 256 seeded targets of the 2048^2 D2 grid (PAPER.md:153,
    the largest grid of Table 1): excludes GPU drift at 4.2 M cells as the source of the 1.4 % by which the L1/L2
    columns of that row differ from print (test_paper_table1_D2_uniform_on_gpu below)."""
    lay, x, y, h, sig, dx, dy, Fx, Fy = d2_uniform_gpu(torch_cuda, 2048)
    idx = np.sort(np.random.default_rng(2048).choice(lay.n_cells, size=256, replace=False))
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sig, r["kxc"][idx], r["kyc"][idx], lay.unit, dx=dx, dy=dy)
    emax, l2 = errors(Fx[idx], Fy[idx], ox, oy)
    assert emax <= 1e-11 and l2 <= 1e-12, (emax, l2)


@pytest.mark.parametrize("Nk", [2048, 128, 256, 512, 1024])
def test_paper_table1_D2_uniform_on_gpu(torch_cuda, golden, Nk):
    """PAPER.md:147-153 Table 1, all six columns, from the GPU force (the oracle only reaches Nk = 256 in the CPU
    suite's time budget; Nk = 1024 is 1.1e12 pairs)."""
    row = [r for r in golden("paper_table1_D2_uniform.txt") if int(r[0]) == Nk][0]
    lay, x, y, h, sig, dx, dy, Fx, Fy = d2_uniform_gpu(torch_cuda, Nk)
    ax, ay = F_D2_xy(x, y, 0.5)
    R = np.hypot(x, y)
    eR = (Fx * x + Fy * y) / R - (ax * x + ay * y) / R
    A = h ** 2
    got = list(_norms(Fx - ax, A)) + list(_norms(eR, A))
    for g, p in zip(got, row[1:]):
        if Nk == 2048:
            # 4.2 M cells, 1.8e13 pairs: the L-infinity columns agree to the printed digits, the 1- and 2-norms
            # to 1.4 % (3.60e-6 vs the printed 3.55e-6).  The GPU sum itself agrees with the long-double oracle to
            # 1e-11 at this size (test_slope_kernel_vs_oracle_at_2048_squared), so the difference is the paper's:
            # its primitive -ln(v+r) cancels (R4).  This row is held to 2 %.
            assert abs(g - float(p)) <= 0.02 * float(p), (got, row)
        else:
            assert _agree_3_digits(g, p), (got, row)


def test_paper_table2_D22_uniform_on_gpu(torch_cuda, golden):
    row = [r for r in golden("paper_table2_D22_uniform.txt") if int(r[0]) == 128][0]
    lay = uniform_layout(128, -1.0, -1.0, 2 / 128, 16)
    x, y, h = cell_centres(lay)
    Fx, Fy = gpu_force_linear(torch_cuda, lay, d22_sigma(x, y), *d22_slopes(x, y))
    a1 = F_D2_xy(x, y, 0.4, 0.0, 0.5)
    a2 = F_D2_xy(x, y, 0.4, 0.0, -0.5)
    A = h ** 2
    got = list(_norms(Fx - a1[0] - a2[0], A)) + list(_norms(Fy - a1[1] - a2[1], A))
    for g, p in zip(got, row[1:]):
        assert _agree_3_digits(g, p), (got, row)


def _paper_mode(Nk):
    """The paper's zone-wise quadtrees (P = 1): direct slope kernel up to N_k = 512, from N_k = 1024 the regrouped
    lattice mode (the leaves packed into padded 16 x 16 blocks, three-plane function lattices)."""
    return "lattice" if Nk >= 1024 else "direct"


@pytest.mark.parametrize("L,Nk", [(2, 128), (2, 256), (3, 128), (3, 256), (2, 512), (3, 512), (2, 1024), (3, 1024),
                                  (2, 2048), (3, 2048)])
def test_paper_table3_ILR_Linf_on_gpu(torch_cuda, golden, L, Nk):
    """PAPER.md:203-220 Table 3 L-infinity columns on the paper's zone-wise quadtree (P = 1).  The N_k = 1024 and
    2048 layouts (1,172,176 / 1,419,424 / 4,688,632 / 5,677,336 leaves) are Table 8's workloads (PAPER.md:350-357:
    671 s, 1,050 s, 1.06e4 s and 1.62e4 s per evaluation on the paper's P100)."""
    row = [r for r in golden("paper_table3_ILR_Linf.txt") if int(r[0]) == L and int(r[1]) == Nk][0]
    lay = paper_ilr_layout(Nk, L, "D2")
    leaves = {(2, 1024): 1172176, (3, 1024): 1419424, (2, 2048): 4688632, (3, 2048): 5677336}   # Table 8
    assert lay.n_cells == leaves.get((L, Nk), lay.n_cells)
    x, y, h = cell_centres(lay)
    Fx, Fy = gpu_force_linear(torch_cuda, lay, d2_sigma(x, y, 0.5), *d2_slopes(x, y, 0.5), mode=_paper_mode(Nk))
    ax, ay = F_D2_xy(x, y, 0.5)
    R = np.hypot(x, y)
    assert _agree_3_digits(np.abs(Fx - ax).max(), row[2])
    assert _agree_3_digits(np.abs((Fx * x + Fy * y) / R - (ax * x + ay * y) / R).max(), row[3])


@pytest.mark.parametrize("L,Nk", [(2, 128), (3, 128), (2, 256), (3, 256), (2, 512), (3, 512), (2, 1024), (3, 1024)])
def test_paper_table5_VLR_Linf_on_gpu(torch_cuda, golden, L, Nk):
    """PAPER.md:274-291 Table 5 L-infinity columns on the paper's VLR quadtrees (P = 1; Table 9's workloads)."""
    row = [r for r in golden("paper_table5_VLR_Linf.txt") if int(r[0]) == L and int(r[1]) == Nk][0]
    lay = paper_vlr_layout(Nk, L, "D2")
    x, y, h = cell_centres(lay)
    Fx, Fy = gpu_force_linear(torch_cuda, lay, d2_sigma(x, y, 0.5), *d2_slopes(x, y, 0.5), mode=_paper_mode(Nk))
    ax, ay = F_D2_xy(x, y, 0.5)
    R = np.hypot(x, y)
    if not row[2].endswith("?"):                                   # see the fixture's header for the one misprint
        assert _agree_3_digits(np.abs(Fx - ax).max(), row[2])
    assert _agree_3_digits(np.abs((Fx * x + Fy * y) / R - (ax * x + ay * y) / R).max(), row[3])


@pytest.mark.parametrize("rule,L,Nk", [(r, L, Nk) for r in ("ILR", "VLR") for (L, Nk) in
                                        [(2, 128), (3, 128), (2, 256), (3, 256), (2, 512), (3, 512), (2, 1024), (3, 1024)]]
                         + [("ILR", 2, 2048), ("ILR", 3, 2048)])
def test_paper_tables4_6_D22_Linf_on_gpu(torch_cuda, golden, rule, L, Nk):
    """PAPER.md:235-252 Table 4 (ILR, incl. the N_k = 2048 rows :241, :252; AMR(2, D22)-2048 has the 4,984,672 leaves
    of Table 8) and :303-320 Table 6 (VLR), double disk, L-infinity of the x and y errors."""
    row = [r for r in golden("paper_table4_6_D22_Linf.txt") if r[0] == rule and int(r[1]) == L and int(r[2]) == Nk][0]
    lay = (paper_ilr_layout if rule == "ILR" else paper_vlr_layout)(Nk, L, "D22")
    if (rule, L, Nk) == ("ILR", 2, 2048):
        assert lay.n_cells == 4984672
    x, y, h = cell_centres(lay)
    sig, (sx, sy) = d22_sigma(x, y), d22_slopes(x, y)
    Fx, Fy = gpu_force_linear(torch_cuda, lay, sig, sx, sy, mode=_paper_mode(Nk))
    a1 = F_D2_xy(x, y, 0.4, 0.0, 0.5)
    a2 = F_D2_xy(x, y, 0.4, 0.0, -0.5)
    ex, ey = Fx - a1[0] - a2[0], Fy - a1[1] - a2[1]
    if Nk == 2048:
        # the largest layouts of the paper (5.0 M and ~6 M leaves).  Three of the four printed L-infinity values of the
        # two N_k = 2048 rows are reproduced to the printed digits; AMR(3, D22) L_x,inf comes out 2.441e-5 against the
        # printed 2.46E-05 (0.8 %).  The GPU sum itself is checked here against the long-double oracle at the two
        # targets that carry the maxima plus 22 seeded ones, so the difference is not this implementation's: like the
        # 1.4 % of Table 1's N_k = 2048 row it is attributed to the paper's cancelling primitive (R4), and
        # the N_k = 2048 rows are held to 1 %.
        # (On lattices of more than 4,096 units the slope path takes own-cell per-patch weights, sg_api.cu: with owned
        # weights the rounding error of these two layouts was 1.4e-11.)
        idx = np.unique(np.concatenate([[np.argmax(np.abs(ex)), np.argmax(np.abs(ey))],
                                        np.random.default_rng(2048 + L).choice(lay.n_cells, 22, replace=False)]))
        r = cell_rects(lay)
        ox, oy, _ = oracle.force(r, sig, r["kxc"][idx], r["kyc"][idx], lay.unit, dx=sx, dy=sy)
        emax, l2 = errors(Fx[idx], Fy[idx], ox, oy)
        assert emax <= 1e-11, (emax, l2)
    for got, printed in ((np.abs(ex).max(), row[3]), (np.abs(ey).max(), row[4])):
        if not printed.endswith("?"):                              # see the fixture's header
            if Nk == 2048:
                assert abs(got - float(printed)) <= 0.01 * float(printed), (got, row)
            else:
                assert _agree_3_digits(got, printed), (got, row)


@pytest.mark.parametrize("Nk,bound_owned,bound_neutral", [(256, 5e-13, 5e-13), (512, 3e-12, 8e-13), (1024, None, 2e-12)])
def test_slope_path_rounding_vs_lattice_extent(torch_cuda, monkeypatch, Nk, bound_owned, bound_neutral):
    """The table of DESIGN.md section 8, reproducibly: rounding error of the slope path in lattice mode against the
    long-double oracle on the paper's AMR(3, D22) quadtrees (48 seeded targets), with own-cell ("neutral") per-patch
    weights -- what the library uses on the slope path at every extent (measured 9.2e-14, 1.5e-13, 3.9e-13) -- and with
    the owned 16 x 16 weights of round 2 (test aid SG_LATTICE_OWNED_SLOPE_WEIGHTS, lattices of up to 4,096 units = N_k
    512 here; measured 1.4e-13, 8.9e-13).  The bounds leave a factor ~3-5 over the measured values; all are far inside
    the 1e-11 gate."""
    from paper_2001_02765_b200 import SgDisk
    lay = paper_ilr_layout(Nk, 3, "D22")
    x, y, _ = cell_centres(lay)
    sig, (sx, sy) = d22_sigma(x, y), d22_slopes(x, y)
    idx = np.sort(np.random.default_rng(1).choice(lay.n_cells, 48, replace=False))
    r = cell_rects(lay)
    ox, oy, _ = oracle.force(r, sig, r["kxc"][idx], r["kyc"][idx], lay.unit, dx=sx, dy=sy)

    def run():
        with SgDisk.from_layout(lay, device=0) as d:
            d.set_interaction_mode("lattice")
            d.set_density_linear(*[torch_cuda.as_tensor(a).cuda() for a in (sig, sx, sy)])
            Fx, Fy = d.force()
            torch_cuda.cuda.synchronize()
            return errors(Fx.cpu().numpy()[idx], Fy.cpu().numpy()[idx], ox, oy)[0]
    assert run() <= bound_neutral                   # the default
    if bound_owned is not None:                     # lattice extent <= 4,096: the owned weights can be brought back
        monkeypatch.setenv("SG_LATTICE_OWNED_SLOPE_WEIGHTS", "1")
        assert run() <= bound_owned
