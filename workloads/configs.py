"""Layouts and densities for the five BASELINE.json configs and the paper's own grids.

Conventions (shared with include/sg_disk.h, restated, not imported):
  * level 0 is the coarsest; ``cell_width[l+1] == cell_width[l] / 2``;
  * a *patch* is ``P x P`` leaf cells of one level; ``(level, i0, j0)`` is the index of its
    lower-left cell on that level's lattice, counted from the domain origin ``(x0, y0)``;
  * only leaf patches are listed ("restricted to the leaf nodes");
  * cell order is ``[patch][j][i]`` (i = x fastest), patches sorted by (level, j0, i0);
  * the integer lattice unit is half the finest cell width, so cell edges are even multiples
    of ``2**(n_levels-1-level)`` and every cell centre is an integer as well.

Nothing here evaluates the force kernel; it only builds rectangles and samples sigma.
"""
from __future__ import annotations

import dataclasses
import math
import numpy as np

CONFIG_NAMES = {
    1: "cfg1_uniform64_kuzmin",
    2: "cfg2_two_level_7168",
    3: "cfg3_galactic_4level_53248",
    4: "cfg4_protoplanetary_cap2",
    5: "cfg5_uniform1024_kuzmin",
}


@dataclasses.dataclass
class Layout:
    n_levels: int
    cell_width: np.ndarray      # float64 [n_levels]
    x0: float
    y0: float
    P: int
    patches: np.ndarray         # int32 [n_patches, 3] = (level, i0, j0), sorted (level, j0, i0)

    @property
    def n_patches(self) -> int:
        return int(self.patches.shape[0])

    @property
    def n_cells(self) -> int:
        return self.n_patches * self.P * self.P

    @property
    def unit(self) -> float:
        """Physical length of one lattice unit (half the finest cell width)."""
        return float(self.cell_width[-1]) / 2.0


def _sorted_patches(rows) -> np.ndarray:
    a = np.asarray(sorted(rows, key=lambda r: (r[0], r[2], r[1])), dtype=np.int32).reshape(-1, 3)
    return a


def cell_rects(lay: Layout):
    """Expand the patch list into per-cell integer rectangles in library cell order.

    Returns dict of int64 arrays ``kxl, kxr, kyd, kyu, kxc, kyc, level`` (lattice units).
    """
    P = lay.P
    lev = lay.patches[:, 0].astype(np.int64)
    cw = (2 << (lay.n_levels - 1 - lev)).astype(np.int64)          # cell width in lattice units
    ii = np.arange(P, dtype=np.int64)
    # [patch, j, i]
    kxl = (lay.patches[:, 1].astype(np.int64)[:, None, None] + ii[None, None, :]) * cw[:, None, None]
    kyd = (lay.patches[:, 2].astype(np.int64)[:, None, None] + ii[None, :, None]) * cw[:, None, None]
    kxl = np.broadcast_to(kxl, (lay.n_patches, P, P)).reshape(-1)
    kyd = np.broadcast_to(kyd, (lay.n_patches, P, P)).reshape(-1)
    cwc = np.repeat(cw, P * P)
    return dict(kxl=kxl.copy(), kxr=kxl + cwc, kyd=kyd.copy(), kyu=kyd + cwc,
                kxc=kxl + cwc // 2, kyc=kyd + cwc // 2, level=np.repeat(lev, P * P))


def cell_centres(lay: Layout):
    r = cell_rects(lay)
    u = lay.unit
    return lay.x0 + r["kxc"] * u, lay.y0 + r["kyc"] * u, (r["kxr"] - r["kxl"]) * u


# ----------------------------------------------------------------------------------------
# densities
# ----------------------------------------------------------------------------------------
def kuzmin_sigma(x, y, M=1.0, a=0.2):
    R2 = x * x + y * y
    return a * M / (2.0 * np.pi * (R2 + a * a) ** 1.5)


def _spiral_sigma(x, y):
    R = np.maximum(np.hypot(x, y), 0.05)
    th = np.arctan2(y, x)
    return np.exp(-R / 3.0) * (1.0 + 0.1 * np.cos(2.0 * th - 2.0 * np.log(R) / math.tan(math.radians(15.0))))


def _ppd_sigma(x, y):
    R = np.hypot(x, y)
    th = np.arctan2(y, x)
    t_in = 0.5 * (1.0 + np.tanh((R - 0.1) / 0.02))
    t_out = 0.5 * (1.0 - np.tanh((R - 1.0) / 0.02))
    return (t_in * t_out / np.maximum(R, 0.05)
            + 0.5 * np.exp(-((R - 0.5) ** 2 / 0.03 ** 2 + (th - np.pi / 4) ** 2 / 0.3 ** 2)))


def d2_sigma(x, y, alpha=0.5, sigma0=1.0, xc=0.0, yc=0.0):
    """PAPER.md:122 Eq. 7 (input density only)."""
    s = 1.0 - ((x - xc) ** 2 + (y - yc) ** 2) / alpha ** 2
    return sigma0 * np.where(s > 0, np.abs(s) ** 1.5, 0.0)


def d2_slopes(x, y, alpha=0.5, sigma0=1.0, xc=0.0, yc=0.0):
    """Exact d(sigma)/dx, d(sigma)/dy of Eq. 7 at the point (Taylor coefficients of Eq. 6)."""
    s = 1.0 - ((x - xc) ** 2 + (y - yc) ** 2) / alpha ** 2
    g = np.where(s > 0, -3.0 * sigma0 * np.sqrt(np.abs(s)) / alpha ** 2, 0.0)
    return g * (x - xc), g * (y - yc)


def d22_sigma(x, y, alpha=0.4):
    return d2_sigma(x, y, alpha, 1.0, 0.0, 0.5) + d2_sigma(x, y, alpha, 1.0, 0.0, -0.5)


def d22_slopes(x, y, alpha=0.4):
    a = d2_slopes(x, y, alpha, 1.0, 0.0, 0.5)
    b = d2_slopes(x, y, alpha, 1.0, 0.0, -0.5)
    return a[0] + b[0], a[1] + b[1]


# ----------------------------------------------------------------------------------------
# layouts
# ----------------------------------------------------------------------------------------
def uniform_layout(n: int, x0: float, y0: float, h: float, P: int) -> Layout:
    assert n % P == 0
    rows = [(0, i, j) for j in range(0, n, P) for i in range(0, n, P)]
    return Layout(1, np.array([h]), x0, y0, P, _sorted_patches(rows))


def nested_layout(n_levels: int, n: int, half_extent: float, P: int) -> Layout:
    """Concentric nested grid: every level is an n x n-cell square centred on the origin, level
    l covering |x|,|y| <= half_extent / 2**l, with its central (n/2)^2 replaced by level l+1."""
    assert n % (2 * P) == 0 and (n // 4) % P == 0
    h0 = 2.0 * half_extent / n
    rows = []
    for l in range(n_levels):
        c = (n // 2) * (1 << l)                 # lattice index of the origin on level l
        lo, hi = c - n // 2, c + n // 2
        rlo, rhi = c - n // 4, c + n // 4
        for j in range(lo, hi, P):
            for i in range(lo, hi, P):
                inside = (rlo <= i < rhi) and (rlo <= j < rhi)
                if inside and l < n_levels - 1:
                    continue
                rows.append((l, i, j))
    return Layout(n_levels, h0 / 2.0 ** np.arange(n_levels), -half_extent, -half_extent, P,
                  _sorted_patches(rows))


def random_refined_layout(seed: int, n0: int, P: int, n_levels: int, frac: float, half_extent: float = 1.0) -> Layout:
    """Irregular hierarchy for edge-case tests: an n0 x n0-patch base grid; on every level a seeded random fraction
    `frac` of the leaf patches is replaced by its four children.  No 2:1 balancing, ragged level shapes, patches of
    every parity, levels with holes."""
    rng = np.random.default_rng(seed)
    leaves = [(0, i * P, j * P) for j in range(n0) for i in range(n0)]
    for l in range(n_levels - 1):
        nxt = []
        for (lv, i0, j0) in leaves:
            if lv == l and rng.uniform() < frac:
                nxt += [(l + 1, 2 * i0 + a * P, 2 * j0 + b * P) for b in (0, 1) for a in (0, 1)]
            else:
                nxt.append((lv, i0, j0))
        leaves = nxt
    h0 = 2.0 * half_extent / (n0 * P)
    return Layout(n_levels, h0 / 2.0 ** np.arange(n_levels), -half_extent, -half_extent, P, _sorted_patches(leaves))


def _cfg2_layout() -> Layout:
    rows = []
    for j in range(0, 64, 8):
        for i in range(0, 64, 8):
            if 16 <= i < 48 and 16 <= j < 48:
                continue
            rows.append((0, i, j))
    for j in range(32, 96, 8):
        for i in range(32, 96, 8):
            rows.append((1, i, j))
    return Layout(2, np.array([1 / 32, 1 / 64]), -1.0, -1.0, 8, _sorted_patches(rows))


def _gradient_refined_layout(sigma_fn, n0: int, x0: float, y0: float, h0: float, P: int,
                             max_level: int, thresh: float = 0.05, floor: float = 1e-6) -> Layout:
    """Patch-wise gradient-driven refinement, then 2:1 balance across faces and corners.

    A leaf patch of level l is refined (replaced by its 4 children on level l+1) iff the max over
    its cells of |grad sigma| * h_l / max(sigma, floor) exceeds ``thresh``; grad by centred
    differences of cell-centre samples with the halo sampled from the formula.
    """
    npatch0 = n0 // P
    leaves = {(0, pi, pj) for pj in range(npatch0) for pi in range(npatch0)}   # patch indices (i0/P)

    def wants(l, pi, pj):
        h = h0 / 2 ** l
        i = np.arange(-1, P + 1)
        xc = x0 + (pi * P + i + 0.5) * h
        yc = y0 + (pj * P + i + 0.5) * h
        X, Y = np.meshgrid(xc, yc, indexing="xy")
        s = sigma_fn(X, Y)
        gx = (s[1:-1, 2:] - s[1:-1, :-2]) / (2 * h)
        gy = (s[2:, 1:-1] - s[:-2, 1:-1]) / (2 * h)
        crit = np.hypot(gx, gy) * h / np.maximum(s[1:-1, 1:-1], floor)
        return bool(crit.max() > thresh)

    def refine(key):
        l, pi, pj = key
        leaves.discard(key)
        for dj in (0, 1):
            for di in (0, 1):
                leaves.add((l + 1, 2 * pi + di, 2 * pj + dj))

    for l in range(max_level):
        for key in sorted(k for k in leaves if k[0] == l):
            if wants(*key):
                refine(key)

    def covering_leaf(l, pi, pj):
        """Leaf that covers patch-index (pi,pj) of level l, looking at l and coarser."""
        while l >= 0:
            if (l, pi, pj) in leaves:
                return (l, pi, pj)
            l, pi, pj = l - 1, pi >> 1, pj >> 1
        return None

    changed = True
    while changed:
        changed = False
        for key in sorted(leaves, key=lambda k: -k[0]):
            if key not in leaves:
                continue
            l, pi, pj = key
            if l < 2:
                continue
            nmax = npatch0 << l
            for dj in (-1, 0, 1):
                for di in (-1, 0, 1):
                    qi, qj = pi + di, pj + dj
                    if (di == 0 and dj == 0) or not (0 <= qi < nmax and 0 <= qj < nmax):
                        continue
                    c = covering_leaf(l, qi, qj)
                    if c is not None and c[0] < l - 1:
                        refine(c)
                        changed = True
    rows = [(l, pi * P, pj * P) for (l, pi, pj) in leaves]
    nl = max(r[0] for r in rows) + 1
    return Layout(nl, h0 / 2.0 ** np.arange(nl), x0, y0, P, _sorted_patches(rows))


# frozen facts about each layout, asserted by the tests and bench
_EXPECTED = {
    1: dict(n_patches=16, n_cells=4096),
    2: dict(n_patches=112, n_cells=7168),
    3: dict(n_patches=208, n_cells=53248),
    4: dict(n_patches=1753, n_cells=448768, patches_per_level=(93, 316, 1344)),
    5: dict(n_patches=4096, n_cells=1048576),
}


def expected_counts(cfg: int):
    return _EXPECTED.get(cfg)


def make_config(cfg: int):
    """Return (Layout, sigma[n_cells] float64 in library cell order) for BASELINE.json config cfg."""
    if cfg == 1:
        lay = uniform_layout(64, -1.0, -1.0, 1 / 32, 16)
        x, y, _ = cell_centres(lay)
        return lay, kuzmin_sigma(x, y)
    if cfg == 2:
        lay = _cfg2_layout()
        x, y, _ = cell_centres(lay)
        xi = np.random.default_rng(1).uniform(-1.0, 1.0, lay.n_cells)
        return lay, kuzmin_sigma(x, y) * (1.0 + 0.05 * xi)
    if cfg == 3:
        lay = nested_layout(4, 128, 16.0, 16)
        x, y, _ = cell_centres(lay)
        return lay, _spiral_sigma(x, y)
    if cfg == 4:
        lay = _gradient_refined_layout(_ppd_sigma, 256, -1.2, -1.2, 2.4 / 256, 16, max_level=2)
        x, y, _ = cell_centres(lay)
        return lay, _ppd_sigma(x, y)
    if cfg == 5:
        lay = uniform_layout(1024, -1.0, -1.0, 1 / 512, 16)
        x, y, _ = cell_centres(lay)
        xi = np.random.default_rng(7).uniform(-1.0, 1.0, lay.n_cells)
        return lay, kuzmin_sigma(x, y) * (1.0 + 0.01 * xi)
    raise ValueError(f"unknown config {cfg}")


def make_config4_variant(max_level: int):
    """BASELINE.json config 4 with another level cap (R14: the frozen config uses cap 2 = 448,768 leaves;
    cap 3 gives 1,342,720 leaves on four levels, the literal cap 5 gives 12,150,016 on six)."""
    lay = _gradient_refined_layout(_ppd_sigma, 256, -1.2, -1.2, 2.4 / 256, 16, max_level=max_level)
    x, y, _ = cell_centres(lay)
    return lay, _ppd_sigma(x, y)


def sample_targets(lay: Layout, n: int, seed: int) -> np.ndarray:
    """n distinct cell indices, stratified by level (equal share per level, remainder to the
    finest), drawn without replacement with default_rng(seed)."""
    rng = np.random.default_rng(seed)
    lev = np.repeat(lay.patches[:, 0], lay.P * lay.P)
    levels = np.unique(lev)
    if n >= lay.n_cells:
        return np.arange(lay.n_cells, dtype=np.int64)
    share = n // len(levels)
    out = []
    for k, l in enumerate(levels):
        idx = np.nonzero(lev == l)[0]
        want = share if k < len(levels) - 1 else n - share * (len(levels) - 1)
        want = min(want, idx.size)
        out.append(rng.choice(idx, size=want, replace=False))
    return np.sort(np.concatenate(out)).astype(np.int64)


# ----------------------------------------------------------------------------------------
# the paper's own grids (zone-wise quadtree = patches with P = 1)
# ----------------------------------------------------------------------------------------
def _paper_band_layout(Nk: int, L: int, centres, alpha: float, band_of_level) -> Layout:
    """Level-1 (paper numbering) uniform Nk x Nk zones on [-1,1]^2; a zone of paper-level m is
    refined iff | R_c - alpha | < band_of_level(m+1) with R_c measured from the nearest disk centre.
    Reading A13/A14 of SURVEY.md section 8(c), pinned against the zone counts of Tables 8 and 9."""
    h1 = 2.0 / Nk
    jj, ii = np.meshgrid(np.arange(Nk, dtype=np.int64), np.arange(Nk, dtype=np.int64), indexing="ij")
    arr = np.stack([np.zeros(Nk * Nk, dtype=np.int64), ii.reshape(-1), jj.reshape(-1)], axis=1)   # (level, i, j)
    leaves = []
    for m in range(1, L + 1):                       # paper level m == our level m-1
        l = m - 1
        h = h1 / 2 ** l
        if m == L:
            leaves.append(arr)
            break
        xc = -1.0 + (arr[:, 1] + 0.5) * h
        yc = -1.0 + (arr[:, 2] + 0.5) * h
        Rc = np.min([np.hypot(xc - cx, yc - cy) for (cx, cy) in centres], axis=0)
        ref = np.abs(Rc - alpha) < band_of_level(m + 1)
        leaves.append(arr[~ref])
        a = arr[ref]
        # children in the order (dj, di) = (0,0), (0,1), (1,0), (1,1) of every refined zone
        kids = np.empty((a.shape[0], 4, 3), dtype=np.int64)
        kids[:, :, 0] = l + 1
        kids[:, :, 1] = 2 * a[:, None, 1] + np.array([0, 1, 0, 1])
        kids[:, :, 2] = 2 * a[:, None, 2] + np.array([0, 0, 1, 1])
        arr = kids.reshape(-1, 3)
    rows = np.concatenate(leaves, axis=0)
    order = np.lexsort((rows[:, 1], rows[:, 2], rows[:, 0]))          # sorted by (level, j0, i0)
    return Layout(L, h1 / 2.0 ** np.arange(L), -1.0, -1.0, 1, rows[order].astype(np.int32))


def paper_ilr_layout(Nk: int, L: int, disk: str = "D2") -> Layout:
    centres, alpha = ([(0.0, 0.0)], 0.5) if disk == "D2" else ([(0.0, 0.5), (0.0, -0.5)], 0.4)
    return _paper_band_layout(Nk, L, centres, alpha, lambda m: 0.05 / 2 ** (m - 1))


def paper_vlr_layout(Nk: int, L: int, disk: str = "D2") -> Layout:
    centres, alpha = ([(0.0, 0.0)], 0.5) if disk == "D2" else ([(0.0, 0.5), (0.0, -0.5)], 0.4)
    h1 = 2.0 / Nk
    return _paper_band_layout(Nk, L, centres, alpha, lambda m: 12.8 * h1 / 2 ** (m - 1))
