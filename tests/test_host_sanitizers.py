"""Host code under AddressSanitizer + UndefinedBehaviorSanitizer (compute-sanitizer is closed on
the GPU pool, but the host side needs no GPU): the library's layout builder (csrc/sg_layout.cpp, the
CUDA-free half of sg_create) and the C oracle are compiled with -fsanitize=address,undefined -fno-sanitize-recover
into two small drivers (tests/sanitize/) and run on the layouts and pin cases of this suite.  A finding aborts the
driver (non-zero exit status) and fails the test; results are also compared with the ordinary builds."""
import os
import subprocess

import numpy as np
import pytest

import oracle
from paper_2001_02765_b200 import SgDisk, binding
from workloads import Layout, make_config, cell_rects, paper_ilr_layout, nested_layout, random_refined_layout
from workloads.configs import _sorted_patches

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1", "-fopenmp"]
ENV = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1",
           OMP_NUM_THREADS="4")


@pytest.fixture(scope="module")
def drivers(tmp_path_factory):
    out = tmp_path_factory.mktemp("sanitize")
    lay = str(out / "layout_driver")
    subprocess.check_call(["g++", "-std=c++17", *SAN, os.path.join(ROOT, "tests", "sanitize", "layout_driver.cpp"),
                           os.path.join(ROOT, "paper_2001_02765_b200", "csrc", "sg_layout.cpp"), "-o", lay])
    objs = []
    for tag, defs in (("f80", []), ("f64", ["-DSG_ORACLE_DOUBLE"])):
        o = str(out / f"oracle_{tag}.o")
        subprocess.check_call(["gcc", "-std=c11", "-fno-fast-math", *SAN, *defs, "-c",
                               os.path.join(ROOT, "oracle", "sg_oracle.c"), "-o", o])
        objs.append(o)
    orc = str(out / "oracle_driver")
    subprocess.check_call(["gcc", "-std=c11", *SAN, os.path.join(ROOT, "tests", "sanitize", "oracle_driver.c"), *objs,
                           "-o", orc, "-lm"])
    return lay, orc


def _run(exe, text):
    p = subprocess.run([exe], input=text, capture_output=True, text=True, env=ENV, timeout=600)
    assert p.returncode == 0, f"sanitizer finding or crash (exit {p.returncode}):\n{p.stderr[-4000:]}"
    assert "runtime error" not in p.stderr and "AddressSanitizer" not in p.stderr, p.stderr[-4000:]
    return p.stdout


def _layout_text(lay):
    rows = "\n".join(f"{l} {i} {j}" for l, i, j in lay.patches.tolist())
    return f"{lay.n_levels} {lay.P} {lay.n_patches}\n" + " ".join(repr(float(w)) for w in lay.cell_width) + "\n" + rows + "\n"


def _fig1():
    l0 = [(0, i, j) for j in range(4) for i in range(4) if (i, j) not in ((1, 1), (2, 2))]
    l1 = [(1, 2, 2), (1, 3, 3)] + [(1, 4 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    l2 = [(2, 4 + di, 6 + dj) for dj in (0, 1) for di in (0, 1)] + [(2, 6 + di, 4 + dj) for dj in (0, 1) for di in (0, 1)]
    return Layout(3, np.array([0.25, 0.125, 0.0625]), 0.0, 0.0, 1, _sorted_patches(l0 + l1 + l2))


LAYOUTS = {
    "cfg1": lambda: make_config(1)[0], "cfg2": lambda: make_config(2)[0], "cfg3": lambda: make_config(3)[0],
    "ilr_p1": lambda: paper_ilr_layout(32, 3), "fig1_unbalanced": _fig1, "nest5_p4": lambda: nested_layout(5, 32, 8.0, 4),
    "ragged_p2": lambda: random_refined_layout(11, 24, 2, 4, 0.3),
}


@pytest.mark.parametrize("name", sorted(LAYOUTS))
def test_layout_builder_under_asan_ubsan(drivers, name):
    lay = LAYOUTS[name]()
    got = _run(drivers[0], _layout_text(lay)).split()
    assert int(got[0]) == 0, got
    with SgDisk.from_layout(lay, device=-1) as d:                  # the ordinary build, host-only context
        info = d.layout_info()
    assert [int(v) for v in got[1:8]] == [info[k] for k in ("n_cells", "n_vertices", "n_vertex_x", "n_vertex_y",
                                                            "n_target_x", "n_target_y", "balanced")]


def test_refused_layouts_under_asan_ubsan(drivers):
    """The validation paths (overlap, duplicate, off-lattice origin, level out of range, widths not halving, empty
    list): refused with the library's error codes, without a sanitizer finding."""
    base = make_config(2)[0]
    def variant(patches=None, cw=None, P=None, n_levels=None):
        return Layout(n_levels or base.n_levels, np.array(cw if cw is not None else base.cell_width), base.x0, base.y0,
                      P or base.P, np.asarray(base.patches if patches is None else patches, dtype=np.int32).reshape(-1, 3))
    p = base.patches
    fine = p[p[:, 0] == p[:, 0].max()][0]
    cases = {
        "duplicate": variant(np.vstack([p, p[:1]])),
        "overlap": variant(np.vstack([p, [[fine[0] - 1, (fine[1] // 2 // base.P) * base.P, (fine[2] // 2 // base.P) * base.P]]])),
        "off_lattice": variant(np.vstack([p[1:], [[p[0][0], p[0][1] + 1, p[0][2]]]])),
        "level_out_of_range": variant(np.vstack([p, [[base.n_levels, 0, 0]]])),
        "negative_origin": variant(np.vstack([p, [[0, -base.P, 0]]])),
        "widths_not_halving": variant(cw=[1.0, 0.3][:base.n_levels] if base.n_levels == 2 else [1.0] * base.n_levels),
        "empty": variant(np.zeros((0, 3), dtype=np.int32)),
    }
    for name, lay in cases.items():
        got = _run(drivers[0], _layout_text(lay)).split()
        assert int(got[0]) in (binding.SG_ERR_ARG, binding.SG_ERR_LAYOUT), (name, got)


def test_oracle_under_asan_ubsan(drivers):
    """Both builds of the oracle on config 2 (two levels, coincident grid lines: the modified primitive runs), zeroth
    order and with slope terms, 96 seeded targets: no finding, and the same numbers as the ordinary -O2 library."""
    lay, sigma = make_config(2)
    r = cell_rects(lay)
    rng = np.random.default_rng(5)
    idx = np.sort(rng.choice(lay.n_cells, 96, replace=False))
    dx, dy = rng.normal(size=lay.n_cells), rng.normal(size=lay.n_cells)
    for slopes in (0, 1):
        head = f"{lay.n_cells} {idx.size} {slopes} {lay.unit!r} 1.5\n"
        cells = "\n".join(f"{a} {b} {c} {d} {s!r} {e!r} {g!r}" for a, b, c, d, s, e, g in
                          zip(r["kxl"].tolist(), r["kxr"].tolist(), r["kyd"].tolist(), r["kyu"].tolist(),
                              sigma.tolist(), dx.tolist(), dy.tolist()))
        tg = "\n".join(f"{a} {b}" for a, b in zip(r["kxc"][idx].tolist(), r["kyc"][idx].tolist()))
        got = np.array([[float(v) for v in ln.split()] for ln in _run(drivers[1], head + cells + "\n" + tg + "\n").splitlines()])
        kw = dict(dx=dx, dy=dy) if slopes else {}
        for prec, cols in (("f80", (0, 1)), ("f64", (2, 3))):
            ox, oy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, G=1.5, precision=prec, **kw)
            s = max(np.abs(ox).max(), np.abs(oy).max())
            assert np.abs(got[:, cols[0]] - ox).max() <= 1e-15 * s and np.abs(got[:, cols[1]] - oy).max() <= 1e-15 * s
