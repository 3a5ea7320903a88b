import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")

# the library NaN-fills its partial-sum buffer at allocation when this is set: a slot that no kernel writes then shows
# up as NaN in Fx, Fy instead of passing as a lucky zero of fresh device memory (see ensure_partials in sg_api.cu)
os.environ.setdefault("SG_POISON_PARTIALS", "1")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def read_golden(name):
    """Rows of a whitespace-separated fixture under tests/golden (lines starting with # skipped)."""
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def golden():
    return read_golden


# Oracle samples of the three large BASELINE.json configs, computed ONCE per session (long-double oracle, all host
# cores) and shared by the direct-mode and lattice-mode parity tests.  Coverage is what the configs state, independent
# of the host's core count: cfg 3 all 53,248 targets, cfg 4 4,096 seeded targets stratified by
# level, cfg 5 4,096 targets drawn without replacement with default_rng(7 + 1000) (BASELINE.json configs[4]).
LARGE_CONFIG_SAMPLES = {3: None, 4: 4096, 5: 4096}
_large_cache = {}


def large_config_oracle(cfg):
    """(layout, sigma, idx, oracle Fx[idx], oracle Fy[idx]) of BASELINE.json config 3, 4 or 5."""
    if cfg not in _large_cache:
        import numpy as np
        import oracle
        from workloads import make_config, cell_rects, sample_targets
        lay, sigma = make_config(cfg)
        n = LARGE_CONFIG_SAMPLES[cfg]
        if n is None:
            idx = np.arange(lay.n_cells, dtype=np.int64)
        elif cfg == 5:
            idx = np.sort(np.random.default_rng(7 + 1000).choice(lay.n_cells, size=n, replace=False)).astype(np.int64)
        else:
            idx = sample_targets(lay, n, 1000 + cfg)
        r = cell_rects(lay)
        ox, oy, _ = oracle.force(r, sigma, r["kxc"][idx], r["kyc"][idx], lay.unit, precision="f80")
        _large_cache[cfg] = (lay, sigma, idx, ox, oy)
    return _large_cache[cfg]


@pytest.fixture(scope="session")
def large_oracle():
    return large_config_oracle


def pytest_sessionstart(session):
    """Build the in-tree CUDA library (nvcc cross-compiles without a GPU) and the C oracle once."""
    from paper_2001_02765_b200.build import build as build_lib
    from oracle.build import build as build_oracle
    build_lib()
    build_oracle()
