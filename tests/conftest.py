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


def pytest_sessionstart(session):
    """Build the in-tree CUDA library (nvcc cross-compiles without a GPU) and the C oracle once."""
    from paper_2001_02765_b200.build import build as build_lib
    from oracle.build import build as build_oracle
    build_lib()
    build_oracle()
