import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running CPU test")


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def golden():
    return read_golden


@pytest.fixture(autouse=True)
def _default_debug_knobs():
    """rosen_debug_set knobs are process-wide: whatever a test set is back at its default for the next one, pass or fail."""
    yield
    from paper_1704_04381_b200 import binding
    if binding._lib is not None:
        for knob in ("lattice_hash_min_n", "realspace_cell_min_n", "realspace_cand_cap", "hash_blocks_per_sm"):
            binding._lib.rosen_debug_set(knob.encode(), 0)
