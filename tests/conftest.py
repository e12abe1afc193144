import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_addoption(parser):
    parser.addoption("--full-oracle", action="store_true", default=False,
                     help="full-size GPU parity tests compare EVERY query row of two heads with the fp64 oracle instead of "
                          "the deterministic row sample (SURVEY 8(c) large-config strategy; minutes of CPU time per config)")


@pytest.fixture
def full_oracle(request):
    return request.config.getoption("--full-oracle")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")


def golden(name):
    """Rows of a tests/golden/*.txt fixture: '|'-separated cells, '#' comments."""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append([c.strip() for c in line.split("|")])
    return rows


@pytest.fixture(scope="session")
def golden_rows():
    return golden
