import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running GPU parity case")


def read_golden(name):
    """Numbers of a tests/golden/*.txt fixture (lines starting with # are the citation)."""
    vals = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                vals += [float(t) for t in line.split()]
    return vals


@pytest.fixture(scope="session")
def golden():
    return read_golden
