import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: test needs a CUDA device (run with -m gpu on a B200)")
    config.addinivalue_line("markers", "slow: long-running oracle pin (still CPU only)")


def read_golden(name):
    """tests/golden/<name>: '#' lines are comments/citations, the rest whitespace-separated fields"""
    rows = []
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                rows.append(line.split())
    return rows


@pytest.fixture(scope="session")
def po():
    from oracle import pyoracle
    return pyoracle
