import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")
    config.addinivalue_line("markers", "slow: full-size parity case (minutes)")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: '#' comments, then 'key value...' lines -> dict key -> list[float]."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            parts = line.split()
            out[parts[0]] = [float(x) for x in parts[1:]]
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
