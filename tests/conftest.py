import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GOLDEN = os.path.join(ROOT, "tests", "golden")


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: '#' comments, 'key = v1 v2 ...' lines."""
    out = {}
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if not line:
                continue
            key, val = line.split("=")
            out[key.strip()] = [float(v) for v in val.split()]
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
