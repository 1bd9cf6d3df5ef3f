"""pytest configuration: registers the ``gpu`` marker (tests that need a B200)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


def read_golden(name):
    """Parse tests/golden/<name>: '#' comments, 'key = value' lines -> dict of floats."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
