import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def load_golden():
    out = {}
    path = os.path.join(ROOT, "tests", "golden", "paper_values.txt")
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        key, val, _cite = [s.strip() for s in line.split("|", 2)]
        out[key] = float(val)
    return out


@pytest.fixture(scope="session")
def golden():
    return load_golden()
