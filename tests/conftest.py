import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def golden():
    """tests/golden/closed_forms.txt -> {name: float}; every line cites the passage it follows."""
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            k, v = line.split()[:2]
            out[k] = float(v)
    return out
