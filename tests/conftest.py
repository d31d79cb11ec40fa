import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (runs the CUDA path through the C ABI)")


def read_golden(name):
    """tests/golden/<name>: 'key = v v v [| v v]' lines, '#' comments (with citations)."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if not line:
                continue
            k, v = line.split("=", 1)
            parts = [[float(x) for x in p.split()] for p in v.split("|")]
            out[k.strip()] = parts if len(parts) > 1 else parts[0]
    return out


@pytest.fixture(scope="session")
def golden():
    return read_golden
