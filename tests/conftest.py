import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def load_golden(name):
    """Parse tests/golden/<name>: 'key = v v v ; v v v' lines, '#' comments."""
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line or "=" not in line:
                continue
            key, val = line.split("=", 1)
            rows = [[float(x) for x in row.split()] for row in val.split(";")]
            out[key.strip()] = rows
    return out


@pytest.fixture(scope="session")
def golden_trace():
    return load_golden("handworked_trace.txt")
