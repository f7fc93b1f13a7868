import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a B200 (run with -m gpu on the GPU box)")


def load_golden(name):
    """Parse tests/golden/<name>: lines 'key: d0 d1 .. | values'."""
    import numpy as np

    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, rest = line.split(":", 1)
            shape, vals = rest.split("|")
            shape = [int(v) for v in shape.split()]
            out[key.strip()] = np.array([float(v) for v in vals.split()]).reshape(shape)
    return out


@pytest.fixture(scope="session")
def golden_hand():
    return load_golden("hand_example.txt")
