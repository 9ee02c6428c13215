import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: long-running (full-size configs)")


def load_worked_example():
    path = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")
    out = {}
    with open(path) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, *vals = line.split()
            out.setdefault(key, []).append([float(v) if "." in v else int(v) for v in vals])
    return out


@pytest.fixture(scope="session")
def worked_example():
    return load_worked_example()
