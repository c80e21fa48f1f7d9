import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    import __graft_entry__

    __graft_entry__.ensure_built()  # fresh checkout: compile libkvtier.so (nvcc, sm_100a) and the oracles (gcc)


def read_golden(name):
    """tests/golden/*.txt: '#' comments, whitespace-separated integers."""
    path = os.path.join(ROOT, "tests", "golden", name)
    vals = []
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0]
            vals.extend(int(x) for x in line.split())
    return vals


@pytest.fixture(scope="session")
def golden():
    return read_golden
