import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    """GPU tests fail loudly (not skip) when selected on a box without CUDA; they are only
    deselected by -m "not gpu"."""
    return


@pytest.fixture(scope="session")
def golden_dense():
    path = os.path.join(ROOT, "tests", "golden", "dense_trotter.txt")
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or line.startswith("exact"):
                continue
            key, vals = line.split("|")
            out[tuple(int(t) for t in key.split())] = [float(t) for t in vals.split()]
    return out
