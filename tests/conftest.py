import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# The oracle's matrices are small: BLAS threads beyond a few only spin (and on a box that is busy with
# something else an unlimited pool makes the CPU suite crawl).  Limit the pools for the whole session.
try:
    import numpy  # noqa: F401  (loads the BLAS whose pool is limited)
    import threadpoolctl
    _BLAS_LIMIT = threadpoolctl.threadpool_limits(limits=min(4, os.cpu_count() or 1))
except Exception:          # pragma: no cover - threadpoolctl is optional
    _BLAS_LIMIT = None


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


def read_oracle_trajectory(name):
    """Rows of a stored oracle trajectory written by tests/golden/make_oracle_twin.py:
    dicts with step, C, sweeps, status, delta, chi_max_live, gate_err, chi_sum."""
    path = os.path.join(ROOT, "tests", "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t = line.split()
            rows.append(dict(step=int(t[0]), C=float(t[1]), sweeps=int(t[2]), status=int(t[3]), delta=float(t[4]),
                             chi_max_live=int(t[5]), gate_err=float(t[6]), chi_sum=int(t[7]),
                             sens=float(t[8]) if len(t) > 8 else -1.0))
    # tolerance of C at each step: north_star's 1e-6 where the trajectory is defined that well, else 50 x the
    # running max of the oracle's own sensitivity to a one-ulp perturbation (tests/golden/make_oracle_twin.py)
    env = 0.0
    for r in rows:
        if r["sens"] == r["sens"] and r["sens"] > 0.0:
            env = max(env, r["sens"])
        r["tol_C"] = max(1e-6, 50.0 * env)
    return rows
