"""Writes tests/golden/dense_trotter.txt from oracle/dense_check.py ONLY (exact 2^N evolution).

Run from the repo root:  python tests/golden/make_golden.py
Values: C after Trotter steps 1..10 for BASELINE.json parameters (J=1, h=0.9, dt=0.05,
H = -J sum ZZ - h sum X, observable Z_c), pin P1 of SURVEY.md §8(c).  Nothing here touches
the CUDA path or oracle/pepo_oracle.py.
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "..", ".."))
from oracle import dense_check as dc  # noqa: E402

CASES = [(2, 2, 0, 0), (3, 3, 1, 1), (1, 4, 0, 1), (2, 3, 0, 1), (1, 6, 0, 2)]

if __name__ == "__main__":
    path = os.path.join(os.path.dirname(__file__), "dense_trotter.txt")
    with open(path, "w") as f:
        f.write("# Lx Ly cx cy | C(step 1..10), dense 2^N first-order Trotter, J=1 h=0.9 dt=0.05 (oracle/dense_check.py)\n")
        for (Lx, Ly, cx, cy) in CASES:
            vals = dc.dense_trotter_correlation(Lx, Ly, cx, cy, 1.0, 0.9, 0.05, 10)
            f.write("%d %d %d %d | %s\n" % (Lx, Ly, cx, cy, " ".join("%.15f" % v for v in vals)))
        f.write("# exact e^{-iHt} on 3x3 centre (1,1) at t=0.5 (Trotter-error context)\n")
        f.write("exact 3 3 1 1 0.5 | %.15f\n" % dc.dense_exact_correlation(3, 3, 1, 1, 1.0, 0.9, 0.5))
    print("wrote", path)
