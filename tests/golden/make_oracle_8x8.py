"""Writes tests/golden/oracle_8x8_chi24.txt from oracle/pepo_oracle.py ONLY: the reduced-chi twin
of BASELINE configs[3] (8x8 open grid, Z at (3,3), J=1 h=0.9 dt=0.05, BP tol 1e-9, damping 0.5)
at chi_max = 24, 30 steps - the largest chi at which the CPU oracle finishes in ~20 minutes.

Run from the repo root:  python tests/golden/make_oracle_8x8.py     (about 20 min on 8 cores)
Columns: step, C(t), BP sweeps, BP status, max bond dimension.  Nothing here touches the CUDA path.
"""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "..", ".."))
from oracle import pepo_oracle as po  # noqa: E402

if __name__ == "__main__":
    chi, steps = 24, 30
    st = po.PEPOState(8, 8, 3, 3, 1.0, 0.9, 0.05, chi)
    path = os.path.join(os.path.dirname(__file__), "oracle_8x8_chi24.txt")
    with open(path, "w") as f:
        f.write("# 8x8 centre (3,3) chi_max 24, J=1 h=0.9 dt=0.05, BP tol 1e-9 damping 0.5 (oracle/pepo_oracle.py)\n")
        f.write("# step C sweeps status chi_max_live\n")
        for s in range(1, steps + 1):
            st.trotter_step()
            status, sweeps, delta = st.bp_converge(1e-9, 0.5)
            f.write("%d %.15f %d %d %d\n" % (s, st.correlation(), sweeps, status, max(st.bond_dims())))
            f.flush()
    print("wrote", path)
