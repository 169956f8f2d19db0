"""Writes a stored oracle trajectory tests/golden/oracle_<Lx>x<Ly>_chi<chi>.txt from
oracle/pepo_oracle.py ONLY (nothing here touches the CUDA path): the reduced-chi twins of BASELINE
configs[1], [3], [4] (same grid, centre, J=1 h=0.9 dt=0.05, same BP tolerance and damping, same
number of steps; only chi_max is reduced to what the CPU oracle finishes in minutes).

Run from the repo root, e.g.
    python tests/golden/make_oracle_twin.py --grid 10 10 --centre 4 4 --chi 8 --steps 30 --tol 1e-8
    python tests/golden/make_oracle_twin.py --grid 4 4 --centre 1 1 --chi 16 --steps 60 --tol 1e-10
    python tests/golden/make_oracle_twin.py --grid 8 8 --centre 3 3 --chi 24 --steps 40 --tol 1e-9
Columns: step, C(t), BP sweeps (both phases), BP status, BP delta, max live bond dimension, gate_err,
sum of all bond dimensions.  A status-1 line is an exhausted budget.
"""
import argparse
import os
import sys
import time

sys.path.insert(0, os.path.join(os.path.dirname(__file__), "..", ".."))
from oracle import pepo_oracle as po  # noqa: E402

if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--grid", type=int, nargs=2, required=True)
    ap.add_argument("--centre", type=int, nargs=2, required=True)
    ap.add_argument("--chi", type=int, required=True)
    ap.add_argument("--steps", type=int, required=True)
    ap.add_argument("--tol", type=float, required=True)
    ap.add_argument("--damping", type=float, default=0.5)
    ap.add_argument("--max-sweeps", type=int, default=100)
    ap.add_argument("--max-sweeps-damped", type=int, default=1000)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    Lx, Ly = a.grid
    cx, cy = a.centre
    st = po.PEPOState(Lx, Ly, cx, cy, 1.0, 0.9, 0.05, a.chi)
    name = a.out or "oracle_%dx%d_chi%d.txt" % (Lx, Ly, a.chi)
    path = os.path.join(os.path.dirname(__file__), name)
    t0 = time.time()
    with open(path, "w") as f:
        f.write("# %dx%d centre (%d,%d) chi_max %d, J=1 h=0.9 dt=0.05, BP tol %g damping %g budgets %d/%d "
                "(oracle/pepo_oracle.py via tests/golden/make_oracle_twin.py)\n"
                % (Lx, Ly, cx, cy, a.chi, a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped))
        f.write("# step C sweeps status delta chi_max_live gate_err chi_sum\n")
        for s in range(1, a.steps + 1):
            st.trotter_step()
            status, sweeps, delta = st.bp_converge(a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped)
            chis = st.bond_dims()
            f.write("%d %.15f %d %d %.6e %d %.12e %d\n" % (s, st.correlation(), sweeps, status, delta,
                                                       max(chis), st.gate_err, sum(chis)))
            f.flush()
            sys.stderr.write("step %d done, %.0f s\n" % (s, time.time() - t0))
    print("wrote", path)
