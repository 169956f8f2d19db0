"""BP replay at sizes no oracle trajectory reaches (for the BP half of a step).

    python tests/replay_bp_on_gpu_state.py --grid 8 --centre 3 --chi 32 --steps 40 --tol 1e-9 [--max-replays 4]

Runs the GPU trajectory (BASELINE configs[3] geometry by default), and on every step whose bp_converge
needed more than 100 sweeps or returned status 1 loads the GPU's (psi, lambda) into the CPU oracle
(tests-only code: imports oracle/), runs the ORACLE's bp_converge + correlation with the same budgets
on that state, and prints both sides: status, sweep count, delta, C, the per-sweep deltas at a few
budgets, and the largest message difference.  It answers "is a non-converging BP step a property of
the method (reading R6/R7) or of the CUDA path?".  Output of one run: profiles/r2_bp_replay_8x8_chi32.md.
"""
import argparse
import os
import sys
import time

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
import numpy as np  # noqa: E402

from oracle import pepo_oracle as po  # noqa: E402
from paper_2606_30985_b200 import binding as B  # noqa: E402


def to_oracle(sim, L, c, chi):
    st = po.PEPOState(L, L, c, c, 1.0, 0.9, 0.05, chi)
    dims = sim.bond_dims()
    for e in range(sim.n_bonds):
        st.lam[e] = sim.get_lambda(e)
    for v in range(L * L):
        shape = [dims[st.lat.bond_id(v, d)] for d in st.lat.legs(v)] + [4]
        st.psi[v] = sim.get_site(v % L, v // L).reshape(shape, order="F").copy()
    return st


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--grid", type=int, default=8)
    ap.add_argument("--centre", type=int, default=3)
    ap.add_argument("--chi", type=int, default=32)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--tol", type=float, default=1e-9)
    ap.add_argument("--damping", type=float, default=0.5)
    ap.add_argument("--first", type=int, default=1)
    ap.add_argument("--max-replays", type=int, default=4)
    a = ap.parse_args()
    L, c, chi, tol, d = a.grid, a.centre, a.chi, a.tol, a.damping
    sim = B.Pepo(L, L, c, c, 1.0, 0.9, 0.05, chi, tol, d)
    replays = 0
    budgets = (1, 2, 3, 5, 10, 20, 50, 100)
    for step in range(1, a.steps + 1):
        sim.trotter_step()
        status, sweeps, delta = sim.bp_converge()
        C = sim.correlation()
        dims = sim.bond_dims()
        print("GPU step %d C=%.12f status %d sweeps %d delta %.3e flags %d chi[%d,%d]"
              % (step, C, status, sweeps, delta, sim.stats()["last_bp_flags"], min(dims), max(dims)), flush=True)
        if step < a.first or not (sweeps > 100 or status == 1) or replays >= a.max_replays:
            continue
        replays += 1
        st = to_oracle(sim, L, c, chi)
        msgs, dl = st._init_messages(), []
        for _ in range(100):
            msgs, de, _ = st._bp_sweep(msgs, 0.0)
            dl.append(de)
            if de < tol:
                break
        sim.set_option("bp_damping", 0.0)
        gd = []
        for k in budgets:
            sim.set_option("bp_max_sweeps", k)
            _, sw_, d_ = sim.bp_converge()
            gd.append((k, sw_, d_))
        sim.set_option("bp_max_sweeps", 100)
        sim.set_option("bp_damping", d)
        print("  undamped delta after k sweeps, GPU   : " + " ".join("%d:%.3e" % (k, x) for k, _, x in gd), flush=True)
        print("  undamped delta after k sweeps, oracle: " + " ".join("%d:%.3e" % (k, dl[min(k, len(dl)) - 1]) for k in budgets), flush=True)
        t0 = time.time()
        so, swo, do = st.bp_converge(tol, d)
        co = st.correlation()
        print("  ORACLE on the GPU state: C=%.12f status %d sweeps %d delta %.3e (%.0f s)" % (co, so, swo, do, time.time() - t0), flush=True)
        sg, swg, dg = sim.bp_converge()
        cg = sim.correlation()
        worst = 0.0
        for e in range(sim.n_bonds):
            v1, d1, v2, d2 = st.lat.bond_sites(e)
            for g, o in ((sim.get_message(e, True), st.msgs[(v1, d1)]), (sim.get_message(e, False), st.msgs[(v2, d2)])):
                worst = max(worst, min(np.abs(g - o).max(), np.abs(g + o).max()))
        print("  GPU on the same state  : C=%.12f status %d sweeps %d delta %.3e ; max |message difference| (up to sign) %.3e"
              % (cg, sg, swg, dg, worst), flush=True)


if __name__ == "__main__":
    main()
