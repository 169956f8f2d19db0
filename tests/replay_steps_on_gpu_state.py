"""Whole-step replay at sizes no oracle trajectory reaches in reasonable time.

    python tests/replay_steps_on_gpu_state.py --grid 4 --centre 1 --chi 60 --tol 1e-10 --first 47 --last 56

Runs the CUDA path to step --first, loads ITS state (psi, lambda) into the CPU oracle (tests-only code:
imports oracle/), then advances both sides step by step to --last from that common state and prints, per
step: C(t) of both, the discarded weight of both, the largest lambda difference over all bonds and, where
tests/golden/ holds the oracle's own trajectory of the configuration, the distance of the CUDA path from it.
It separates "the CUDA step differs from the oracle's step" (would show here, from identical inputs) from
"two trajectories of the same map drift apart" (shows only against the stored trajectory).
Output of one run: profiles/cfg2_segment_replay.md.
"""
import argparse
import os
import sys
import time

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), ".."))
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
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
    ap.add_argument("--grid", type=int, default=4)
    ap.add_argument("--centre", type=int, default=1)
    ap.add_argument("--chi", type=int, default=60)
    ap.add_argument("--tol", type=float, default=1e-10)
    ap.add_argument("--damping", type=float, default=0.5)
    ap.add_argument("--first", type=int, default=47)
    ap.add_argument("--last", type=int, default=56)
    ap.add_argument("--golden", default=None, help="stored oracle trajectory under tests/golden/ (optional)")
    a = ap.parse_args()
    L, c, chi = a.grid, a.centre, a.chi
    rows = None
    name = a.golden or "oracle_%dx%d_chi%d.txt" % (L, L, chi)
    if os.path.exists(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)):
        import conftest
        rows = conftest.read_oracle_trajectory(name)
    sim = B.Pepo(L, L, c, c, 1.0, 0.9, 0.05, chi, a.tol, a.damping)
    for _ in range(a.first):
        sim.trotter_step()
    st = to_oracle(sim, L, c, chi)
    print("| step | C oracle (from the CUDA state at step %d) | C CUDA | diff | gate_err oracle | gate_err CUDA | rel | max dlambda | "
          "CUDA vs stored trajectory: dC | d gate_err rel | oracle s |" % a.first)
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for s in range(a.first + 1, a.last + 1):
        t0 = time.time()
        st.trotter_step()
        st.bp_converge(a.tol, a.damping, 100, 1000)
        Co = st.correlation()
        sim.trotter_step()
        sim.bp_converge()
        Cg = sim.correlation()
        gg = sim.stats()["gate_err"]
        dl = max(float(np.max(np.abs(sim.get_lambda(e) - np.asarray(st.lam[e])))) for e in range(sim.n_bonds))
        if rows is not None and s <= len(rows):
            r = rows[s - 1]
            gold = "%.3e | %.2e" % (abs(Cg - r["C"]), abs(gg - r["gate_err"]) / gg)
        else:
            gold = "- | -"
        print("| %d | %.15f | %.15f | %.1e | %.12e | %.12e | %.1e | %.1e | %s | %.0f |"
              % (s, Co, Cg, abs(Co - Cg), st.gate_err, gg, abs(st.gate_err - gg) / gg, dl, gold, time.time() - t0), flush=True)
    sim.close()


if __name__ == "__main__":
    main()
