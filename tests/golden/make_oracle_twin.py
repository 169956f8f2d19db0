"""Writes a stored oracle trajectory tests/golden/oracle_<Lx>x<Ly>_chi<chi>.txt from
oracle/pepo_oracle.py ONLY (nothing here touches the CUDA path): the reduced-chi twins of BASELINE
configs[1], [3], [4] (same grid, centre, J=1 h=0.9 dt=0.05, same BP tolerance and damping, same
number of steps; only chi_max is reduced to what the CPU oracle finishes in minutes).

Run from the repo root, e.g.
    python tests/golden/make_oracle_twin.py --grid 10 10 --centre 4 4 --chi 8 --steps 30 --tol 1e-8
    python tests/golden/make_oracle_twin.py --grid 4 4 --centre 1 1 --chi 16 --steps 60 --tol 1e-10
    python tests/golden/make_oracle_twin.py --grid 8 8 --centre 3 3 --chi 24 --steps 40 --tol 1e-9
Columns: step, C(t), BP sweeps (both phases), BP status, BP delta, max live bond dimension, gate_err,
sum of all bond dimensions, sens.  A status-1 line is an exhausted budget.

--sens N (default 0): N more oracle states run in lockstep, identical except that after step 5 every
entry of every site tensor is multiplied ONCE by (1 + 1e-15 g), g ~ N(0,1) from default_rng(seed = 1..N):
a one-ulp perturbation.  sens = max over the N copies of |C - C_perturbed| at that step = how far the
truncated trajectory amplifies rounding, i.e. to how many digits C(t) is defined at all by the algorithm
in fp64.  The parity tests compare the CUDA path to C within max(1e-6, 50 x running max of sens).

Where the plain trajectory takes hours (4x4 chi 60: ~5 min per saturated step) the perturbed copies can be
run separately and merged in afterwards:
    python tests/golden/make_oracle_twin.py <same arguments> --perturbed-only K    # writes <out>.pertK
    python tests/golden/make_oracle_twin.py <same arguments> --merge-sens          # sens column from all <out>.pertK
(the stored C stays the one of the unperturbed run; only the last column and the header change).
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
    ap.add_argument("--sens", type=int, default=0)
    ap.add_argument("--perturbed-only", type=int, default=0)
    ap.add_argument("--merge-sens", action="store_true")
    a = ap.parse_args()
    Lx, Ly = a.grid
    cx, cy = a.centre
    import numpy as np
    if a.perturbed_only or a.merge_sens:
        import glob
        name = a.out or "oracle_%dx%d_chi%d.txt" % (Lx, Ly, a.chi)
        path = os.path.join(os.path.dirname(__file__), name)
        if a.perturbed_only:
            k = a.perturbed_only
            tw = po.PEPOState(Lx, Ly, cx, cy, 1.0, 0.9, 0.05, a.chi)
            t0 = time.time()
            with open(path + ".pert%d" % k, "w") as f:
                f.write("# perturbed copy %d (1e-15 relative, default_rng(%d), after step 5) of %s\n# step C status\n" % (k, k, name))
                for s in range(1, a.steps + 1):
                    tw.trotter_step()
                    if s == 5:
                        rng = np.random.default_rng(k)
                        for v in range(Lx * Ly):
                            tw.psi[v] = tw.psi[v] * (1.0 + 1e-15 * rng.standard_normal(tw.psi[v].shape))
                    stw, _, _ = tw.bp_converge(a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped)
                    f.write("%d %.15f %d\n" % (s, tw.correlation(), stw))
                    f.flush()
                    sys.stderr.write("step %d done, %.0f s\n" % (s, time.time() - t0))
            sys.exit(0)
        perts = []
        for pf in sorted(glob.glob(path + ".pert*")):
            perts.append({int(l.split()[0]): (float(l.split()[1]), int(l.split()[2])) for l in open(pf) if not l.startswith("#")})
        lines = open(path).read().splitlines()
        out = []
        for l in lines:
            if l.startswith("# sens:"):
                continue
            if l.startswith("# step"):
                out.append("# sens: %d copies perturbed once by 1e-15 (relative, seeded) after step 5, run separately "
                           "(--perturbed-only) and merged; -1 = beyond the last step the copies reached" % len(perts))
                out.append("# step C sweeps status delta chi_max_live gate_err chi_sum sens")
                continue
            if l.startswith("#"):
                out.append(l); continue
            w = l.split()[:8]
            s, C, status = int(w[0]), float(w[1]), int(w[3])
            have = [p[s] for p in perts if s in p]
            if not have: sens = -1.0
            else: sens = max((abs(c - C) if (stw == 0 and status == 0) else float("nan")) for c, stw in have)
            out.append(" ".join(w) + " %.3e" % sens)
        open(path, "w").write("\n".join(out) + "\n")
        print("merged %d perturbed copies into %s" % (len(perts), path))
        sys.exit(0)
    st = po.PEPOState(Lx, Ly, cx, cy, 1.0, 0.9, 0.05, a.chi)
    twins = [po.PEPOState(Lx, Ly, cx, cy, 1.0, 0.9, 0.05, a.chi) for _ in range(a.sens)]
    name = a.out or "oracle_%dx%d_chi%d.txt" % (Lx, Ly, a.chi)
    path = os.path.join(os.path.dirname(__file__), name)
    t0 = time.time()
    with open(path, "w") as f:
        f.write("# %dx%d centre (%d,%d) chi_max %d, J=1 h=0.9 dt=0.05, BP tol %g damping %g budgets %d/%d "
                "(oracle/pepo_oracle.py via tests/golden/make_oracle_twin.py)\n"
                % (Lx, Ly, cx, cy, a.chi, a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped))
        f.write("# sens: %d copies perturbed once by 1e-15 (relative, seeded) after step 5\n" % a.sens)
        f.write("# step C sweeps status delta chi_max_live gate_err chi_sum sens\n")
        for s in range(1, a.steps + 1):
            st.trotter_step()
            status, sweeps, delta = st.bp_converge(a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped)
            chis = st.bond_dims()
            C = st.correlation()
            sens = 0.0
            for k, tw in enumerate(twins):
                tw.trotter_step()
                if s == 5:
                    rng = np.random.default_rng(k + 1)
                    for v in range(Lx * Ly):
                        tw.psi[v] = tw.psi[v] * (1.0 + 1e-15 * rng.standard_normal(tw.psi[v].shape))
                stw, _, _ = tw.bp_converge(a.tol, a.damping, a.max_sweeps, a.max_sweeps_damped)
                sens = max(sens, abs(tw.correlation() - C) if (stw == 0 and status == 0) else float("nan"))
            f.write("%d %.15f %d %d %.6e %d %.12e %d %.3e\n" % (s, C, sweeps, status, delta,
                                                             max(chis), st.gate_err, sum(chis), sens if a.sens else -1.0))
            f.flush()
            sys.stderr.write("step %d done, %.0f s\n" % (s, time.time() - t0))
    print("wrote", path)
