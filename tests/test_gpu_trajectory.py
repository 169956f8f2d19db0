"""GPU-vs-oracle parity of the full hot path through the C ABI (-m gpu): C(t) trajectories,
bond dimensions, Schmidt spectra, BP sweep counts.  Tolerances from BASELINE.json north_star:
1e-10 absolute on untruncated configs, 1e-6 absolute on truncated configs."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

J, H, DT = 1.0, 0.9, 0.05


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_30985_b200 import binding
    return torch, binding


def _run_gpu(B, Lx, Ly, cx, cy, chi_max, steps, tol, damping=0.0, opts=None, **kw):
    sim = B.Pepo(Lx, Ly, cx, cy, J, H, DT, chi_max, tol, damping, **kw)
    for k, v in (opts or {}).items():
        sim.set_option(k, v)
    out = []
    for _ in range(steps):
        sim.trotter_step()
        status, sweeps, delta = sim.bp_converge()
        out.append(dict(C=sim.correlation(), status=status, sweeps=sweeps, delta=delta,
                        chi=sim.bond_dims(), gate_err=sim.stats()["gate_err"]))
    return sim, out


def _compare(out_g, out_o, tol_c, sweeps_slack=0):
    for t, (g, o) in enumerate(zip(out_g, out_o)):
        assert g["chi"] == o["chi"], "bond dims differ at step %d: %s vs %s" % (t + 1, g["chi"], o["chi"])
        assert abs(g["C"] - o["C"]) <= tol_c, "C differs at step %d: %.15g vs %.15g" % (t + 1, g["C"], o["C"])
        assert g["status"] == o["status"]
        assert abs(g["sweeps"] - o["sweeps"]) <= sweeps_slack, (t + 1, g["sweeps"], o["sweeps"])
        assert abs(g["gate_err"] - o["gate_err"]) <= 1e-9 + 1e-6 * o["gate_err"]


def test_config1_3x3_chi8(gpu, golden_dense):
    """BASELINE configs[0]: 3x3, chi_max 8, 10 steps, centre (1,1), BP tol 1e-10 undamped."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    sim, out_g = _run_gpu(B, 3, 3, 1, 1, 8, 10, 1e-10)
    st, out_o = po.run_trajectory(3, 3, 1, 1, J, H, DT, 8, 10, 1e-10)
    _compare(out_g, out_o, 1e-10, sweeps_slack=1)
    # pin P6: within 2e-9 of the dense Trotterised evolution (tests/golden/dense_trotter.txt)
    dense = golden_dense[(3, 3, 1, 1)]
    for t in range(10):
        assert abs(out_g[t]["C"] - dense[t]) < 5e-9
    # lambda spectra agree bond by bond
    for e in range(sim.n_bonds):
        assert np.allclose(sim.get_lambda(e), st.lam[e], rtol=0, atol=1e-10)
    s = sim.stats()
    assert s["arena_high_water"] <= s["arena_model_bytes"] * 1.02 + 65536
    sim.close()


@pytest.mark.parametrize("Lx,Ly,cx,cy", [(2, 2, 0, 0), (1, 4, 0, 1), (2, 3, 0, 1), (1, 6, 0, 2)])
def test_untruncated_small_grids_vs_dense(gpu, golden_dense, Lx, Ly, cx, cy):
    """Untruncated (chi_max 64 >= any live chi for 8 steps): GPU == oracle to 1e-10 and, on
    trees (1xN) or for <= 8 steps, == exact dense evolution (pins P1-P4)."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    sim, out_g = _run_gpu(B, Lx, Ly, cx, cy, 64, 8, 1e-12)
    st, out_o = po.run_trajectory(Lx, Ly, cx, cy, J, H, DT, 64, 8, 1e-12)
    _compare(out_g, out_o, 1e-10, sweeps_slack=2)
    dense = golden_dense[(Lx, Ly, cx, cy)]
    for t in range(8):
        assert abs(out_g[t]["C"] - dense[t]) < 2e-10, (t, out_g[t]["C"], dense[t])
    sim.close()


def test_closed_forms(gpu):
    """P5: J=0 -> C(n dt) = cos(2 h n dt), all chi stay 1; h=0 -> C = 1."""
    torch, B = gpu
    sim = B.Pepo(3, 3, 1, 1, 0.0, H, DT, 8, 1e-12)
    for n in range(1, 6):
        sim.trotter_step(); sim.bp_converge()
        assert abs(sim.correlation() - np.cos(2 * H * n * DT)) < 1e-13
        assert set(sim.bond_dims()) == {1}
    sim.close()
    sim = B.Pepo(3, 3, 1, 1, J, 0.0, DT, 8, 1e-12)
    for n in range(1, 4):
        sim.trotter_step(); sim.bp_converge()
        assert abs(sim.correlation() - 1.0) < 1e-13
        assert set(sim.bond_dims()) == {1}
    sim.close()


@pytest.mark.parametrize("chi_max,steps", [(8, 24), (16, 16)])
def test_config2_twin_4x4(gpu, chi_max, steps):
    """Reduced-chi twin of BASELINE configs[1] (4x4, centre (1,1), damping 0.5 on
    non-convergence): heavily truncated trajectory, tolerance 1e-6."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    sim, out_g = _run_gpu(B, 4, 4, 1, 1, chi_max, steps, 1e-10, 0.5)
    st, out_o = po.run_trajectory(4, 4, 1, 1, J, H, DT, chi_max, steps, 1e-10, 0.5)
    _compare(out_g, out_o, 1e-6, sweeps_slack=3)
    sim.close()


def test_householder_only_matches_adaptive(gpu):
    """Cholesky path and forced Householder path give the same trajectory (R9)."""
    torch, B = gpu
    sim1, a = _run_gpu(B, 3, 3, 1, 1, 8, 8, 1e-10)
    sim2, b = _run_gpu(B, 3, 3, 1, 1, 8, 8, 1e-10, opts={"force_householder": 1})
    for x, y in zip(a, b):
        assert x["chi"] == y["chi"] and abs(x["C"] - y["C"]) < 1e-11
    assert sim2.stats()["n_cholesky"] == 0
    sim1.close(); sim2.close()


def test_bp_is_read_only(gpu):
    """R16: bp_converge / correlation do not change (psi, lambda); skipping them cannot change
    later results."""
    torch, B = gpu
    sim1, a = _run_gpu(B, 3, 3, 1, 1, 8, 5, 1e-10)
    sim2 = B.Pepo(3, 3, 1, 1, J, H, DT, 8, 1e-10)
    for _ in range(5):
        sim2.trotter_step()
    sim2.bp_converge()
    assert sim2.correlation() == a[-1]["C"]
    sim1.close(); sim2.close()


def test_init_errors(gpu):
    torch, B = gpu
    with pytest.raises(B.PepoError) as e:
        B.Pepo(3, 3, 5, 1, J, H, DT, 8, 1e-10)
    assert e.value.code == -1
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.PepoError) as e:
        B.Pepo(3, 3, 1, 1, J, H, DT, 8, 1e-10, arena=small)
    assert e.value.code == -2 and "needed" in str(e.value)
    sim = B.Pepo(2, 2, 0, 0, J, H, DT, 4, 1e-10)
    with pytest.raises(B.PepoError):
        sim.correlation()          # no messages yet
    sim.close()


def test_config4_twin_8x8_chi24_vs_stored_oracle(gpu):
    """Reduced-chi twin of BASELINE configs[3] (8x8, Z at (3,3), BP tol 1e-9, damping 0.5) at
    chi_max = 24, 30 steps, against the oracle trajectory stored by tests/golden/make_oracle_8x8.py
    (about 20 CPU-minutes, so not recomputed here).  Truncated config: 1e-6 on C (north_star);
    observed 1e-12 while BP converges in < 25 sweeps and 3e-10 at step 30."""
    import os
    torch, B = gpu
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_8x8_chi24.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#")]
    assert len(rows) == 30
    sim = B.Pepo(8, 8, 3, 3, J, H, DT, 24, 1e-9, 0.5)
    for r in rows:
        step, c_o, sweeps_o, status_o, chi_o = int(r[0]), float(r[1]), int(r[2]), int(r[3]), int(r[4])
        sim.trotter_step()
        status, sweeps, delta = sim.bp_converge()
        c = sim.correlation()
        assert status == status_o, step
        assert max(sim.bond_dims()) == chi_o, step
        assert abs(c - c_o) <= (1e-9 if step <= 23 else 1e-6), (step, c, c_o)
        # the stop test delta < 1e-9 sits on a slowly (later non-monotonically) decaying tail, so a
        # rounding-level difference in psi (a different summation order in the SVD kernel is enough)
        # moves the crossing by a few sweeps: observed +-3 between two GPU kernel variants that both
        # match C(t) to 5e-13.  The count is compared loosely and only while BP converges quickly;
        # C, the acceptance quantity of north_star, is stationary in the messages.
        if sweeps_o <= 24:
            assert abs(sweeps - sweeps_o) <= 4, (step, sweeps, sweeps_o)
    sim.close()


def test_pipelined_schedule_is_bit_identical_to_serial(gpu):
    """The multi-stream schedule of a Trotter step (option "pipeline" = number of piece streams,
    0 = serial) only reorders independent gates: C(t), bond dimensions and the site tensors must be bit-identical to
    the serial schedule (no kernel may take its launch configuration from the batch composition)."""
    torch, B = gpu
    res = []
    for pl in (0, 2, 4):
        sim = B.Pepo(4, 4, 1, 1, J, H, DT, 16, 1e-10, 0.5)
        sim.set_option("pipeline", pl)
        cs = []
        for _ in range(24):
            sim.trotter_step()
            sim.bp_converge()
            cs.append(sim.correlation())
        res.append((cs, sim.bond_dims(), sim.get_site(1, 1).copy(), sim.get_site(3, 2).copy()))
        sim.close()
    for r in res[1:]:
        assert res[0][0] == r[0]
        assert list(res[0][1]) == list(r[1])
        assert (res[0][2] == r[2]).all() and (res[0][3] == r[3]).all()


def test_symmetric_trotter_step_vs_oracle(gpu):
    """SURVEY NEXT-3, PAPER eq. (6): option trotter_order = 2 (half field gate, bond sweep, half
    field gate) against the oracle's order = 2 (itself pinned to the dense symmetric splitting in
    test_oracle_pins.py): untruncated window of 3x3 to 1e-10, truncated 4x4 chi 8 to 1e-6, and the
    closed form C(n dt) = cos(2 h n dt) at J = 0."""
    import math
    torch, B = gpu
    from oracle import pepo_oracle as po
    from oracle import dense_check as dc
    sim, out_g = _run_gpu(B, 3, 3, 1, 1, 8, 10, 1e-10, opts={"trotter_order": 2})
    st, out_o = po.run_trajectory(3, 3, 1, 1, J, H, DT, 8, 10, 1e-10, order=2)
    _compare(out_g, out_o, 1e-10, sweeps_slack=1)
    dense = dc.dense_trotter_correlation(3, 3, 1, 1, J, H, DT, 3, order=2)
    for t in range(3):                       # chi_max = 8 truncates from step 4 on
        assert abs(out_g[t]["C"] - dense[t]) < 1e-12
    sim.close()
    sim, out_g = _run_gpu(B, 4, 4, 1, 1, 8, 16, 1e-10, damping=0.5, opts={"trotter_order": 2})
    st, out_o = po.run_trajectory(4, 4, 1, 1, J, H, DT, 8, 16, 1e-10, 0.5, order=2)
    _compare(out_g, out_o, 1e-6, sweeps_slack=4)
    sim.close()
    sim = B.Pepo(3, 3, 1, 1, 0.0, H, DT, 8, 1e-12, 0.0)
    sim.set_option("trotter_order", 2)
    for n in range(1, 5):
        sim.trotter_step()
        sim.bp_converge()
        assert abs(sim.correlation() - math.cos(2 * H * n * DT)) < 1e-13
    sim.close()


def test_diagnostics_bond_entropy_and_trap_flag(gpu):
    """SURVEY NEXT-2, PAPER Table 1 (L373-L380, L451-L457): pepo_bond_entropy against the oracle's
    S_e (pinned to the dense operator-Schmidt spectrum in test_oracle_pins.py) along a truncated
    4x4 run, S = 0 on the product operator, and the trap flag = converged with >= 30 sweeps."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    sim = B.Pepo(4, 4, 1, 1, J, H, DT, 8, 1e-10, 0.5)
    st = po.PEPOState(4, 4, 1, 1, J, H, DT, 8)
    assert np.all(sim.bond_entropy() == 0.0)
    for step in range(12):
        sim.trotter_step()
        st.trotter_step()
        S_g = sim.bond_entropy()
        S_o = np.array([st.bond_entropy(e) for e in range(st.lat.n_bonds)])
        assert np.allclose(S_g, S_o, rtol=0, atol=1e-9), (step, np.abs(S_g - S_o).max())
        status, sweeps, delta = sim.bp_converge()
        assert sim.stats()["last_bp_trap"] == (1 if (status == 0 and sweeps >= 30) else 0)
    assert S_g.max() > 0.1
    sim.close()


@pytest.mark.parametrize("shape", [(3, 3, 1, 1), (1, 5, 0, 2), (5, 2, 3, 0), (4, 3, 2, 1), (2, 2, 0, 0)])
def test_pipelined_schedule_on_irregular_lattices(gpu, shape):
    """Classes with one gate, empty classes, chains and non-square grids: the multi-stream schedule
    must give the serial schedule's C(t), bond dimensions and tensors bit for bit, with and without
    the confirming Jacobi sweep being skipped only at the 1e-12 level (jacobi_early)."""
    torch, B = gpu
    Lx, Ly, cx, cy = shape
    res = {}
    for name, opts in (("serial", {"pipeline": 0}), ("piped", {"pipeline": 4}), ("piped2", {"pipeline": 2}),
                       ("noearly", {"pipeline": 4, "jacobi_early": 0.0})):
        sim = B.Pepo(Lx, Ly, cx, cy, J, H, DT, 6, 1e-10, 0.5)
        for k, v in opts.items():
            sim.set_option(k, v)
        cs = []
        for _ in range(12):
            sim.trotter_step()
            sim.bp_converge()
            cs.append(sim.correlation())
        res[name] = (cs, list(sim.bond_dims()), sim.get_site(cx, cy).copy())
        sim.close()
    for name in ("piped", "piped2"):
        assert res[name][0] == res["serial"][0], name
        assert res[name][1] == res["serial"][1], name
        assert (res[name][2] == res["serial"][2]).all(), name
    assert res["noearly"][1] == res["serial"][1]
    assert max(abs(a - b) for a, b in zip(res["noearly"][0], res["serial"][0])) < 1e-12


def test_async_site_upload_equals_synchronous(gpu):
    """pepo_set_site_async + the piece-by-piece field gate (the step starts on the sites that have
    arrived) must give bit for bit what pepo_set_site gives, on both schedules and both Trotter
    orders; pepo_site_order lists every site once."""
    torch, B = gpu
    L, chi = 4, 12
    sim = B.Pepo(L, L, 1, 1, J, H, DT, chi, 1e-10, 0.5)
    while min(sim.bond_dims()) < chi:
        sim.trotter_step()
    order = sim.site_order()
    assert sorted(order) == sorted((x, y) for y in range(L) for x in range(L))
    host = {}
    for (x, y) in order:
        a = sim.get_site(x, y)
        p = torch.empty(a.size, dtype=torch.float64).pin_memory()
        p.numpy()[:] = a
        host[(x, y)] = p
    lam = [sim.get_lambda(e) for e in range(sim.n_bonds)]
    chis = sim.bond_dims()

    def step(use_async):
        sim.set_bond_dims(chis)
        for e, l in enumerate(lam):
            sim.set_lambda(e, l)
        for (x, y) in order:
            (sim.set_site_async if use_async else sim.set_site)(x, y, host[(x, y)].numpy())
        sim.trotter_step()
        sim.bp_converge()
        return sim.correlation(), sim.get_site(1, 1).copy(), sim.get_site(3, 0).copy(), list(sim.bond_dims())

    for opts in ({"pipeline": 4, "trotter_order": 1}, {"pipeline": 4, "trotter_order": 2},
                 {"pipeline": 0, "trotter_order": 1}):
        for k, v in opts.items():
            sim.set_option(k, v)
        a, b, c2 = step(False), step(True), step(True)
        for r in (b, c2):
            assert a[0] == r[0] and a[3] == r[3], opts
            assert (a[1] == r[1]).all() and (a[2] == r[2]).all(), opts
    sim.close()
