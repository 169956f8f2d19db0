"""GPU-vs-oracle parity of the BP sweep (a14) in the regimes the trajectory tests do not reach on
their own (-m gpu): the damped restart of eq. (19), the exhausted-budget
exit (L251-L256), the grouped on-device stop test (option bp_group) including grids with more than
one batch of sites per sweep, and the oracle's BP replayed on late-time GPU states."""
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


def _oracle_from_gpu(sim, Lx, Ly, cx, cy, chi_max):
    """Load the GPU's (psi, lambda) into an oracle state through the packed boundary layout."""
    from oracle import pepo_oracle as po
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, chi_max)
    dims = sim.bond_dims()
    for e in range(sim.n_bonds):
        st.lam[e] = sim.get_lambda(e)
    for v in range(Lx * Ly):
        x, y = v % Lx, v // Lx
        shape = [dims[st.lat.bond_id(v, d)] for d in st.lat.legs(v)] + [4]
        st.psi[v] = sim.get_site(x, y).reshape(shape, order="F").copy()
    return st


def _msg_diff(sim, st, up_to_sign=False):
    worst = 0.0
    for e in range(sim.n_bonds):
        v1, d1, v2, d2 = st.lat.bond_sites(e)
        for g, o in ((sim.get_message(e, True), st.msgs[(v1, d1)]), (sim.get_message(e, False), st.msgs[(v2, d2)])):
            d = np.abs(g - o).max()
            if up_to_sign:
                d = min(d, np.abs(g + o).max())
            worst = max(worst, d)
    return worst


def _bp(sim, tol, damping, n1, n2, group=8):
    sim.set_option("bp_tol", tol)
    sim.set_option("bp_damping", damping)
    sim.set_option("bp_max_sweeps", n1)
    sim.set_option("bp_max_sweeps_damped", n2)
    sim.set_option("bp_group", group)
    status, sweeps, delta = sim.bp_converge()
    return status, sweeps, delta, sim.correlation()


@pytest.mark.parametrize("grid,chi,steps", [((4, 4, 1, 1), 8, 30), ((3, 3, 1, 1), 8, 10), ((6, 6, 2, 2), 4, 14)])
def test_damped_restart_and_exhausted_budget_vs_oracle(gpu, grid, chi, steps):
    """Same state on both sides (the GPU's, loaded into the oracle), same budgets: phase 2 of R7 must
    give the oracle's status, sweep count (exact when a budget is hit), delta, messages and C.  6x6 has
    36 sites = two batches of sites per sweep (PEPO_BP_MAXS = 32)."""
    torch, B = gpu
    Lx, Ly, cx, cy = grid
    sim = B.Pepo(Lx, Ly, cx, cy, J, H, DT, chi, 1e-10, 0.5)
    for _ in range(steps):
        sim.trotter_step()
    st = _oracle_from_gpu(sim, Lx, Ly, cx, cy, chi)
    # (tol, damping d, undamped budget, damped budget)
    cases = [(1e-10, 0.5, 100, 1000),      # plain
             (1e-10, 0.5, 1, 1000),        # damped restart forced after one sweep
             (1e-10, 0.3, 2, 1000),        # d != 1/2 tells d from 1 - d
             (1e-10, 0.5, 3, 4),           # both budgets exhausted: status 1, 7 sweeps
             (1e-10, 0.0, 3, 4),           # no damping configured: status 1 after phase 1
             (1e-10, 0.7, 0, 5),           # straight into phase 2, exhausted
             (1e-10, 0.5, 5, 11)]          # budget not a multiple of the group size
    for tol, d, n1, n2 in cases:
        so, swo, do = st.bp_converge(tol, d, n1, n2)
        co = st.correlation()
        for group in (8, 1, 3):
            sg, swg, dg, cg = _bp(sim, tol, d, n1, n2, group)
            assert sg == so, (tol, d, n1, n2, group)
            if so == 1:
                assert swg == swo == n1 + (n2 if d > 0 else 0)
                assert abs(dg - do) <= 1e-9 * do + 1e-14, (dg, do)
                # identical iteration history from the deterministic init: element-wise messages
                assert _msg_diff(sim, st) < 1e-11
                assert abs(cg - co) <= 1e-10 * max(1.0, abs(co))
            else:
                # delta crosses tol on a geometric tail: the crossing may move by one sweep with rounding
                assert abs(swg - swo) <= 1, (swg, swo)
                assert _msg_diff(sim, st, up_to_sign=(swg != swo)) < 1e-8
                assert abs(cg - co) <= 1e-12 * max(1.0, abs(co)) + 1e-14
    sim.close()


def test_bp_group_is_bit_identical(gpu):
    """The grouped on-device stop test (bp_group sweeps enqueued per read-back) must give exactly the
    sweep-by-sweep loop: same sweep count, delta, messages (bit for bit) and C, in both phases, also
    on a grid with two site batches per sweep (7x5 = 35 sites)."""
    torch, B = gpu
    for (Lx, Ly, cx, cy, chi, steps) in [(4, 4, 1, 1, 8, 40), (7, 5, 3, 2, 4, 12)]:
        sim = B.Pepo(Lx, Ly, cx, cy, J, H, DT, chi, 1e-10, 0.5)
        for _ in range(steps):
            sim.trotter_step()
        for (n1, n2) in [(100, 1000), (2, 1000), (4, 9)]:
            ref = None
            for group in (1, 2, 5, 8):
                r = _bp(sim, 1e-10, 0.5, n1, n2, group)
                msgs = [sim.get_message(e, f) for e in range(sim.n_bonds) for f in (True, False)]
                if ref is None:
                    ref = (r, msgs)
                else:
                    assert r == ref[0], (group, r, ref[0])
                    assert all(np.array_equal(a, b) for a, b in zip(msgs, ref[1])), group
        sim.close()


def test_oracle_bp_replayed_on_late_gpu_state_8x8_chi32(gpu):
    """BP replay (SURVEY 8(d)(3) for the BP half of a step): the GPU's 8x8 chi_max = 32 state of
    BASELINE configs[3]'s geometry at step 24 (no oracle trajectory is affordable at this chi) is
    loaded into the oracle, whose bp_converge + correlation must agree with the GPU's on status,
    sweep count, delta, messages and C.  At this step BP wanders with delta ~ 1 for ~35 sweeps before
    it drops into the basin of its fixed point (43 sweeps)."""
    torch, B = gpu
    L, chi = 8, 32
    sim = B.Pepo(L, L, 3, 3, J, H, DT, chi, 1e-9, 0.5)
    for _ in range(24):
        sim.trotter_step()
    sg, swg, dg = sim.bp_converge()
    cg = sim.correlation()
    st = _oracle_from_gpu(sim, L, L, 3, 3, chi)
    so, swo, do = st.bp_converge(1e-9, 0.5)
    co = st.correlation()
    assert (sg, so) == (0, 0) and abs(swg - swo) <= 2, (swg, swo)
    assert swo > 30
    assert abs(cg - co) <= 1e-12
    assert _msg_diff(sim, st, up_to_sign=True) < 1e-8
    # exhausted budgets on the same state: exact sweep count, delta and messages
    so, swo, do = st.bp_converge(1e-9, 0.5, 20, 10)
    sg, swg, dg, cg = _bp(sim, 1e-9, 0.5, 20, 10)
    assert (sg, swg) == (so, swo) == (1, 30)
    assert abs(dg - do) <= 1e-6 * do
    assert _msg_diff(sim, st) < 1e-9
    assert abs(cg - st.correlation()) <= 1e-9 * max(1.0, abs(cg))
    sim.close()


def test_zero_norm_message_is_flagged_and_nan_is_an_error(gpu):
    """R7: a message update with zero norm keeps the old message and is flagged (stats.last_bp_flags
    bit 0; the oracle does the same); a NaN in a site tensor makes bp_converge fail with -4 instead of
    reporting a converged delta of 0."""
    torch, B = gpu
    sim = B.Pepo(3, 3, 1, 1, J, H, DT, 4, 1e-10, 0.5)
    for _ in range(3):
        sim.trotter_step()
    sim.bp_converge()
    assert sim.stats()["last_bp_flags"] == 0
    st = _oracle_from_gpu(sim, 3, 3, 1, 1, 4)
    a = sim.get_site(0, 0)
    sim.set_site(0, 0, np.zeros_like(a))                  # corner tensor = 0: its outgoing updates have zero norm
    st.psi[0] = np.zeros_like(st.psi[0])
    status, sweeps, delta = sim.bp_converge()
    assert sim.stats()["last_bp_flags"] & 1
    so, swo, do = st.bp_converge(1e-10, 0.5)
    assert (status, sweeps) == (so, swo)
    assert _msg_diff(sim, st, up_to_sign=True) < 1e-9
    bad = a.copy(); bad[0] = np.nan
    sim.set_site(0, 0, bad)
    with pytest.raises(B.PepoError) as e:
        sim.bp_converge()
    assert e.value.code == -4
    assert sim.stats()["last_bp_flags"] & 2
    sim.close()


def test_alpha_ladder_and_observe_match_the_oracle(gpu):
    """SURVEY NEXT-2 / PAPER.md L451-L457: the third BP stage (option bp_ladder, alpha = 0.8) and the trap
    remediation call pepo_observe against the oracle's bp_converge(damping2=...) / observe on the same
    state (4x4 chi 8 at step 52, where BP needs 37 / 69 / 42 sweeps at alpha = 1 / 0.5 / 0.8): stage,
    sweep counts (exact when a budget is hit), status and C for (1) a healthy step, (2) budgets that
    only the third stage meets, (3) a forced 'drop' that makes every alpha look trapped (status 2),
    (4) the same drop excused by a doubled gate_err."""
    torch, B = gpu
    sim = B.Pepo(4, 4, 1, 1, J, H, DT, 8, 1e-10, 0.5)
    for _ in range(52):
        sim.trotter_step()
    st = _oracle_from_gpu(sim, 4, 4, 1, 1, 8)
    st.gate_err = sim.stats()["gate_err"]
    sim.set_option("bp_ladder", 1)
    # (1) healthy: first call accepts (reference C(0) = 1: a drop, but the first reference gate_err is 0)
    so = st.observe(1e-10, 0.5, 0.2)
    sg = sim.observe()
    assert sg[0] == so[0] == 0 and sg[3] == so[3] == 0
    assert abs(sg[1] - so[1]) < 1e-12 and abs(sg[2] - so[2]) <= 1
    # (2) small budgets: only alpha = 0.8 converges
    sim.set_option("bp_max_sweeps", 5); sim.set_option("bp_max_sweeps_damped", 45)
    s_o, n_o, _ = st.bp_converge(1e-10, 0.5, 5, 45, damping2=0.2)
    s_g, n_g, _ = sim.bp_converge()
    assert (s_g, s_o) == (0, 0) and st.bp_stage == 2 and sim.stats()["last_bp_stage"] == 2
    assert abs(n_g - n_o) <= 1 and n_o > 50
    assert abs(sim.correlation() - st.correlation()) < 1e-12
    sim.set_option("bp_ladder", 0)
    assert sim.bp_converge()[0] == 1 and sim.stats()["last_bp_stage"] == 1          # without the ladder: exhausted
    sim.set_option("bp_ladder", 1)
    sim.set_option("bp_max_sweeps", 100); sim.set_option("bp_max_sweeps_damped", 1000)
    # (3) forced drop: the reference says C should be 10x larger, gate_err quiet -> every alpha is retried
    # from the init, all reach the same fixed point -> status 2 ("raise chi"), reference kept
    c0 = so[1]
    st.obs_prev_C, st.obs_prev_gerr = 10.0 * c0, st.gate_err
    sim.set_option("observe_ref_C", 10.0 * c0); sim.set_option("observe_ref_gate_err", st.gate_err)
    so3 = st.observe(1e-10, 0.5, 0.2)
    sg3 = sim.observe()
    assert sg3[0] == so3[0] == 2 and sg3[3] == so3[3] == 2
    assert abs(sg3[1] - so3[1]) < 1e-12 and abs(sg3[2] - so3[2]) <= 3 and so3[2] > 120
    # (4) the same drop with a gate_err more than twice the reference's is accepted at once
    st.obs_prev_gerr = 0.4 * st.gate_err
    sim.set_option("observe_ref_gate_err", 0.4 * st.gate_err)
    so4 = st.observe(1e-10, 0.5, 0.2)
    sg4 = sim.observe()
    assert sg4[0] == so4[0] == 0 and sg4[3] == so4[3] == 0 and abs(sg4[1] - so4[1]) < 1e-12
    sim.close()


def test_leading_schmidt_vector_init_matches_oracle_and_converges_where_uniform_fails(gpu):
    """Reading R7b (option bp_init = 1): BP started from e_0 on every bond.  On the 8x8 chi_max = 32 state
    at step 28 the uniform init of R7 exhausts both budgets on the GPU and in the oracle alike
    (profiles/r2_bp_replay_8x8_chi32.md); from e_0 the damped stage converges in a few dozen sweeps on both
    sides, to the same messages and the same C, which continues the curve of the chi_max = 24 twin
    (tests/golden/oracle_8x8_chi24_40.txt: C(28) = 0.27895)."""
    torch, B = gpu
    L, chi = 8, 32
    sim = B.Pepo(L, L, 3, 3, J, H, DT, chi, 1e-9, 0.5)
    for _ in range(28):
        sim.trotter_step()
    sim.set_option("bp_max_sweeps_damped", 300)
    sg, swg, _ = sim.bp_converge()
    assert sg == 1 and swg == 400                                  # uniform init: 100 + 300 sweeps, not converged
    sim.set_option("bp_init", 1)
    sg, swg, dg = sim.bp_converge()
    cg = sim.correlation()
    st = _oracle_from_gpu(sim, L, L, 3, 3, chi)
    st.bp_init = "e0"
    so, swo, do = st.bp_converge(1e-9, 0.5, 100, 300)
    co = st.correlation()
    assert (sg, so) == (0, 0) and abs(swg - swo) <= 1 and swo < 200
    assert abs(cg - co) < 1e-12 and abs(cg - 0.279) < 1e-3
    assert _msg_diff(sim, st, up_to_sign=(swg != swo)) < 1e-8
    sim.close()

