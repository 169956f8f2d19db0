"""GPU-vs-oracle parity of SURVEY NEXT-1 (-m gpu): belief propagation on the norm network with chi x chi
matrix messages, the Bethe norm of Table 1 (L373-L380, L550), PSEUDO_SQRT
(L315-L317) and the matrix absorb / de-absorb of the gate environment (L318, L336)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

J, H, DT = 1.0, 0.9, 0.05
BACK = {"U": "D", "D": "U", "L": "R", "R": "L"}


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_30985_b200 import binding
    return torch, binding


def _oracle_from_gpu(sim, Lx, Ly, cx, cy, chi_max):
    from oracle import pepo_oracle as po
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, chi_max)
    dims = sim.bond_dims()
    for e in range(sim.n_bonds):
        st.lam[e] = sim.get_lambda(e)
    for v in range(Lx * Ly):
        shape = [dims[st.lat.bond_id(v, d)] for d in st.lat.legs(v)] + [4]
        st.psi[v] = sim.get_site(v % Lx, v // Lx).reshape(shape, order="F").copy()
    return st


def _msg_diff(sim, st):
    """Oracle Min[(v, d)] = message arriving at v through leg d; the message sent by v1 over bond e arrives
    at v2 through d2."""
    worst = 0.0
    for e in range(sim.n_bonds):
        v1, d1, v2, d2 = st.lat.bond_sites(e)
        worst = max(worst, np.abs(sim.get_norm_message(e, True) - st.Min[(v2, d2)]).max(),
                    np.abs(sim.get_norm_message(e, False) - st.Min[(v1, d1)]).max())
    return worst


def test_tree_fixed_point_and_bethe_norm(gpu):
    """SURVEY 8(f) pins on the device: 1x5 chain, 6 untruncated steps - the matrix messages converge to
    diag(lambda_e) and the Bethe norm is 1."""
    torch, B = gpu
    sim = B.Pepo(1, 5, 0, 2, J, H, DT, 64, 1e-12, 0.0)
    for _ in range(6):
        sim.trotter_step()
    status, sweeps, delta = sim.norm_bp_converge(1e-13, 0.0, 50)
    assert status == 0 and sweeps <= 3
    for e in range(sim.n_bonds):
        lam = sim.get_lambda(e)
        for f in (True, False):
            assert np.abs(sim.get_norm_message(e, f) - np.diag(lam)).max() < 1e-10      # gauge defect of the eps_cut = 1e-11 pruning
    assert abs(sim.bethe_norm() - 1.0) < 1e-10
    sim.check_guards()
    sim.close()


@pytest.mark.parametrize("grid,chi,steps", [((3, 3, 1, 1), 4, 16), ((4, 3, 1, 1), 6, 12), ((2, 2, 0, 0), 16, 8)])
def test_matrix_message_sweeps_and_bethe_norm_vs_oracle(gpu, grid, chi, steps):
    """Same state on both sides (the GPU's): sweep count, delta, every matrix message element-wise and the
    Bethe norm of pepo_norm_bp_converge / pepo_bethe_norm against the oracle, undamped and damped."""
    torch, B = gpu
    Lx, Ly, cx, cy = grid
    sim = B.Pepo(Lx, Ly, cx, cy, J, H, DT, chi, 1e-10, 0.5)
    for _ in range(steps):
        sim.trotter_step()
    st = _oracle_from_gpu(sim, Lx, Ly, cx, cy, chi)
    for damping, budget in ((0.0, 400), (0.5, 400), (0.0, 3)):
        sim.set_lambda(0, sim.get_lambda(0))                      # forget the messages: next call starts from diag(lambda)
        st.norm_bp_init()
        so, no, do = st.norm_bp_converge(1e-12, damping, budget)
        sg, ng, dg = sim.norm_bp_converge(1e-12, damping, budget)
        assert sg == so and abs(ng - no) <= (0 if so == 1 else 1), (damping, budget, ng, no)
        if so == 1:
            assert abs(dg - do) <= 1e-6 * do + 1e-15
        assert _msg_diff(sim, st) < 1e-9
        assert abs(sim.bethe_norm() - st.bethe_norm()) < 1e-9
    sim.check_guards()
    sim.close()


def test_gates_in_the_matrix_environment_vs_oracle(gpu):
    """Option env = 1: every Trotter step is preceded by norm-BP from diag(lambda) and its gates absorb the
    PSEUDO_SQRT of the incoming matrix messages.  3x3 chi_max 4, 20 steps, against the oracle doing the same
    (pinned in test_oracle_pins.py: exact while untruncated, separates from the diagonal environment once
    truncation is active): bond dimensions, lambda, C(t); and on the chain the two environments coincide."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    sim = B.Pepo(3, 3, 1, 1, J, H, DT, 4, 1e-12, 0.0)
    ref = B.Pepo(3, 3, 1, 1, J, H, DT, 4, 1e-12, 0.0)
    sim.set_option("env", 1)
    st = po.PEPOState(3, 3, 1, 1, J, H, DT, 4)
    sep = 0.0
    for t in range(20):
        sim.set_lambda(0, sim.get_lambda(0))
        sg, ng, _ = sim.norm_bp_converge(1e-12, 0.0, 500)
        st.norm_bp_init()
        so, no, _ = st.norm_bp_converge(1e-12, 0.0, 500)
        assert sg == so == 0 and abs(ng - no) <= 1
        sim.trotter_step(); st.trotter_step(); ref.trotter_step()
        assert sim.bond_dims() == st.bond_dims(), t
        sim.bp_converge(); st.bp_converge(1e-12); ref.bp_converge()
        cg, co = sim.correlation(), st.correlation()
        assert abs(cg - co) < 1e-9, (t, cg, co)
        sep = max(sep, abs(cg - ref.correlation()))
    for e in range(sim.n_bonds):
        assert np.allclose(sim.get_lambda(e), st.lam[e], rtol=0, atol=1e-9)
    assert sep > 1e-9                        # the BP gauge does change the truncated run (oracle: 1e-7 by step 20)
    sim.check_guards()
    sim.close(); ref.close()
    a = B.Pepo(1, 5, 0, 2, J, H, DT, 8, 1e-12, 0.0)
    b = B.Pepo(1, 5, 0, 2, J, H, DT, 8, 1e-12, 0.0)
    b.set_option("env", 1)
    for t in range(10):
        b.set_lambda(0, b.get_lambda(0))
        b.norm_bp_converge(1e-13, 0.0, 50)
        a.trotter_step(); b.trotter_step()
        a.bp_converge(); b.bp_converge()
        assert abs(a.correlation() - b.correlation()) < 1e-10
    a.close(); b.close()
