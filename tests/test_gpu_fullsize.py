"""GPU parity at BASELINE.json's full sizes (-m gpu), in the launch configuration bench.py times:

* config 3: all 120 permutations of the (4,40,40,40,40) tensor bit-exact; Cholesky-QR of the
  256000 x 40 / 256000 x 160 matrices against the oracle's Householder QR;
* config 2 sizes: gate replay on the seeded synthetic saturated 4x4 chi = 60 state - the oracle's
  single Algorithm-1 gate on the same inputs, compared through gauge-invariant quantities
  (lambda, chi_new, sampled entries of the two-site tensor; reading R17);
* config 2 physics: the first steps of the real 4x4 chi_max = 60 run against the oracle
  trajectory (bonds still small, so the oracle finishes in seconds) and, on the saturated state
  bench.py times, properties that hold at any size (normalised lambda, descending spectrum,
  read-only BP, |C| <= 1).
"""
import itertools

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


def test_config3_all_120_permutations_bit_exact(gpu):
    torch, B = gpu
    from paper_2606_30985_b200 import inputs
    chi = 40
    shape = [chi, chi, chi, chi, 4]                       # column-major dims of C-order (4,chi,chi,chi,chi)
    src = inputs.normal_tensor(shape, seed=1)
    d_src = torch.from_numpy(src).cuda()
    d_dst = torch.empty_like(d_src)
    # oracle on the full tensor: the definition itself (R10 = numpy.transpose on the column-major
    # shape; oracle.permute_listing1 is pinned to it on small tensors in tests/test_oracle_pins.py)
    t = src.reshape(shape, order="F")
    for perm in itertools.permutations(range(5)):
        want = np.transpose(t, perm).flatten(order="F")
        got = B.permute(d_src, shape, perm, dst=d_dst).cpu().numpy()
        assert np.array_equal(got.view(np.int64), want.view(np.int64)), perm


@pytest.mark.parametrize("m,n", [(256000, 40), (256000, 160)])
def test_config3_cholqr_vs_oracle(gpu, m, n):
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    A = inputs.normal_tensor((m, n), seed=1).reshape((m, n), order="F")
    d_A = torch.from_numpy(np.asfortranarray(A).flatten(order="F")).cuda()
    Q, R, info = B.cholqr(d_A, m, n)
    assert int(info.item()) == 0
    Qh = Q.cpu().numpy().reshape((m, n), order="F")
    Rh = R.cpu().numpy().reshape((n, n), order="F")
    assert np.allclose(np.tril(Rh, -1), 0.0)
    fro = np.linalg.norm(A)
    assert np.linalg.norm(Qh @ Rh - A) / fro <= 1e-12
    assert np.linalg.norm(Qh.T @ Qh - np.eye(n)) <= 1e-11
    # against the oracle's Householder factor, rows sign-normalised (unique for full column rank)
    _, Ro = po.householder_qr(A)
    sg = np.sign(np.diag(Rh)) * np.sign(np.diag(Ro))
    assert np.linalg.norm(Rh - sg[:, None] * Ro) / np.linalg.norm(Ro) <= 1e-11


def _load_synthetic(sim, Lx, Ly, chi):
    from paper_2606_30985_b200 import inputs
    chis, psi, lam = inputs.synthetic_state(Lx, Ly, chi)
    sim.set_bond_dims(chis)
    for e, l in enumerate(lam):
        sim.set_lambda(e, l)
    for v, t in psi.items():
        sim.set_site(v % Lx, v // Lx, t)
    return chis, psi, lam


def _oracle_state(Lx, Ly, chi, only_sites=None):
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    st = po.PEPOState(Lx, Ly, 1, 1, J, H, DT, chi)
    chis, psi, lam = inputs.synthetic_state(Lx, Ly, chi)
    for v in range(Lx * Ly):
        if only_sites is not None and v not in only_sites:
            continue
        x, y = v % Lx, v // Lx
        dims = [chis[inputs.bond_id(Lx, Ly, x, y, d)] for d in inputs.site_legs(Lx, Ly, x, y)] + [4]
        st.psi[v] = np.asarray(psi[v]).reshape(dims, order="F").copy()
    st.lam = [np.asarray(l) for l in lam]
    return st


def _two_site_samples(t1, ax1, t2, ax2, idx1, idx2):
    """Theta[i1, i2] = sum_c t1[i1 with cut=c] t2[i2 with cut=c] on sampled multi-indices."""
    a = np.moveaxis(t1, ax1, -1)
    b = np.moveaxis(t2, ax2, -1)
    return np.einsum("sc,sc->s", a[tuple(idx1.T)], b[tuple(idx2.T)])


def _gate_replay(B, Lx, Ly, chi, bond, seed, ns=6000, max_inflight=0, opts=None):
    """One Algorithm-1 gate on the seeded synthetic state, GPU vs oracle, through
    gauge-invariant quantities (R17): chi_new, lambda, and the gated two-site tensor Theta = psi1 . psi2
    on sampled entries in the ENVIRONMENT-WEIGHTED norm - the norm the simple update optimises and the
    one the oracle's own pin uses (tests/test_oracle_pins.py::test_gate_update_preserves_two_site_operator):
    the de-absorb division by sqrt(lambda) (lambda graded over six decades here) amplifies rounding of
    the small-weight rows by up to 1e3 per leg in the unweighted norm, on both sides alike.
    Tolerance: 1e-12 relative (north_star: QR/SVD reconstructions within 1e-12 relative Frobenius)."""
    from paper_2606_30985_b200 import inputs
    sim = B.Pepo(Lx, Ly, 1, 1, J, H, DT, chi, 1e-10, 0.5, max_inflight=max_inflight)
    for k, v in (opts or {}).items():
        sim.set_option(k, v)
    _load_synthetic(sim, Lx, Ly, chi)
    nh = Ly * (Lx - 1)
    if bond < nh:
        v1 = (bond // (Lx - 1)) * Lx + bond % (Lx - 1); v2 = v1 + 1
    else:
        v1 = bond - nh; v2 = v1 + Lx
    st = _oracle_state(Lx, Ly, chi, only_sites=(v1, v2))
    sim.apply_bond(bond)
    st.apply_bond_gate(bond)
    assert sim.bond_dims()[bond] == st.lam[bond].size == chi
    lam_g = sim.get_lambda(bond)
    # lambda_k are singular values / norm: absolute accuracy u * s_0 each (1e-13 of the largest)
    assert np.max(np.abs(lam_g - st.lam[bond])) <= 1e-13
    assert np.allclose(lam_g, st.lam[bond], rtol=1e-9, atol=1e-13)
    _, d1, _, d2 = st.lat.bond_sites(bond)
    legs1, legs2 = st.lat.legs(v1), st.lat.legs(v2)
    g1 = sim.get_site(v1 % Lx, v1 // Lx).reshape(st.psi[v1].shape, order="F")
    g2 = sim.get_site(v2 % Lx, v2 // Lx).reshape(st.psi[v2].shape, order="F")
    ax1, ax2 = legs1.index(d1), legs2.index(d2)
    rng = np.random.default_rng(seed)
    def sample(shape):
        cols = []
        for s_ in shape:
            u = rng.random(ns)
            u[ns // 2:] = u[ns // 2:] ** 3            # half the samples biased to the heavy (small-index) rows
            cols.append(np.minimum((u * s_).astype(np.int64), s_ - 1))
        return np.stack(cols, axis=1)
    def weights(v, legs, ax, idx):
        w = np.ones(ns)
        col = 0
        for a, d in enumerate(legs):
            if a == ax:
                continue
            w *= np.sqrt(st.lam[st.lat.bond_id(v, d)])[idx[:, col]]
            col += 1
        return w
    idx1 = sample([s_ for a, s_ in enumerate(g1.shape) if a != ax1])
    idx2 = sample([s_ for a, s_ in enumerate(g2.shape) if a != ax2])
    w = weights(v1, legs1, ax1, idx1) * weights(v2, legs2, ax2, idx2)
    th_g = _two_site_samples(g1, ax1, g2, ax2, idx1, idx2)
    th_o = _two_site_samples(st.psi[v1], ax1, st.psi[v2], ax2, idx1, idx2)
    rel = np.linalg.norm((th_g - th_o) * w) / np.linalg.norm(th_o * w)
    s = sim.stats()
    sim.close()
    return rel, s


@pytest.mark.parametrize("which", ["corner-edge", "edge-interior", "interior-interior"])
def test_gate_replay_4x4_chi60(gpu, which):
    """One Algorithm-1 gate at config 2's full size (chi = 60, m up to 216000) on the same seeded inputs."""
    torch, B = gpu
    from paper_2606_30985_b200 import inputs
    L, chi = 4, 60
    bond = {"corner-edge": inputs.bond_id(L, L, 0, 0, "R"),
            "edge-interior": inputs.bond_id(L, L, 0, 1, "R"),
            "interior-interior": inputs.bond_id(L, L, 1, 1, "R")}[which]
    rel, _ = _gate_replay(B, L, L, chi, bond, seed=7)
    assert rel <= 1e-12, rel


@pytest.mark.parametrize("orient", [0, 1, 2])
def test_gate_replay_svd_orientation(gpu, orient):
    """Option svd_orient: the QR preconditioner of the Jacobi SVD on K (0), on K^T (2) or on whichever is
    more graded (1, default).  Every choice must give the oracle's gate to 1e-12 - orient 2
    forces the transposed iteration and the transposed bridges on a square 240 x 240 core - and the adaptive
    choice may not need more sweeps than the better of the two fixed ones (plus one)."""
    torch, B = gpu
    from paper_2606_30985_b200 import inputs
    L, chi = 4, 60
    bond = inputs.bond_id(L, L, 1, 1, "R")
    rel, s = _gate_replay(B, L, L, chi, bond, seed=7, opts={"svd_orient": orient})
    assert rel <= 1e-12, rel
    test_gate_replay_svd_orientation.sweeps[orient] = s["jacobi_sweeps"]
    if len(test_gate_replay_svd_orientation.sweeps) == 3:
        sw = test_gate_replay_svd_orientation.sweeps
        assert sw[1] <= min(sw[0], sw[2]) + 1, sw


test_gate_replay_svd_orientation.sweeps = {}


def test_gate_replay_config5_interior_shape(gpu):
    """BASELINE configs[4]'s interior-interior gate shape: m = chi^3 = 804357 >= 8e5 rows, n = 4 chi =
    372 columns per site, chi = 93 (the 10x10 run's chi_max is 94).  The smallest grid with two adjacent
    4-legged sites is 4x3; the oracle's single gate (Householder QR of two 804357 x 372 matrices and the
    SVD of the literal 1488 x 1488 core) takes about a minute."""
    torch, B = gpu
    from paper_2606_30985_b200 import inputs
    Lx, Ly, chi = 4, 3, 93
    bond = inputs.bond_id(Lx, Ly, 1, 1, "R")
    rel, s = _gate_replay(B, Lx, Ly, chi, bond, seed=13, max_inflight=1)
    assert s["n_cholesky"] == 2 and s["n_chol_failed"] == 0
    assert rel <= 1e-12, rel


def test_config2_first_steps_vs_oracle(gpu):
    """BASELINE configs[1] from the product operator: 8 steps (bonds up to ~41) against the oracle."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    steps = 8
    sim = B.Pepo(4, 4, 1, 1, J, H, DT, 60, 1e-10, 0.5)
    st = po.PEPOState(4, 4, 1, 1, J, H, DT, 60)
    for t in range(steps):
        sim.trotter_step()
        st.trotter_step()
        assert sim.bond_dims() == st.bond_dims(), (t + 1, sim.bond_dims(), st.bond_dims())
        sg, swg, _ = sim.bp_converge()
        so, swo, _ = st.bp_converge(1e-10, 0.5)
        assert sg == so and abs(swg - swo) <= 1
        assert abs(sim.correlation() - st.correlation()) <= 1e-10
    sim.close()


def test_config2_saturated_whole_step_vs_oracle(gpu):
    """BASELINE configs[1] at FULL size, one whole Trotter step + BP in the saturated regime (every bond = 60,
    truncation active: 24 Algorithm-1 gates with 240 x 240 cores, interior m = 216000): the CUDA path's own
    state after step 30 is loaded into the oracle (tests-only), both sides take step 31 from identical
    inputs.  Compared: every bond's lambda (gauge invariant), the discarded weight, C(t), BP status.
    The oracle needs 2-5 min for this step on the box's host cores."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    L, chi = 4, 60
    sim = B.Pepo(L, L, 1, 1, J, H, DT, chi, 1e-10, 0.5)
    for _ in range(30):
        sim.trotter_step()
    dims = sim.bond_dims()
    assert min(dims) == chi
    st = po.PEPOState(L, L, 1, 1, J, H, DT, chi)
    for e in range(sim.n_bonds):
        st.lam[e] = sim.get_lambda(e)
    for v in range(L * L):
        shape = [dims[st.lat.bond_id(v, d)] for d in st.lat.legs(v)] + [4]
        st.psi[v] = sim.get_site(v % L, v // L).reshape(shape, order="F").copy()
    st.trotter_step()
    so, swo, _ = st.bp_converge(1e-10, 0.5)
    sim.trotter_step()
    sg, swg, _ = sim.bp_converge()
    assert sim.bond_dims() == st.bond_dims()
    for e in range(sim.n_bonds):
        assert np.max(np.abs(sim.get_lambda(e) - np.asarray(st.lam[e]))) <= 1e-12, e
    ge = sim.stats()["gate_err"]
    assert ge > 1e-8 and abs(ge - st.gate_err) <= 1e-9 * st.gate_err          # truncation is active
    assert sg == so == 0 and abs(swg - swo) <= 2
    assert abs(sim.correlation() - st.correlation()) <= 1e-12
    sim.close()


def test_config2_saturated_properties(gpu):
    """On the state bench.py times (every bond = 60 after the physical preparation) no oracle run
    is affordable: check what holds at any size."""
    torch, B = gpu
    sim = B.Pepo(4, 4, 1, 1, J, H, DT, 60, 1e-10, 0.5)
    n = 0
    while min(sim.bond_dims()) < 60 and n < 40:
        sim.trotter_step()
        n += 1
    assert min(sim.bond_dims()) == 60
    sim.trotter_step()
    for e in range(sim.n_bonds):
        lam = sim.get_lambda(e)
        assert abs(np.linalg.norm(lam) - 1.0) < 1e-12
        assert np.all(np.diff(lam) <= 0) and lam[-1] > 0
    before = [sim.get_site(x, y).copy() for y in range(4) for x in range(4)]
    status, sweeps, delta = sim.bp_converge()
    c = sim.correlation()
    after = [sim.get_site(x, y) for y in range(4) for x in range(4)]
    assert all(np.array_equal(a, b) for a, b in zip(before, after))          # R16: BP is read-only
    assert status in (0, 1) and abs(c) <= 1.0 + 1e-9
    s = sim.stats()
    assert 0.0 <= s["gate_err"] < 1e-3
    assert s["arena_high_water"] <= s["arena_model_bytes"] * 1.02 + 65536
    sim.close()


@pytest.mark.parametrize("chi", [72, 100])
def test_gate_replay_large_core_3x3(gpu, chi):
    """Cores above 256 (chi 65..104) take the cluster-of-16 form of the Jacobi kernel:
    one Algorithm-1 gate on a corner-edge bond of the 3x3 chi = 72 / 100 synthetic state (core
    288^2 / 400^2) against the oracle on the same seeded inputs."""
    torch, B = gpu
    from paper_2606_30985_b200 import inputs
    bond = inputs.bond_id(3, 3, 0, 0, "R")
    rel, _ = _gate_replay(B, 3, 3, chi, bond, seed=11)
    assert rel <= 1e-12, rel
