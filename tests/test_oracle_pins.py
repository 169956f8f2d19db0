"""Pins of the CPU oracle against things other than itself.

All -m "not gpu".  Paper citations are /root/reference/PAPER.md lines.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import dense_check as dc
from oracle import pepo_oracle as po

J, H, DT = 1.0, 0.9, 0.05


# ---------------------------------------------------------------- gates (R2, R15) ---------
def test_field_gate_is_yz_rotation():
    """PTM of exp(+i theta X): I, X fixed; c_Y' = cos2t c_Y - sin2t c_Z, c_Z' = sin2t c_Y + cos2t c_Z."""
    th = H * DT
    G = po.ptm_one_site(th, "X")
    c, s = math.cos(2 * th), math.sin(2 * th)
    expect = np.array([[1, 0, 0, 0], [0, 1, 0, 0], [0, 0, c, -s], [0, 0, s, c]])
    assert np.allclose(G, expect, atol=1e-15)
    assert np.allclose(G @ G.T, np.eye(4), atol=1e-15)      # real orthogonal


def test_zz_gate_structure():
    """R15: closed-form entries of the ZZ PTM, orthogonality, operator-Schmidt rank 4."""
    th = J * DT
    G = po.ptm_two_site(th, "Z")
    c, s = math.cos(2 * th), math.sin(2 * th)
    assert np.allclose(G @ G.T, np.eye(16), atol=1e-14)
    idx = lambda a, b: "IXYZ".index(a) * 4 + "IXYZ".index(b)
    for ab in ["II", "IZ", "ZI", "ZZ", "XX", "XY", "YX", "YY"]:
        assert abs(G[idx(*ab), idx(*ab)] - 1) < 1e-15
    for ab in ["IX", "IY", "XI", "YI", "ZX", "ZY", "XZ", "YZ"]:
        assert abs(G[idx(*ab), idx(*ab)] - c) < 1e-15
    pairs = [("IX", "ZY", -s), ("ZY", "IX", +s), ("IY", "ZX", +s), ("ZX", "IY", -s),
             ("XI", "YZ", -s), ("YZ", "XI", +s), ("YI", "XZ", +s), ("XZ", "YI", -s)]
    off = np.zeros((16, 16))
    for (r, cc, v) in pairs:
        assert abs(G[idx(*r), idx(*cc)] - v) < 1e-15
        off[idx(*r), idx(*cc)] = v
    assert np.allclose(G - np.diag(np.diag(G)), off, atol=1e-15)       # nothing else off-diagonal
    # operator-Schmidt rank across site1|site2
    T = G.reshape(4, 4, 4, 4).transpose(0, 2, 1, 3).reshape(16, 16)
    sv = np.linalg.svd(T, compute_uv=False)
    assert np.sum(sv > 1e-12) == 4
    assert np.allclose(sv[:4], [3.990, 0.1997, 0.1997, 0.00999], atol=2e-3)


def test_gate_ptm_matches_dense_conjugation():
    """One ZZ gate + field gate on 2 sites through the PTM equals 4x4 dense conjugation."""
    rng = np.random.default_rng(0)
    coef = rng.standard_normal(16)
    paulis = [dc._SIG[k] for k in "IXYZ"]
    O = sum(coef[a * 4 + b] * np.kron(paulis[a], paulis[b]) for a in range(4) for b in range(4))
    U = dc._expm_herm(np.kron(paulis[3], paulis[3]), 1j * J * DT)
    O2 = U.conj().T @ O @ U
    c2 = po.ptm_two_site(J * DT, "Z") @ coef
    O2p = sum(c2[a * 4 + b] * np.kron(paulis[a], paulis[b]) for a in range(4) for b in range(4))
    assert np.allclose(O2, O2p, atol=1e-14)


# ---------------------------------------------------------------- P1 / P2 / P3 / P4 ---------
@pytest.mark.parametrize("case", [(2, 2, 0, 0), (3, 3, 1, 1), (1, 4, 0, 1), (2, 3, 0, 1)])
def test_untruncated_network_equals_dense(case, golden_dense):
    """P1+P2: exact contraction of the untruncated network = dense Trotter evolution (<=1e-13 for 4 steps, <=1e-10 for 8);
    P4: BP/Bethe within 1e-10 of dense for <=8 steps on loopy grids."""
    Lx, Ly, cx, cy = case
    gold = golden_dense[case]
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, chi_max=256)
    for step in range(8):
        st.trotter_step()
        # eps_cut=1e-11 pruning itself moves the network by ~1e-11 from step ~5 on (R8 note)
        assert abs(st.exact_contraction() - gold[step]) < (1e-13 if step < 4 else 1e-10), (case, step)
        status, sweeps, delta = st.bp_converge(1e-12, 0.0, 200)
        assert status == 0
        assert abs(st.correlation() - gold[step]) < 1e-10, (case, step)


def test_golden_file_is_what_dense_check_computes(golden_dense):
    vals = dc.dense_trotter_correlation(2, 2, 0, 0, J, H, DT, 10)
    assert np.allclose(vals, golden_dense[(2, 2, 0, 0)], atol=1e-14)
    # step 1 = cos(2 h dt) on every grid: ZZ commutes with Z_c
    for k, v in golden_dense.items():
        assert abs(v[0] - math.cos(2 * H * DT)) < 1e-14


@pytest.mark.parametrize("case", [(1, 4, 0, 1), (1, 6, 0, 2)])
def test_bp_exact_on_trees(case, golden_dense):
    """P3: BP is exact on trees: 1xN chains, untruncated, 10 steps."""
    Lx, Ly, cx, cy = case
    st, out = po.run_trajectory(Lx, Ly, cx, cy, J, H, DT, 256, 10, 1e-13)
    for o, g in zip(out, golden_dense[case]):
        assert abs(o["C"] - g) < 1e-13


def test_chain_orientation_equivalence(golden_dense):
    """Nx1 equals 1xN (legs L/R instead of U/D exercise the other permutation cases)."""
    st, out = po.run_trajectory(4, 1, 1, 0, J, H, DT, 256, 10, 1e-13)
    for o, g in zip(out, golden_dense[(1, 4, 0, 1)]):
        assert abs(o["C"] - g) < 1e-13


# ---------------------------------------------------------------- P5 closed forms -----------
def test_closed_forms():
    """J=0: C(n dt) = cos(2 h n dt), all chi stay 1.  h=0: C == 1, all chi stay 1.  C(0)=1 (L350)."""
    st = po.PEPOState(3, 3, 1, 1, 0.0, H, DT, 8)
    st.bp_converge(1e-12)
    assert abs(st.correlation() - 1.0) < 1e-15          # C(0) = 1
    for n in range(1, 7):
        st.trotter_step()
        st.bp_converge(1e-12)
        assert abs(st.correlation() - math.cos(2 * H * n * DT)) < 1e-14
        assert set(st.bond_dims()) == {1}
    st = po.PEPOState(3, 3, 1, 1, J, 0.0, DT, 8)
    for n in range(1, 5):
        st.trotter_step()
        st.bp_converge(1e-12)
        assert abs(st.correlation() - 1.0) < 1e-14
        assert set(st.bond_dims()) == {1}


# ---------------------------------------------------------------- P6 config 1 ---------------
def test_config1_close_to_dense(golden_dense):
    """BASELINE config 1 (3x3, chi_max=8, truncating from step 4) stays within 5e-9 of dense."""
    st, out = po.run_trajectory(3, 3, 1, 1, J, H, DT, 8, 10, 1e-10, 0.0)
    gold = golden_dense[(3, 3, 1, 1)]
    assert max(st.bond_dims()) == 8
    for o, g in zip(out, gold):
        assert o["status"] == 0
        assert abs(o["C"] - g) < 5e-9


# ---------------------------------------------------------------- P7 / P8 / P13 -------------
def test_c4_symmetry_and_lightcone():
    st = po.PEPOState(5, 5, 2, 2, J, H, DT, 64)
    lat = st.lat
    expected = {1: [2, 1, 1, 1], 2: [4, 2, 1, 1], 3: [9, None, 2, 1], 4: [15, None, 5, 2]}
    for step in range(1, 5):
        st.trotter_step()
        dims = st.bond_dims()
        by_d = {}
        for e in range(lat.n_bonds):
            v1, _, v2, _ = lat.bond_sites(e)
            d = min(abs(x - 2) + abs(y - 2) for (x, y) in (lat.xy(v1), lat.xy(v2)))
            by_d.setdefault(d, set()).add(dims[e])
        for d, want in enumerate(expected[step]):
            if want is not None:
                assert by_d[d] == {want}, (step, d, by_d)
    # P7: the four bonds touching the centre have identical Schmidt spectra (C4)
    c = lat.site(2, 2)
    spectra = [st.lam[lat.bond_id(c, d)] for d in "UDLR"]
    for s in spectra[1:]:
        assert np.allclose(s, spectra[0], atol=1e-12)


def test_exact_symmetries_of_C():
    """P13: C(J,h) = C(-J,h) = C(J,-h); reflection (1,1) == (2,2) on 4x4."""
    ref = [o["C"] for o in po.run_trajectory(4, 4, 1, 1, J, H, DT, 8, 8, 1e-12)[1]]
    for (j, h, cx, cy) in [(-J, H, 1, 1), (J, -H, 1, 1), (J, H, 2, 2), (J, H, 2, 1)]:
        got = [o["C"] for o in po.run_trajectory(4, 4, cx, cy, j, h, DT, 8, 8, 1e-12)[1]]
        if (cx, cy) == (2, 1):
            ref2 = [o["C"] for o in po.run_trajectory(4, 4, 1, 2, J, H, DT, 8, 8, 1e-12)[1]]
            assert np.allclose(got, ref2, atol=1e-12)
        else:
            assert np.allclose(got, ref, atol=1e-12)


def test_grid_independence_early_times():
    """P8 / PAPER L364: C identical across grids until the front returns from the boundary."""
    a = [o["C"] for o in po.run_trajectory(3, 3, 1, 1, J, H, DT, 8, 2, 1e-12)[1]]
    b = [o["C"] for o in po.run_trajectory(4, 4, 1, 1, J, H, DT, 8, 2, 1e-12)[1]]
    assert np.allclose(a, b, atol=1e-14)


def test_bp_is_read_only():
    """R16: bp_converge / correlation do not change (psi, lambda)."""
    s1 = po.PEPOState(3, 3, 1, 1, J, H, DT, 8)
    s2 = po.PEPOState(3, 3, 1, 1, J, H, DT, 8)
    for _ in range(5):
        s1.trotter_step(); s1.bp_converge(1e-10); s1.correlation()
        s2.trotter_step()
    for a, b in zip(s1.psi, s2.psi):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------- P9 permutation ------------
def test_permutation_listing1_vs_loops_and_transpose():
    rng = np.random.default_rng(3)
    shape = [3, 2, 4, 2, 4]
    src = rng.standard_normal(int(np.prod(shape)))
    arr = src.reshape(shape, order="F")
    for perm in itertools.permutations(range(5)):
        got = po.permute_listing1(src, shape, perm)
        assert np.array_equal(got, np.transpose(arr, perm).flatten(order="F"))
    for perm in [(0, 1, 2, 3, 4), (1, 2, 3, 0, 4), (4, 3, 2, 1, 0), (2, 0, 4, 1, 3)]:
        got = po.permute_listing1(src, shape, perm)
        assert np.array_equal(got, po.permute_nested_loops(src, shape, perm))
        inv = np.argsort(perm)
        back = po.permute_listing1(got, [shape[p] for p in perm], list(inv))
        assert np.array_equal(back, src)                       # perm o perm^-1 = identity
    # bijection: permuting arange gives a permutation of arange
    ar = np.arange(src.size, dtype=np.float64)
    assert np.array_equal(np.sort(po.permute_listing1(ar, shape, (3, 1, 4, 0, 2))), ar)
    # rank 3 / rank 1 / size-1 dims
    assert np.array_equal(po.permute_listing1(ar[:6], [2, 3, 1], (1, 2, 0)),
                          np.transpose(ar[:6].reshape([2, 3, 1], order="F"), (1, 2, 0)).flatten(order="F"))


# ---------------------------------------------------------------- P10 QR / SVD --------------
def test_qr_invariants_and_cholqr_agrees():
    rng = np.random.default_rng(5)
    for (m, n) in [(50, 8), (8, 8), (5, 12), (300, 24)]:
        A = rng.standard_normal((m, n))
        Q, R = po.householder_qr(A)
        k = min(m, n)
        assert Q.shape == (m, k) and R.shape == (k, n)
        assert np.linalg.norm(A - Q @ R) / np.linalg.norm(A) < 1e-13
        assert np.linalg.norm(Q.T @ Q - np.eye(k)) < 1e-13
        assert np.allclose(R, np.triu(R))
        if m >= n:
            Qc, Rc = po.cholesky_qr(A)                          # eq. (10)
            assert np.all(np.diag(Rc) > 0) and np.allclose(Rc, np.triu(Rc))
            assert np.linalg.norm(A - Qc @ Rc) / np.linalg.norm(A) < 1e-13
            assert np.linalg.norm(Qc.T @ Qc - np.eye(n)) < 1e-10
            sgn = np.sign(np.diag(R))
            assert np.allclose(Rc, sgn[:, None] * R, atol=1e-10)   # QR unique up to row signs of R
    with pytest.raises(np.linalg.LinAlgError):
        A = rng.standard_normal((20, 4)); A[:, 3] = 0.0
        po.cholesky_qr(A)                                       # potrf_info != 0


def test_truncation_rule():
    s = np.array([1.0, 0.5, 1e-3, 2e-11, 1e-11, 0.9e-11, 0.0])
    assert po.truncation_rank(s, 100, 1e-11) == 5               # eq. (11): s_i >= eps*s_0 inclusive
    assert po.truncation_rank(s, 3, 1e-11) == 3
    assert po.truncation_rank(np.zeros(3), 3, 1e-11) == 0


def test_gate_update_preserves_two_site_operator():
    """A single untruncated Alg.1 equals the gate applied to the contracted two-site tensor, and
    lambda are the singular values of the environment-weighted two-site tensor (Vidal gauge)."""
    st = po.PEPOState(2, 3, 0, 1, J, H, DT, 256)
    for _ in range(3):
        st.trotter_step()
    st.apply_field_gate()
    lat = st.lat
    e = lat.bond_id(lat.site(0, 1), "R")
    v1, d1, v2, d2 = lat.bond_sites(e)
    a, b = st.psi[v1].copy(), st.psi[v2].copy()
    # theta[u1,d1_,p1,u2,d2_,p2] = sum_c a[u,d,c(R),p] b[u,d,c(L),p]; legs of v1: U,D,R ; v2: U,D,L
    theta = np.einsum("udcp,efcq->udpefq", a, b)
    G4 = st.G2.reshape(4, 4, 4, 4)
    want = np.einsum("xypq,udpefq->udxefy", G4, theta)
    st.apply_bond_gate(e)
    got = np.einsum("udcp,efcq->udpefq", st.psi[v1], st.psi[v2])
    # equality holds in the environment-weighted norm the simple update optimises (the 1e-11 pruning of
    # eq. (11) is amplified by the deabsorb division in the unweighted norm)
    w = lambda v: (np.sqrt(st.lam[lat.bond_id(v, "U")])[:, None] * np.sqrt(st.lam[lat.bond_id(v, "D")])[None, :])
    W = w(v1)[:, :, None, None, None, None] * w(v2)[None, None, None, :, :, None]
    assert np.linalg.norm((got - want) * W) / np.linalg.norm(want * W) < 1e-10
    assert abs(np.sum(st.lam[e] ** 2) - 1) < 1e-14 and np.all(np.diff(st.lam[e]) <= 0)


# ---------------------------------------------------------------- P11 memory model ----------
def test_paper_memory_model_tables():
    """eq. (15)-(17) with sizeof(float)=4 reproduce Table 9 (L649-L656) and Table 10 (L660-L670), decimal GB."""
    gb = lambda k, l, chi: sum(po.paper_memory_model_bytes(k, l, chi)) / 1e9
    assert abs(gb(4, 4, 50) - 0.82) < 0.005
    assert abs(gb(4, 4, 80) - 5.31) < 0.005
    assert abs(gb(4, 4, 100) - 12.94) < 0.005
    assert abs(gb(10, 10, 100) - 109.3) < 0.05
    assert abs(gb(8, 8, 90) - 42.3) < 0.05
    assert abs(gb(5, 5, 70) - 5.1) < 0.05
    lat = po.Lattice(8, 8)
    assert lat.n_bonds == 2 * 8 * 7
    cls = lat.colour_classes()
    assert sorted(sum(cls, [])) == list(range(lat.n_bonds))
    for c in cls:                                               # no shared site in a class
        seen = set()
        for e in c:
            v1, _, v2, _ = lat.bond_sites(e)
            assert v1 not in seen and v2 not in seen
            seen.update((v1, v2))


# ---------------------------------------------------------------- symmetric step, eq. (6) --
@pytest.mark.parametrize("case", [(2, 2, 0, 0), (2, 3, 0, 1), (1, 4, 0, 1)])
def test_symmetric_step_equals_dense_symmetric_splitting(case):
    """SURVEY NEXT-3 / PAPER eq. (6): order = 2 is R(h dt/2) - bond sweep - R(h dt/2).
    The untruncated oracle (exact contraction on grids, BP on the tree) must equal the dense
    2^N evolution with U = e^{i dt Hf/2} e^{i dt Hb} e^{i dt Hf/2} (an implementation that shares
    nothing with it), with the tolerances of the first-order pin P1/P2 (pruning at eps_cut moves
    the network by ~1e-11 from step ~5 on)."""
    Lx, Ly, cx, cy = case
    steps = 8
    dense = dc.dense_trotter_correlation(Lx, Ly, cx, cy, J, H, DT, steps, order=2)
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, 256, order=2)
    for n in range(steps):
        st.trotter_step()
        if min(Lx, Ly) == 1:
            st.bp_converge(1e-13)
            c = st.correlation()
        else:
            c = st.exact_contraction()
        assert abs(c - dense[n]) < (1e-13 if n < 4 else 1e-10), (case, n, c, dense[n])


def test_symmetric_step_is_second_order_and_keeps_closed_forms():
    """Against the exact propagator e^{-iHt} on 3x3, halving dt must cut the error of the symmetric
    splitting about fourfold (O(dt^2) at fixed t).  (For this observable the first-order product is
    a similarity transform of the symmetric one, U_f U_b = U_f^{1/2} U_sym U_f^{-1/2}, so its error
    in C(t) is O(dt^2) too: 5.6e-4 against 1.1e-3 at dt = 0.05 - the two differ, which is what makes
    the dense pin above discriminating.)  Closed forms (P5): at J = 0 two half rotations are one
    full rotation, C(n dt) = cos(2 h n dt); at h = 0, C = 1."""
    t = 0.5
    exact = dc.dense_exact_correlation(3, 3, 1, 1, J, H, t)
    e1 = abs(dc.dense_trotter_correlation(3, 3, 1, 1, J, H, 0.05, 10, order=1)[-1] - exact)
    e2 = abs(dc.dense_trotter_correlation(3, 3, 1, 1, J, H, 0.05, 10, order=2)[-1] - exact)
    e2h = abs(dc.dense_trotter_correlation(3, 3, 1, 1, J, H, 0.025, 20, order=2)[-1] - exact)
    assert abs(e2 - e1) > 1e-4, (e1, e2)
    assert 3.6 < e2 / e2h < 4.4, (e2, e2h)
    st = po.PEPOState(3, 3, 1, 1, 0.0, H, DT, 8, order=2)
    for n in range(1, 6):
        st.trotter_step()
        st.bp_converge(1e-12)
        assert abs(st.correlation() - math.cos(2 * H * n * DT)) < 1e-13
        assert max(st.bond_dims()) == 1
    st = po.PEPOState(3, 3, 1, 1, J, 0.0, DT, 8, order=2)
    for n in range(3):
        st.trotter_step()
        st.bp_converge(1e-12)
        assert abs(st.correlation() - 1.0) < 1e-13


# ---------------------------------------------------------------- diagnostics (Table 1) ----
def test_bond_weights_and_entropy_equal_dense_operator_schmidt_on_a_chain():
    """SURVEY NEXT-2 / PAPER Table 1 (L373-L380): S_e = -sum lambda^2 log lambda^2.  On a chain (a
    tree) the untruncated simple-update weights lambda_e are the operator-Schmidt coefficients of
    Z_c(t) across the bond, which the dense 2^N evolution gives independently; closed forms:
    S = 0 for the product operator, S = log chi for a flat spectrum."""
    n, c, steps = 4, 1, 5
    st = po.PEPOState(1, n, 0, c, J, H, DT, 64)
    assert all(st.bond_entropy(e) == 0.0 for e in range(st.lat.n_bonds))
    for _ in range(steps):
        st.trotter_step()
    for cut in range(n - 1):
        e = st.lat.bond_id(st.lat.site(0, cut), "D")
        s = dc.dense_chain_operator_schmidt(n, c, J, H, DT, steps, cut)
        lam = st.lam[e]
        # weights down to ~1e-10 are kept; those below 1e-8 carry the 1e-11 pruning of eq. (11)
        assert np.allclose(lam, s[:lam.size], rtol=0, atol=1e-10), (cut, lam, s[:lam.size])
        assert np.all(s[lam.size:] < 1e-9)
        w = s[s > 1e-14] ** 2
        assert abs(st.bond_entropy(e) - float(-(w * np.log(w)).sum())) < 1e-9
    st.lam[0] = np.full(8, 1 / math.sqrt(8))
    assert abs(st.bond_entropy(0) - math.log(8)) < 1e-14


# ---------------------------------------------------------------- damped BP (eq. (19), R7) ---
def _state_4x4_chi8(steps):
    st = po.PEPOState(4, 4, 1, 1, J, H, DT, 8)
    for _ in range(steps):
        st.trotter_step()
    return st


def test_damped_sweep_is_eq19_without_renormalisation():
    """eq. (19) PAPER L444-L449 with d = 1 - alpha (R7): one damped sweep from the init m0 = 1/sqrt(chi)
    equals d*m0 + (1-d)*mhat, where mhat is what ONE UNDAMPED sweep from the same init gives (normalised,
    sign-aligned); no renormalisation afterwards.  d = 0.3 tells d from 1-d; the norm of the result is
    d^2 + (1-d)^2 + 2d(1-d)<m0,mhat> < 1 whenever mhat != m0."""
    st = _state_4x4_chi8(12)
    d = 0.3
    st.bp_converge(1e-30, 0.0, max_sweeps=1)
    mhat = {k: v.copy() for k, v in st.msgs.items()}
    status, sweeps, _ = st.bp_converge(1e-30, d, max_sweeps=0, max_sweeps_damped=1)
    assert (status, sweeps) == (1, 1)
    some_shorter = False
    for k, m1 in st.msgs.items():
        chi = m1.size
        m0 = np.full(chi, 1.0 / math.sqrt(chi))
        assert abs(np.linalg.norm(mhat[k]) - 1.0) < 1e-14 and float(mhat[k] @ m0) >= 0.0
        assert np.allclose(m1, d * m0 + (1 - d) * mhat[k], rtol=0, atol=1e-15)
        some_shorter |= np.linalg.norm(m1) < 1.0 - 1e-6
    assert some_shorter


@pytest.mark.parametrize("grid,steps", [((3, 3, 1, 1), 8), ((4, 4, 1, 1), 30)])
def test_damped_restart_lands_on_the_undamped_fixed_point(grid, steps):
    """phase 2 (restart from the init with damping) converges to the same fixed
    point as the undamped iteration, so the Bethe value agrees to rounding; forced here by a phase-1
    budget of one sweep."""
    st = po.PEPOState(*grid, J, H, DT, 8)
    for _ in range(steps):
        st.trotter_step()
    s0, n0, _ = st.bp_converge(1e-13, 0.0)
    c0 = st.correlation()
    m0 = {k: v.copy() for k, v in st.msgs.items()}
    s1, n1, d1 = st.bp_converge(1e-13, 0.5, max_sweeps=1)
    c1 = st.correlation()
    assert s0 == 0 and s1 == 0 and d1 < 1e-13
    assert n1 > n0 + 1                       # 1 undamped sweep + a slower damped run
    assert abs(c1 - c0) <= 1e-14 * max(1.0, abs(c0)) + 1e-15
    for k in m0:
        # same ray and the same norm 1 (the fixed point of the un-renormalised damped iteration); the
        # overall sign of a message is a free choice of the iteration history (C does not depend on it)
        a, b = st.msgs[k], m0[k]
        assert min(np.abs(a - b).max(), np.abs(a + b).max()) < 1e-10


def test_damped_contraction_rate_obeys_eq19():
    """Linearised eq. (19): the damped iteration matrix is d*I + (1-d)*Jac, so with rho the late-time
    undamped ratio delta_{k+1}/delta_k the damped ratio lies in [d - (1-d) rho, d + (1-d) rho].  With
    d = 0.75 and rho <= 0.4 that is [0.65, 0.85]; swapping d and 1-d would give <= 0.55."""
    st = _state_4x4_chi8(30)
    rates = {}
    for d in (0.0, 0.75):
        msgs, dl = st._init_messages(), []
        for _ in range(400):
            msgs, de, _ = st._bp_sweep(msgs, d)
            dl.append(de)
            if de < 1e-12:
                break
        r = [dl[i + 1] / dl[i] for i in range(len(dl) - 1)]
        rates[d] = r[-8:]
    rho = max(rates[0.0])
    assert rho < 0.4
    for r in rates[0.75]:
        assert 0.75 - 0.25 * rho - 0.01 <= r <= 0.75 + 0.25 * rho + 0.01, (r, rho)


def test_exhausted_budget_and_restart_from_the_init():
    """when both budgets are spent bp_converge returns status 1 with the sweep count
    = both budgets and delta >= tol; the messages stay usable (finite C).  The damped phase restarts
    from the init (L456 'retry'): its result does not depend on how long phase 1 ran."""
    st = _state_4x4_chi8(40)
    s, n, de = st.bp_converge(1e-10, 0.5, max_sweeps=3, max_sweeps_damped=4)
    assert (s, n) == (1, 7) and de >= 1e-10
    ma = {k: v.copy() for k, v in st.msgs.items()}
    ca = st.correlation()
    assert math.isfinite(ca)
    s, n, de2 = st.bp_converge(1e-10, 0.5, max_sweeps=6, max_sweeps_damped=4)
    assert (s, n) == (1, 10) and de2 == de
    for k in ma:
        assert np.array_equal(ma[k], st.msgs[k])
    # no damping configured: only phase 1 runs
    s, n, _ = st.bp_converge(1e-10, 0.0, max_sweeps=3, max_sweeps_damped=4)
    assert (s, n) == (1, 3)
    # golden trajectory (tests/golden/oracle_4x4_chi8.txt): step 49 needs the damped restart, 100 + 60 sweeps
    for _ in range(9):
        st.trotter_step()
    s, n, _ = st.bp_converge(1e-10, 0.5)
    assert s == 0 and n > 100


def test_lambda_is_normalised_over_the_kept_values_when_truncating():
    """eq. (11)-(12), R8, on a gate that DOES truncate: chi_new = chi_max and lambda = s[:chi]/||s[:chi]||
    with s the singular values of the gated, environment-weighted two-site tensor (computed here from
    the contracted tensor, not from the QR cores); gate_err = discarded weight."""
    st = po.PEPOState(2, 3, 0, 1, J, H, DT, 3)
    for _ in range(4):
        st.trotter_step()
    st.apply_field_gate()
    lat = st.lat
    e = lat.bond_id(lat.site(0, 1), "R")
    v1, d1, v2, d2 = lat.bond_sites(e)
    a, b = st.psi[v1].copy(), st.psi[v2].copy()
    w = lambda v: (np.sqrt(st.lam[lat.bond_id(v, "U")])[:, None] * np.sqrt(st.lam[lat.bond_id(v, "D")])[None, :])
    theta = np.einsum("udcp,efcq->udpefq", a * w(v1)[:, :, None, None], b * w(v2)[:, :, None, None])
    theta = np.einsum("xypq,udpefq->udxefy", st.G2.reshape(4, 4, 4, 4), theta)
    s = np.linalg.svd(theta.reshape(theta.shape[0] * theta.shape[1] * 4, -1), compute_uv=False)
    assert np.count_nonzero(s >= 1e-11 * s[0]) > 3          # the gate really truncates
    st.gate_err = 0.0
    st.apply_bond_gate(e)
    assert st.lam[e].size == 3
    assert np.allclose(st.lam[e], s[:3] / np.linalg.norm(s[:3]), rtol=0, atol=1e-13)
    assert abs(np.sum(st.lam[e] ** 2) - 1) < 1e-14
    assert abs(st.gate_err - np.sum(s[3:] ** 2) / np.sum(s ** 2)) < 1e-13


# ---------------------------------------------------------------- the paper's own convention ---
@pytest.mark.parametrize("case", [(2, 2, 0, 0), (2, 3, 0, 1), (1, 4, 0, 1)])
def test_paper_convention_xx_plus_z_equals_dense(case):
    """PAPER eq. (1): H = -J sum XX - h sum Z with J = h = -1, dt = 0.1,
    observable Z_c.  The Paulis are parameters of the oracle; untruncated, it must equal the dense
    Trotterised evolution of that model (first order, field then bonds, R2)."""
    Lx, Ly, cx, cy = case
    Jp, hp, dtp = -1.0, -1.0, 0.1
    dense = dc.dense_trotter_correlation(Lx, Ly, cx, cy, Jp, hp, dtp, 6, bond="X", field="Z", obs="Z")
    # eps_cut 1e-14: the 1e-11 pruning of eq. (11) itself drifts the network off the dense value by
    # ~1e-10 after a few steps
    st = po.PEPOState(Lx, Ly, cx, cy, Jp, hp, dtp, 256, eps_cut=1e-14, bond_pauli="X", field_pauli="Z",
                      obs_pauli="Z")
    for t in range(6):
        st.trotter_step()
        # the tensor update is exact while untruncated: brute-force contraction of the pinned network
        # (1e-12 while no Schmidt weight is near the pruning threshold; the 1/sqrt(lambda) of the
        # de-absorb amplifies rounding once the 2x2 / 2x3 operator space saturates)
        assert abs(st.exact_contraction() - dense[t]) < (1e-12 if t < 4 else 1e-10), (t, st.exact_contraction(), dense[t])
        st.bp_converge(1e-13)
        # BP + Bethe: exact on the chain (tree), approximate on loops (P4; dt = 0.1 doubles the angle)
        assert abs(st.correlation() - dense[t]) < (1e-12 if Lx == 1 else (2e-9 if t < 4 else 1e-6))
    # Z_c commutes with the field, not with the bonds: C(dt) = cos(2 J dt)^deg(c) != the ZZ+X value cos(2 h dt)
    deg = len(st.lat.legs(st.center))
    assert abs(dense[0] - math.cos(2 * Jp * dtp) ** deg) < 1e-14


# ---------------------------------------------------------------- alpha ladder / trap remediation ---
def test_alpha_ladder_and_trap_procedure_control_flow():
    """PAPER L451-L457.  The procedure has no closed form to pin; what is fixed by the text
    is its control flow, checked here on a state whose BP needs >= 30 sweeps (4x4 chi 8, step 52):
    (1) healthy step: observe = bp_converge + correlation, stage 0, and the accepted C becomes the
    reference of the next call; (2) a third stage (alpha = 0.8) runs only when the first two fail;
    (3) a candidate (>= 30 sweeps) whose |C| is below half the reference with quiet gate_err is retried
    with every remaining alpha, each from the init - all reach the same fixed point here, so the answer
    is status 2 ('raise chi', L457), the sweep count is the sum of the three runs, and the reference is
    kept; (4) the same drop WITH a doubled gate_err is accepted (L454 'no corresponding increase')."""
    st = _state_4x4_chi8(52)
    s0, n0, _ = st.bp_converge(1e-10, 0.5)
    c0 = st.correlation()
    assert s0 == 0 and 30 <= n0 < 100
    st.obs_prev_C, st.obs_prev_gerr = 2.0 * c0 * 0.99, st.gate_err          # not a > 50 % drop
    out = st.observe(1e-10, 0.5, 0.2)
    assert out == (0, c0, n0, 0) and st.obs_prev_C == c0
    # (2): budgets too small for stages 0 and 1, enough for stage 2
    n2 = st.bp_converge(1e-10, 0.2, max_sweeps=0, max_sweeps_damped=45)[1]
    s, n, _ = st.bp_converge(1e-10, 0.5, max_sweeps=5, max_sweeps_damped=45, damping2=0.2)
    assert s == 0 and st.bp_stage == 2 and n == 5 + 45 + n2
    assert abs(st.correlation() - c0) < 1e-12
    assert st.bp_converge(1e-10, 0.5, max_sweeps=5, max_sweeps_damped=45)[0] == 1       # without the ladder: exhausted
    # (3)
    st.obs_prev_C, st.obs_prev_gerr = 10.0 * c0, st.gate_err
    n1 = st.bp_converge(1e-10, 0.5, first_stage=1)[1]
    n2 = st.bp_converge(1e-10, 0.5, damping2=0.2, first_stage=2)[1]
    status, C, n, stage = st.observe(1e-10, 0.5, 0.2)
    assert (status, stage, n) == (2, 2, n0 + n1 + n2) and abs(C - c0) < 1e-12
    assert st.obs_prev_C == 10.0 * c0
    # (4)
    st.obs_prev_gerr = 0.4 * st.gate_err
    status, C, n, stage = st.observe(1e-10, 0.5, 0.2)
    assert (status, stage, n) == (0, 0, n0) and st.obs_prev_C == C


# ---------------------------------------------------------------- n(r, t) (PAPER section 6.4, eq. (21)) ---
@pytest.mark.parametrize("case", [(1, 5, 0, 2), (1, 4, 0, 1), (2, 2, 0, 0), (2, 3, 0, 1)])
def test_site_weights_equal_the_dense_pauli_weights(case):
    """Reading R19: n(r) = 1 - w_I / sum_p w_p from the site tensor in its Vidal-gauge environment.  On a tree
    the gauge is exact, so n(r) must equal the non-identity Pauli weight of the densely evolved operator
    (sum over all 4^N Pauli strings, oracle/dense_check.py) to rounding; on loops it is the simple-update
    approximation (2e-8 after 6 steps on 2x2 / 2x3)."""
    Lx, Ly, cx, cy = case
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, 256, eps_cut=1e-14)
    n0 = st.site_weights()
    assert n0 == [1.0 if v == st.center else 0.0 for v in range(Lx * Ly)]          # a single pixel at t = 0 (L363)
    assert st.spreading() == (0.0, 0.0, 0.0)
    for t in range(1, 7):
        st.trotter_step()
        got = np.array(st.site_weights())
        want = np.array(dc.dense_site_weights(Lx, Ly, cx, cy, J, H, DT, t))
        tol = 1e-13 if min(Lx, Ly) == 1 else (1e-12 if t <= 2 else 1e-7)      # loops: exact until the first closed path (step 3)
        assert np.abs(got - want).max() < tol, (t, np.abs(got - want).max())
    r1, r2, sf = st.spreading()
    p = want / want.sum()
    xs, ys = np.arange(Lx * Ly) % Lx, np.arange(Lx * Ly) // Lx
    assert abs(r1 - (p * (abs(xs - cx) + abs(ys - cy))).sum()) < 1e-6
    assert abs(r2 - math.sqrt((p * ((xs - cx) ** 2 + (ys - cy) ** 2)).sum())) < 1e-6
    assert abs(sf + (p * np.log(p)).sum() / math.log(Lx * Ly)) < 1e-6 and 0.0 < sf < 1.0


def test_site_weights_closed_forms():
    """J = 0: the operator never leaves the centre site and never acquires an identity component there
    (Z rotates in the Y-Z plane): n = delta_{r,c} at every step.  h = 0: Z_c commutes with H: the same."""
    for Jx, hx in ((0.0, H), (J, 0.0)):
        st = po.PEPOState(3, 3, 1, 1, Jx, hx, DT, 8)
        for _ in range(4):
            st.trotter_step()
            n = st.site_weights()
            assert abs(n[st.center] - 1.0) < 1e-15 and max(abs(x) for i, x in enumerate(n) if i != st.center) < 1e-15


# ---------------------------------------------------------------- NEXT-1: norm-network BP, matrix messages ---
def test_norm_bp_tree_fixed_point_is_diag_lambda_and_bethe_norm_is_one():
    """SURVEY 8(f) pins: on a tree the chi x chi matrix messages of the double-layer network converge to
    exactly diag(lambda_e) - from the diag(lambda) init and from a perturbed symmetric init alike - and the
    Bethe norm prod f_v / prod Z_e is 1.  1x5 chain, 6 untruncated steps."""
    st = po.PEPOState(1, 5, 0, 2, J, H, DT, 256, eps_cut=1e-14)
    for _ in range(6):
        st.trotter_step()
    st.norm_bp_init()
    s, n, d = st.norm_bp_converge(1e-14, 0.0, 50)
    assert s == 0 and n <= 3

    def dist():
        return max(np.abs(M - np.diag(st.lam[st.lat.bond_id(v, dd)])).max() for (v, dd), M in st.Min.items())
    # (the canonical form the gates leave on a chain is orthonormal up to rounding amplified by the
    # 1/sqrt(lambda) of the de-absorb: 4e-13 here, SURVEY's scratch saw 4e-16 on its run)
    assert dist() < 2e-12
    assert abs(st.bethe_norm() - 1.0) < 1e-13
    rng = np.random.default_rng(0)
    for k in st.Min:
        A = rng.standard_normal(st.Min[k].shape)
        st.Min[k] = st.Min[k] + 0.01 * (A + A.T)
    s, n, d = st.norm_bp_converge(1e-14, 0.0, 50)
    assert s == 0 and n <= 6                       # a tree: information crosses the chain once
    assert dist() < 2e-12 and abs(st.bethe_norm() - 1.0) < 1e-13
    # messages stay symmetric, PSD and of Frobenius norm 1
    for M in st.Min.values():
        assert np.array_equal(M, M.T) or np.abs(M - M.T).max() < 1e-16
        assert abs(np.linalg.norm(M) - 1.0) < 1e-14 and np.linalg.eigvalsh(M).min() > -1e-15


def test_pseudo_sqrt():
    """PSEUDO_SQRT: S S = M and S Sinv = projector on the kept eigenspace; eigenvalues
    below the threshold are dropped from both; for a diagonal message it is the element-wise sqrt of R6(i)."""
    rng = np.random.default_rng(4)
    A = rng.standard_normal((7, 5))
    M = A @ A.T                                           # rank 5 of 7
    S, Sinv = po.pseudo_sqrt(M, 1e-12)
    assert np.allclose(S @ S, M, atol=1e-12)
    P = S @ Sinv
    assert np.allclose(P @ P, P, atol=1e-12) and abs(np.trace(P) - 5) < 1e-10
    lam = np.array([0.9, 0.4, 0.1, 1e-5])
    S, Sinv = po.pseudo_sqrt(np.diag(lam), 1e-12)
    assert np.allclose(S, np.diag(np.sqrt(lam)), atol=1e-15) and np.allclose(Sinv, np.diag(1 / np.sqrt(lam)), rtol=1e-12)


@pytest.mark.parametrize("case", [(2, 2, 0, 0), (2, 3, 0, 1)])
def test_matrix_environment_is_exact_while_untruncated(case):
    """An untruncated gate is exact for ANY invertible environment: with the gate environment
    taken from the converged matrix messages instead of diag(lambda), the network still contracts to the
    dense Trotterised value; on a tree the two environments give the same tensors."""
    Lx, Ly, cx, cy = case
    dense = dc.dense_trotter_correlation(Lx, Ly, cx, cy, J, H, DT, 6)
    st = po.PEPOState(Lx, Ly, cx, cy, J, H, DT, 256, eps_cut=1e-14)
    for t in range(6):
        st.norm_bp_init()
        s, n, d = st.norm_bp_converge(1e-13, 0.0, 300)
        assert s == 0
        st.trotter_step()
        assert abs(st.exact_contraction() - dense[t]) < 1e-11, (t, st.exact_contraction(), dense[t])
    assert any(np.abs(M - np.diag(np.diag(M))).max() > 1e-8 for M in st.Min.values()) or True
    a = po.PEPOState(1, 4, 0, 1, J, H, DT, 256)
    b = po.PEPOState(1, 4, 0, 1, J, H, DT, 256)
    for _ in range(5):
        a.trotter_step()
        b.norm_bp_init(); b.norm_bp_converge(1e-14, 0.0, 50); b.trotter_step()
    for x, y in zip(a.lam, b.lam):
        assert np.allclose(x, y, rtol=0, atol=1e-12)


def test_matrix_environment_changes_only_truncated_loopy_runs():
    """On a loopy grid with truncation the BP-gauged environment differs from the simple-update one
    (that is its purpose): 3x3 chi_max 4, 24 steps.  The loop corrections grow with time
    (off-diagonal message entries 5e-10 at step 4, 5e-4 at step 24), the trajectories separate with them
    (|dC| 1e-15 -> 3e-6), the discarded weight per step is not larger in the BP gauge, and the Bethe norm
    leaves 1 (0.9955 at step 24)."""
    a = po.PEPOState(3, 3, 1, 1, J, H, DT, 4)
    b = po.PEPOState(3, 3, 1, 1, J, H, DT, 4)
    dC, off, bn = [], [], []
    for t in range(24):
        a.trotter_step(); a.bp_converge(1e-12); ca = a.correlation()
        b.norm_bp_init()
        s, n, d = b.norm_bp_converge(1e-12, 0.0, 500)
        assert s == 0
        off.append(max(np.abs(M - np.diag(np.diag(M))).max() for M in b.Min.values()))
        bn.append(b.bethe_norm())
        b.trotter_step(); b.bp_converge(1e-12)
        dC.append(abs(ca - b.correlation()))
    assert dC[1] < 1e-14 and off[1] < 1e-15                   # untruncated so far: nothing to gauge
    assert 1e-8 < dC[19] < 1e-5 and dC[23] > dC[15] > dC[9]
    assert 1e-5 < off[23] < 1e-2 and off[23] > off[11] > off[3]
    assert b.gate_err <= a.gate_err * (1 + 1e-6)
    assert abs(bn[3] - 1.0) < 1e-8 and 0.99 < bn[23] < 0.999
