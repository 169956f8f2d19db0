"""Exact dense 2^N Heisenberg evolution - the yardstick the ORACLE is pinned against.

TEST INFRASTRUCTURE ONLY (see ``oracle/pepo_oracle.py`` header).  Deliberately shares no
code with ``pepo_oracle.py`` (own Pauli matrices, own lattice enumeration, 2^N x 2^N complex
matrices instead of Pauli-transfer matrices), so that agreement between the two is a real
cross-check (SURVEY.md §8(c) pin P1).

Follows PAPER.md eq. (3)-(5) (L52-L80): Z_c(t+dt) = U^dag Z_c(t) U, C(t) = Tr[Z_c(t) Z_c]/2^N
(eq. (4)), with the Hamiltonian and Trotter splitting BASELINE.json fixes (DESIGN.md
readings R1, R2):  H = -J sum_<ij> B_i B_j - h sum_i F_i,  U_step = U_field * U_bond with
U_field = prod_i exp(+i h dt F_i), U_bond = prod_<ij> exp(+i J dt B_i B_j), so that
U_step^dag O U_step applies the field conjugation first and the bond conjugation second.
"""
from __future__ import annotations

import numpy as np

_I2 = np.eye(2, dtype=complex)
_SIG = {
    "I": _I2,
    "X": np.array([[0, 1], [1, 0]], dtype=complex),
    "Y": np.array([[0, -1j], [1j, 0]], dtype=complex),
    "Z": np.array([[1, 0], [0, -1]], dtype=complex),
}


def _embed(ops: dict, n: int) -> np.ndarray:
    """Kronecker product over sites 0..n-1 with ``ops[site]`` where given, identity elsewhere."""
    out = np.ones((1, 1), dtype=complex)
    for s in range(n):
        out = np.kron(out, ops.get(s, _I2))
    return out


def _bonds(Lx: int, Ly: int):
    b = []
    for y in range(Ly):
        for x in range(Lx):
            if x + 1 < Lx:
                b.append((y * Lx + x, y * Lx + x + 1))
            if y + 1 < Ly:
                b.append((y * Lx + x, (y + 1) * Lx + x))
    return b


def hamiltonian(Lx, Ly, J, h, bond="Z", field="X"):
    n = Lx * Ly
    H = np.zeros((2 ** n, 2 ** n), dtype=complex)
    for (i, j) in _bonds(Lx, Ly):
        H -= J * _embed({i: _SIG[bond], j: _SIG[bond]}, n)
    for i in range(n):
        H -= h * _embed({i: _SIG[field]}, n)
    return H


def _expm_herm(A: np.ndarray, coeff: complex) -> np.ndarray:
    """exp(coeff * A) for Hermitian A through its eigendecomposition."""
    w, V = np.linalg.eigh(A)
    return (V * np.exp(coeff * w)) @ V.conj().T


def trotter_unitary(Lx, Ly, J, h, dt, bond="Z", field="X", order=1):
    n = Lx * Ly
    Hf = np.zeros((2 ** n, 2 ** n), dtype=complex)
    for i in range(n):
        Hf += h * _embed({i: _SIG[field]}, n)
    Hb = np.zeros((2 ** n, 2 ** n), dtype=complex)
    for (i, j) in _bonds(Lx, Ly):
        Hb += J * _embed({i: _SIG[bond], j: _SIG[bond]}, n)
    if order == 2:
        # symmetric splitting (PAPER eq. (6)): e^{i dt Hf/2} e^{i dt Hb} e^{i dt Hf/2}
        Uh = _expm_herm(Hf, 0.5j * dt)
        return Uh @ _expm_herm(Hb, 1j * dt) @ Uh
    return _expm_herm(Hf, 1j * dt) @ _expm_herm(Hb, 1j * dt)


def dense_trotter_correlation(Lx, Ly, cx, cy, J, h, dt, n_steps, bond="Z", field="X", obs="Z", order=1):
    """C after each of ``n_steps`` Trotter steps (order 1: R2; order 2: eq. (6)), by 2^N x 2^N conjugation."""
    n = Lx * Ly
    c = cy * Lx + cx
    Zc = _embed({c: _SIG[obs]}, n)
    U = trotter_unitary(Lx, Ly, J, h, dt, bond, field, order)
    O = Zc.copy()
    out = []
    for _ in range(n_steps):
        O = U.conj().T @ O @ U
        out.append(float(np.trace(O @ Zc).real) / 2 ** n)
    return out


def dense_exact_correlation(Lx, Ly, cx, cy, J, h, t, bond="Z", field="X", obs="Z"):
    """Tr[e^{iHt} Z_c e^{-iHt} Z_c]/2^N with the exact propagator (Trotter-error context)."""
    n = Lx * Ly
    c = cy * Lx + cx
    Zc = _embed({c: _SIG[obs]}, n)
    U = _expm_herm(hamiltonian(Lx, Ly, J, h, bond, field), -1j * t)
    O = U.conj().T @ Zc @ U
    return float(np.trace(O @ Zc).real) / 2 ** n


def dense_chain_operator_schmidt(n, c, J, h, dt, n_steps, cut, bond="Z", field="X", obs="Z"):
    """Operator-Schmidt coefficients (normalised to unit 2-norm, descending) of the Trotter-evolved
    operator O(n_steps) = (U^dag)^n P_c U^n on an open chain of ``n`` sites, across the cut between
    sites ``cut`` and ``cut + 1``: singular values of O reshaped to (left in x left out) x (right in x
    right out).  On a tree the simple-update bond weights lambda_e of the untruncated network are
    exactly these numbers (Vidal gauge), so this pins lambda and the entanglement-entropy diagnostic
    (PAPER Table 1) to the dense evolution."""
    U = trotter_unitary(1, n, J, h, dt, bond, field)
    O = _embed({c: _SIG[obs]}, n)
    for _ in range(n_steps):
        O = U.conj().T @ O @ U
    nl = cut + 1
    dl, dr = 2 ** nl, 2 ** (n - nl)
    T = O.reshape(dl, dr, dl, dr).transpose(0, 2, 1, 3).reshape(dl * dl, dr * dr)
    s = np.linalg.svd(T, compute_uv=False)
    return s / np.linalg.norm(s)


def dense_site_weights(Lx, Ly, cx, cy, J, h, dt, n_steps, bond="Z", field="X", obs="Z"):
    """Per-site non-identity Pauli weight n(r) of the Trotter-evolved operator O = (U^dag)^n P_c U^n
    (section 6.4): with O = sum_S c_S S over Pauli strings S,
    n(r) = sum_{S: S_r != I} c_S^2 / sum_S c_S^2.  Computed from the full coefficient vector
    c_S = Tr[S O] / 2^N (site 0 is the slowest Kronecker factor, as in _embed)."""
    n = Lx * Ly
    U = trotter_unitary(Lx, Ly, J, h, dt, bond, field)
    O = _embed({cy * Lx + cx: _SIG[obs]}, n)
    for _ in range(n_steps):
        O = U.conj().T @ O @ U
    # tensor with one (row, column) index pair per site, then each pair -> Pauli index p via Tr[P_p . ]/2
    T = O.reshape([2] * (2 * n))
    T = T.transpose([k for s in range(n) for k in (s, n + s)]).reshape([4] * n)       # index (r, c) = 2 r + c per site
    P = np.stack([np.array([_SIG[k][0, 0], _SIG[k][1, 0], _SIG[k][0, 1], _SIG[k][1, 1]]) for k in "IXYZ"]) / 2.0
    # c_p = Tr[P_p M]/2 = sum_{r,c} P_p[c, r] M[r, c] / 2  ->  row of P holds P_p[c, r] at position 2 r + c
    for s in range(n):
        T = np.moveaxis(np.tensordot(P, T, axes=([1], [s])), 0, s)
    w = np.abs(T) ** 2
    tot = w.sum()
    out = []
    for s in range(n):
        ident = np.take(w, 0, axis=s).sum()
        out.append(float(1.0 - ident / tot))
    return out
