"""CPU fp64 ORACLE for the Heisenberg-picture PEPO hot path of arxiv/paper_2606_30985.

THIS FILE IS TEST INFRASTRUCTURE.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  It shares no
code with the CUDA path (``paper_2606_30985_b200/``) and neither imports the other.

It is a plain, slow, step-by-step restatement of the paper's algorithm in numpy fp64
(library primitives used as steps: ``numpy.linalg.qr`` = LAPACK Householder GEQRF+ORGQR,
``numpy.linalg.svd``, ``@``/einsum).  No blocking, fusion or reordering beyond what
the paper states.  Every function cites the PAPER.md passage it follows
(``/root/reference/PAPER.md`` line numbers, section / equation) and, where the paper is
silent or garbled, the DESIGN.md reading (R1..R18, which restate SURVEY.md §8(c) C1..C18).

Conventions:
  * Lattice Lx x Ly, open boundaries, site (x, y), 0<=x<Lx, 0<=y<Ly.
    Neighbours: U=(x,y-1), D=(x,y+1), L=(x-1,y), R=(x+1,y).
  * Site tensor psi_v has the legs [U, D, L, R, P] that exist, P (Pauli,
    dim 4: I,X,Y,Z) last.  The *packed layout* is column-major: first leg
    fastest, P slowest ("column-major flat").  Here a site tensor is a numpy
    array whose axes are in that leg order; ``pack`` flattens with order='F'.
  * Bond ids: horizontal bonds (x,y)-(x+1,y) first, id = y*(Lx-1)+x; then vertical bonds
    (x,y)-(x,y+1), id = Ly*(Lx-1) + y*Lx + x.
  * Hamiltonian actually run (BASELINE.json, R1): H = -J sum ZZ - h sum X, observable Z_c,
    first-order Trotter (R2): per step, field gate on all sites, then the ZZ gates in four
    colour classes (R3).  Bond / field / observable Paulis are parameters so the paper's own
    convention (eq. (1): XX + Z) can also be run.

Pins (tests/test_oracle_*.py, -m "not gpu"): dense 2^N Trotterised evolution
(``oracle/dense_check.py``, shares nothing with this file), exact brute-force network
contraction, closed forms at J=0 / h=0, tree-exactness of BP on 1xN chains, Listing 1 vs
nested loops vs numpy.transpose, QR/SVD invariants, the paper's Table 9/10 memory numbers.
Parity unpinned: the paper's printed C(t) tables (Tables 4, 7) - could not be reproduced by
dense evolution under any convention tried, so they pin nothing.
"""
from __future__ import annotations

import itertools
import math

import numpy as np

# --------------------------------------------------------------------------------------
# Pauli matrices and Pauli-transfer matrices (PTM)
# --------------------------------------------------------------------------------------
_PAULI = [
    np.array([[1, 0], [0, 1]], dtype=complex),     # p=0: I
    np.array([[0, 1], [1, 0]], dtype=complex),     # p=1: X
    np.array([[0, -1j], [1j, 0]], dtype=complex),  # p=2: Y
    np.array([[1, 0], [0, -1]], dtype=complex),    # p=3: Z
]
PAULI_INDEX = {"I": 0, "X": 1, "Y": 2, "Z": 3}


def _expm_i_theta_pauli(theta: float, P: np.ndarray) -> np.ndarray:
    """exp(+i*theta*P) for an involutory P (P@P = 1): cos(theta) 1 + i sin(theta) P."""
    return math.cos(theta) * np.eye(P.shape[0], dtype=complex) + 1j * math.sin(theta) * P


def ptm_one_site(theta: float, pauli: str = "X") -> np.ndarray:
    """4x4 real PTM of the field gate, G[a,b] = Tr[P_a U^dag P_b U]/2, U = exp(+i*theta*P).

    PAPER L81 (eq. (5): conjugation by U maps Paulis to real combinations of Paulis, the
    gate in the Pauli basis is real orthogonal), R2/R15.  New coefficients c' = G c.
    """
    U = _expm_i_theta_pauli(theta, _PAULI[PAULI_INDEX[pauli]])
    G = np.zeros((4, 4))
    for a in range(4):
        for b in range(4):
            G[a, b] = np.trace(_PAULI[a] @ U.conj().T @ _PAULI[b] @ U).real / 2.0
    return G


def ptm_two_site(theta: float, pauli: str = "Z") -> np.ndarray:
    """16x16 real PTM of exp(+i*theta*P(x)P); row index p1'*4+p2', column p1*4+p2 (R15).

    G[(a1 a2),(b1 b2)] = Tr[(P_a1 x P_a2) U^dag (P_b1 x P_b2) U]/4; site 1 = v1 is the
    left Kronecker factor.  PAPER L97-L99 (gate G in R^{D^2 x D^2}).
    """
    P = _PAULI[PAULI_INDEX[pauli]]
    U = _expm_i_theta_pauli(theta, np.kron(P, P))
    G = np.zeros((16, 16))
    for a1 in range(4):
        for a2 in range(4):
            Pa = np.kron(_PAULI[a1], _PAULI[a2])
            for b1 in range(4):
                for b2 in range(4):
                    Pb = np.kron(_PAULI[b1], _PAULI[b2])
                    G[a1 * 4 + a2, b1 * 4 + b2] = np.trace(Pa @ U.conj().T @ Pb @ U).real / 4.0
    return G


# --------------------------------------------------------------------------------------
# Lattice bookkeeping
# --------------------------------------------------------------------------------------
_DIRS = ("U", "D", "L", "R")
_DXY = {"U": (0, -1), "D": (0, 1), "L": (-1, 0), "R": (1, 0)}


class Lattice:
    """Open-boundary Lx x Ly grid, legs [U,D,L,R,P] (L168), 4 colours (L87, R3)."""

    def __init__(self, Lx: int, Ly: int):
        if Lx < 1 or Ly < 1:
            raise ValueError("grid must be at least 1x1")
        self.Lx, self.Ly = Lx, Ly
        self.n_sites = Lx * Ly
        self.n_hbonds = Ly * (Lx - 1)
        self.n_bonds = self.n_hbonds + (Ly - 1) * Lx   # = 2N(N-1) on NxN

    def site(self, x: int, y: int) -> int:
        return y * self.Lx + x

    def xy(self, v: int):
        return v % self.Lx, v // self.Lx

    def neighbour(self, v: int, d: str):
        x, y = self.xy(v)
        dx, dy = _DXY[d]
        x2, y2 = x + dx, y + dy
        if 0 <= x2 < self.Lx and 0 <= y2 < self.Ly:
            return self.site(x2, y2)
        return None

    def legs(self, v: int):
        """Directions present at site v, in canonical order [U, D, L, R]."""
        return [d for d in _DIRS if self.neighbour(v, d) is not None]

    def bond_id(self, v: int, d: str) -> int:
        x, y = self.xy(v)
        if d == "R":
            return y * (self.Lx - 1) + x
        if d == "L":
            return y * (self.Lx - 1) + (x - 1)
        if d == "D":
            return self.n_hbonds + y * self.Lx + x
        if d == "U":
            return self.n_hbonds + (y - 1) * self.Lx + x
        raise ValueError(d)

    def bond_sites(self, e: int):
        """(v1, d1, v2, d2): v1 is the smaller-coordinate site, d_i the leg of v_i on the bond."""
        if e < self.n_hbonds:
            y, x = divmod(e, self.Lx - 1)
            return self.site(x, y), "R", self.site(x + 1, y), "L"
        y, x = divmod(e - self.n_hbonds, self.Lx)
        return self.site(x, y), "D", self.site(x, y + 1), "U"

    def colour_classes(self):
        """R3: 0 = horizontal x even, 1 = horizontal x odd, 2 = vertical y even, 3 = vertical
        y odd; inside a class y outer, x inner ascending.  No two bonds of a class share a
        site."""
        classes = [[], [], [], []]
        for y in range(self.Ly):
            for x in range(self.Lx - 1):
                classes[x % 2].append(y * (self.Lx - 1) + x)
        for y in range(self.Ly - 1):
            for x in range(self.Lx):
                classes[2 + (y % 2)].append(self.n_hbonds + y * self.Lx + x)
        return classes


# --------------------------------------------------------------------------------------
# a4 / a11: tensor permutation (PAPER §4.1, Listing 1)
# --------------------------------------------------------------------------------------
def permute_listing1(src_flat: np.ndarray, shape_in, perm) -> np.ndarray:
    """Listing 1, vectorised over ``idx`` but otherwise literal.

    ``src_flat`` is the column-major flat input of shape ``shape_in`` (first dim fastest).
    ``perm`` follows numpy.transpose on that column-major shape (R10): output dim j is
    input dim perm[j].  ``stride_out[d]`` = destination (column-major) stride of SOURCE dim
    d.  Each element idx: peel coords of idx along the source dims, dot with stride_out,
    scatter dst[out_idx] = src[idx].
    """
    shape_in = [int(s) for s in shape_in]
    ndim = len(shape_in)
    shape_out = [shape_in[perm[j]] for j in range(ndim)]
    out_strides = [1] * ndim
    for j in range(1, ndim):
        out_strides[j] = out_strides[j - 1] * shape_out[j - 1]
    stride_out = [0] * ndim
    for j in range(ndim):
        stride_out[perm[j]] = out_strides[j]
    total = int(np.prod(shape_in, dtype=np.int64)) if ndim else 1
    idx = np.arange(total, dtype=np.int64)
    in_idx = idx.copy()
    out_idx = np.zeros(total, dtype=np.int64)
    for d in range(ndim):                       # Listing 1 lines 9-13
        coord = in_idx % shape_in[d]
        in_idx //= shape_in[d]
        out_idx += coord * stride_out[d]
    dst = np.empty_like(src_flat)
    dst[out_idx] = src_flat[idx]                # Listing 1 line 14 (scatter)
    return dst


def permute_nested_loops(src_flat, shape_in, perm):
    """Pure-Python nested-loop definition of the same permutation (tiny inputs only)."""
    ndim = len(shape_in)
    shape_out = [shape_in[perm[j]] for j in range(ndim)]
    dst = [0.0] * len(src_flat)
    for out_multi in itertools.product(*[range(s) for s in reversed(shape_out)]):
        o = list(reversed(out_multi))           # o[j] = coordinate along output dim j
        i = [0] * ndim
        for j in range(ndim):
            i[perm[j]] = o[j]
        oi = 0
        for j in reversed(range(ndim)):
            oi = oi * shape_out[j] + o[j]
        ii = 0
        for d in reversed(range(ndim)):
            ii = ii * shape_in[d] + i[d]
        dst[oi] = src_flat[ii]
    return np.asarray(dst, dtype=np.asarray(src_flat).dtype)


# --------------------------------------------------------------------------------------
# a5 / a6: QR of the tall-skinny cv matrix (PAPER §4.2)
# --------------------------------------------------------------------------------------
def householder_qr(A: np.ndarray):
    """Reduced Householder QR (LAPACK GEQRF + ORGQR): A (m x n) = Q R with
    Q m x k, R k x n, k = min(m, n) (R13)."""
    Q, R = np.linalg.qr(A, mode="reduced")
    return Q, R


def cholesky_qr(A: np.ndarray, eps: float = 0.0):
    """Cholesky-QR exactly as eq. (10): C = A^T A + eps I, R = chol(C)
    (upper), Q = A R^{-1}.  eps = 0 in fp64 (L231, R9).  Raises numpy LinAlgError when C is
    not positive definite (the paper's potrf_info != 0)."""
    n = A.shape[1]
    C = A.T @ A + eps * np.eye(n)
    L = np.linalg.cholesky(C)            # C = L L^T, R = L^T upper
    R = L.T.copy()
    # Q R = A  <=>  R^T Q^T = A^T  (forward substitution, the paper's TRSM)
    Q = np.linalg.solve(R.T, A.T).T
    return Q, R


def pseudo_sqrt(M: np.ndarray, eps: float):
    """PSEUDO_SQRT of PAPER L315-L317: symmetric eigendecomposition M = V diag(w) V^T; eigenvalues below
    eps * max(w) are zeroed; returns (V sqrt(w) V^T, V w^-1/2 V^T) with the zeroed ones left out of both."""
    w, V = np.linalg.eigh(0.5 * (M + M.T))
    keep = w > eps * max(float(w.max()), 0.0)
    r = np.sqrt(np.where(keep, w, 1.0))
    S = (V * np.where(keep, r, 0.0)) @ V.T
    Sinv = (V * np.where(keep, 1.0 / r, 0.0)) @ V.T
    return S, Sinv


def truncation_rank(s: np.ndarray, chi_max: int, eps_cut: float) -> int:
    """eq. (11): chi_new = min(#{i : s_i >= eps_cut*s_0}, chi_max), s sorted
    descending, count includes i=0 (R8)."""
    if s.size == 0 or s[0] <= 0.0:
        return 0
    return int(min(np.count_nonzero(s >= eps_cut * s[0]), chi_max))


# --------------------------------------------------------------------------------------
# The state and the Trotter step
# --------------------------------------------------------------------------------------
class PEPOState:
    """psi[v] (legs present among [U,D,L,R], then P) and lambda_e per bond.

    Init: all bonds chi=1, lambda=[1]; psi_c[0..0,p] = delta(p, obs),
    psi_v[0..0,p] = delta(p, I) elsewhere.
    """

    def __init__(self, Lx, Ly, cx, cy, J, h, dt, chi_max, eps_cut=1e-11,
                 bond_pauli="Z", field_pauli="X", obs_pauli="Z", order=1):
        self.lat = Lattice(Lx, Ly)
        if not (0 <= cx < Lx and 0 <= cy < Ly):
            raise ValueError("centre outside grid")
        if chi_max < 1 or dt <= 0:
            raise ValueError("bad chi_max / dt")
        self.center = self.lat.site(cx, cy)
        self.J, self.h, self.dt = float(J), float(h), float(dt)
        self.chi_max, self.eps_cut = int(chi_max), float(eps_cut)
        self.obs = PAULI_INDEX[obs_pauli]
        # R2/R15: U = exp(-iH dt) = exp(+i dt (J sum PP + h sum F)) for H = -J sum PP - h sum F
        self.G1 = ptm_one_site(self.h * self.dt, field_pauli)
        self.G2 = ptm_two_site(self.J * self.dt, bond_pauli)
        # order 2 = the symmetric step of PAPER eq. (6): half field gate,
        # all bond gates, half field gate.  order 1 (R2, BASELINE) leaves everything above as it was.
        if order not in (1, 2):
            raise ValueError("order must be 1 or 2")
        self.order = int(order)
        self.G1_half = ptm_one_site(0.5 * self.h * self.dt, field_pauli)
        self.psi = []
        for v in range(self.lat.n_sites):
            t = np.zeros([1] * len(self.lat.legs(v)) + [4])
            t[..., self.obs if v == self.center else 0] = 1.0
            self.psi.append(t)
        self.lam = [np.ones(1) for _ in range(self.lat.n_bonds)]
        # NEXT-1: chi x chi matrix messages of the norm network;
        # None = the diagonal gauge weights mu_e = diag(lambda_e) of reading R6(i).  Min[(v, d)] is the
        # message ARRIVING at site v through its leg d.
        self.Min = None
        self.psqrt_eps = 1e-12           # PSEUDO_SQRT: eigenvalues below eps * largest are zeroed (L315-L317)
        # diagnostics (Table 1): discarded weight of the last step
        self.gate_err = 0.0
        self.qr_log = []     # (m, n, rank-estimate) of every QR, for workload statistics

    # -- helpers ---------------------------------------------------------------------
    def bond_dims(self):
        return [int(l.size) for l in self.lam]

    def pack(self, v):
        """Packed column-major flat copy of psi_v (boundary layout, R11)."""
        return self.psi[v].flatten(order="F")

    def set_packed(self, v, flat):
        self.psi[v] = np.asarray(flat, dtype=np.float64).reshape(self.psi[v].shape, order="F").copy()

    # -- a1: field gate ----------------------------------------------------------------
    def apply_field_gate(self, half=False):
        """a1 (R2): psi_v[...,p'] = sum_p G1[p',p] psi_v[...,p], all sites
        (half = True: the half-angle gate of the symmetric step, eq. (6))."""
        G = self.G1_half if half else self.G1
        for v in range(self.lat.n_sites):
            self.psi[v] = np.tensordot(self.psi[v], G, axes=([-1], [1]))

    # -- a2..a13: Algorithm 1 ------------------------------------------------------------
    def _cv_matrix(self, v, d_cut):
        """Steps 1-3 of Alg. 1 for one site.

        a2: sqrt(mu) of every env bond = sqrt(lambda) element-wise (messages are diagonal in
        the Vidal gauge; R6(i)).  a3: absorb on every non-cut leg.  a4: permute the
        cut leg to the last bond position, reshape (column-major) to m x n, rows = env legs,
        columns = (cut, P) with cut fastest.
        Returns (cv matrix, env_dirs, env_shape, env weights list).
        """
        lat = self.lat
        legs = lat.legs(v)
        t = self.psi[v].copy()
        sq = {}
        for ax, d in enumerate(legs):
            if d == d_cut:
                continue
            if self.Min is not None:
                # NEXT-1: general symmetric PSEUDO_SQRT of the incoming matrix message (L315-L317), absorbed
                # by a chi x chi GEMM on that leg (L318); its pseudo-inverse de-absorbs (L336)
                S, Sinv = pseudo_sqrt(self.Min[(v, d)], self.psqrt_eps)
                sq[d] = ("matrix", Sinv)
                t = np.moveaxis(np.tensordot(t, S, axes=([ax], [0])), -1, ax)
                continue
            w = np.sqrt(self.lam[lat.bond_id(v, d)])            # a2
            sq[d] = w
            shp = [1] * t.ndim
            shp[ax] = w.size
            t = t * w.reshape(shp)                              # a3
        cut_ax = legs.index(d_cut)
        env_axes = [ax for ax in range(len(legs)) if ax != cut_ax]
        perm = env_axes + [cut_ax, len(legs)]
        # a4 through Listing 1 itself (scatter on the column-major flat array)
        flat = permute_listing1(t.flatten(order="F"), t.shape, perm)
        env_shape = [t.shape[ax] for ax in env_axes]
        m = int(np.prod(env_shape, dtype=np.int64)) if env_shape else 1
        n = t.shape[cut_ax] * 4
        cv = flat.reshape((m, n), order="F")
        return cv, [legs[ax] for ax in env_axes], env_shape, sq, perm

    def apply_bond_gate(self, e):
        """Algorithm 1 on bond e, with readings R4 (core shape), R5
        (unnormalised sqrt(s) into psi), R8 (truncation), Householder QR always (R9)."""
        lat = self.lat
        v1, d1, v2, d2 = lat.bond_sites(e)
        chi_c = self.lam[e].size
        Q, R, meta = [], [], []
        for v, d in ((v1, d1), (v2, d2)):
            cv, env_dirs, env_shape, sq, perm = self._cv_matrix(v, d)
            q, r = householder_qr(cv)                                    # a6 (step 4)
            self.qr_log.append((cv.shape[0], cv.shape[1], int(np.linalg.matrix_rank(r)) if r.size < 1 << 16 else -1))
            Q.append(q); R.append(r); meta.append((v, env_dirs, env_shape, sq, perm))
        k1, k2 = R[0].shape[0], R[1].shape[0]
        # a7 (step 5): split the column index of R_i into (c, p) (c fastest),
        # RR4[k1,p1,k2,p2] = sum_c R1[k1;c,p1] R2[k2;c,p2]  (contraction over the cut only, R4)
        A1 = R[0].reshape((k1, chi_c, 4), order="F")
        A2 = R[1].reshape((k2, chi_c, 4), order="F")
        RR4 = np.einsum("kcp,lcq->kplq", A1, A2)
        # a8 (step 6): gate on the D x D physical block
        G4 = self.G2.reshape(4, 4, 4, 4)          # [p1', p2', p1, p2]
        oR4 = np.einsum("abpq,kplq->kalb", G4, RR4)
        # a9 (step 7): SVD on rows (k1,p1'), cols (k2,p2'); eq. (11), (12)
        Mtx = oR4.reshape((k1 * 4, k2 * 4), order="F")
        U, s, Vt = np.linalg.svd(Mtx, full_matrices=False)
        chi_new = truncation_rank(s, self.chi_max, self.eps_cut)
        if chi_new == 0:
            raise FloatingPointError("s0 = 0 in gate update")
        self.gate_err += float(np.sum(s[chi_new:] ** 2) / np.sum(s ** 2))
        s_keep = s[:chi_new]
        lam_new = s_keep / np.linalg.norm(s_keep)                            # eq. (12), R8
        # a10 (step 8/9; R5): M1 = U sqrt(S), M2 = (sqrt(S) V^T)^T
        rs = np.sqrt(s_keep)
        M1 = (U[:, :chi_new] * rs).reshape((k1, 4, chi_new), order="F")      # [k1,p1',c']
        M2 = (Vt[:chi_new, :].T * rs).reshape((k2, 4, chi_new), order="F")   # [k2,p2',c']
        for (q, Mi, (v, env_dirs, env_shape, sq, perm)) in ((Q[0], M1, meta[0]), (Q[1], M2, meta[1])):
            k = q.shape[1]
            # columns of the new cv are (c', p') with c' fastest
            Mmat = np.transpose(Mi, (0, 2, 1)).reshape((k, chi_new * 4), order="F")
            cv_new = q @ Mmat                                               # a10
            shape_perm = list(env_shape) + [chi_new, 4]
            inv = [0] * len(perm)
            for j, pj in enumerate(perm):
                inv[pj] = j
            flat = permute_listing1(cv_new.flatten(order="F"), shape_perm, inv)   # a11
            shape_can = [shape_perm[inv[j]] for j in range(len(inv))]
            t = flat.reshape(shape_can, order="F")
            legs = lat.legs(v)
            for ax, d in enumerate(legs):                                   # a12 deabsorb
                if d in sq:
                    if isinstance(sq[d], tuple):
                        t = np.moveaxis(np.tensordot(t, sq[d][1], axes=([ax], [0])), -1, ax)
                        continue
                    shp = [1] * t.ndim
                    shp[ax] = sq[d].size
                    t = t / sq[d].reshape(shp)
            self.psi[v] = t                                                 # a13 write-back
        self.lam[e] = lam_new                                               # a13: mu <- diag(lambda)
        if self.Min is not None:                                            # both directions, new index basis
            self.Min[(v1, d1)] = np.diag(lam_new)
            self.Min[(v2, d2)] = np.diag(lam_new)

    def trotter_step(self):
        """One first-order step (R2): a1 on all sites, then colours 0..3 (R3), each bond in
        the class order.  PAPER Fig. 1 L310-L342."""
        self.gate_err = 0.0
        if self.order == 2:
            # eq. (6): R(h dt/2) on all sites, the bond sweep, R(h dt/2) on all sites
            self.apply_field_gate(half=True)
            for cls in self.lat.colour_classes():
                for e in cls:
                    self.apply_bond_gate(e)
            self.apply_field_gate(half=True)
            return
        self.apply_field_gate()
        for cls in self.lat.colour_classes():
            for e in cls:
                self.apply_bond_gate(e)

    # -- diagnostics (Table 1) ---------------------------
    def bond_entropy(self, e):
        """S_e = -sum_k lambda_k^2 log lambda_k^2 of the normalised Schmidt weights of bond e
        (eq. (12): sum_k lambda_k^2 = 1)."""
        w = self.lam[e] ** 2
        w = w[w > 0.0]
        return float(-(w * np.log(w)).sum())

    def site_pauli_weights(self, v):
        """w_p = sum_i psi_v[i, p]^2 prod_legs lambda_leg[i_leg], p = I, X, Y, Z: the Pauli-resolved norm of
        site v in its simple-update environment (psi carries sqrt(s) on every leg, R5; the environment of
        the Vidal gauge adds sqrt(lambda) per leg on each of the two layers) - exact on trees."""
        t = self.psi[v] ** 2
        for ax, d in enumerate(self.lat.legs(v)):
            shp = [1] * t.ndim
            shp[ax] = -1
            t = t * self.lam[self.lat.bond_id(v, d)].reshape(shp)
        return t.reshape(-1, 4).sum(axis=0)

    def site_weights(self):
        """n(r, t): per-site non-identity Pauli weight (PAPER section 6.4, Figs. 4-6):
        n(r) = 1 - w_I(r) / sum_p w_p(r).  The paper gives no formula: DESIGN.md reading R19."""
        out = []
        for v in range(self.lat.n_sites):
            w = self.site_pauli_weights(v)
            out.append(float(1.0 - w[0] / w.sum()))
        return out

    def spreading(self):
        """(R_L1, R_L2, S_frac) of PAPER appendix A.3, eq. (21): mean Manhattan radius, RMS
        Euclidean radius from the centre site and the spatial entropy fraction of p(r) = n(r)/sum n(r)."""
        n = np.asarray(self.site_weights())
        p = n / n.sum()
        cx, cy = self.lat.xy(self.center)
        xs = np.array([self.lat.xy(v)[0] for v in range(self.lat.n_sites)])
        ys = np.array([self.lat.xy(v)[1] for v in range(self.lat.n_sites)])
        r1 = float((p * (np.abs(xs - cx) + np.abs(ys - cy))).sum())
        r2 = float(math.sqrt((p * ((xs - cx) ** 2 + (ys - cy) ** 2)).sum()))
        q = p[p > 0.0]
        sfrac = float(-(q * np.log(q)).sum() / math.log(self.lat.n_sites)) if self.lat.n_sites > 1 else 0.0
        return r1, r2, sfrac

    # -- a14: BP on the pinned single-layer network -----------------------------------
    def pinned(self, v):
        """T_v = psi_v[..., p_v], p_c = observable Pauli, else I (step 1)."""
        return self.psi[v][..., self.obs if v == self.center else 0]

    def _init_messages(self):
        """R7: deterministic init m = (1, .., 1)/sqrt(chi) on every directed bond.  ``self.bp_init = "e0"``
        (reading R7b, an option on both sides) starts from the leading Schmidt vector e_0 of each bond
        instead - where the operator is close to the identity that IS the message up to small terms."""
        msgs = {}
        e0 = getattr(self, "bp_init", "uniform") == "e0"
        for v in range(self.lat.n_sites):
            for d in self.lat.legs(v):
                chi = self.lam[self.lat.bond_id(v, d)].size
                # message v -> neighbour across leg d
                if e0:
                    m = np.zeros(chi)
                    m[0] = 1.0
                else:
                    m = np.full(chi, 1.0 / math.sqrt(chi))
                msgs[(v, d)] = m
        return msgs

    def _incoming(self, msgs, v, d):
        """Message arriving at v through its leg d (sent by the neighbour over that bond)."""
        u = self.lat.neighbour(v, d)
        back = {"U": "D", "D": "U", "L": "R", "R": "L"}[d]
        return msgs[(u, back)]

    def _bp_sweep(self, msgs, damping):
        """One Jacobi sweep of eq. (13) PAPER L243-L247 with the details of R7: L2-normalise,
        sign-align with the old message, damp (eq. (19), d = 1 - alpha), delta = eq. (14)."""
        new = {}
        delta = 0.0
        flagged = False
        for v in range(self.lat.n_sites):
            legs = self.lat.legs(v)
            T = self.pinned(v)
            for ax_out, d_out in enumerate(legs):
                t = T
                # contract every other leg with its incoming message, highest axis first
                for ax in reversed(range(len(legs))):
                    if ax == ax_out:
                        continue
                    t = np.tensordot(t, self._incoming(msgs, v, legs[ax]), axes=([ax], [0]))
                mhat = t
                old = msgs[(v, d_out)]
                nrm = math.sqrt(float(np.dot(mhat, mhat)))
                if nrm == 0.0 or not math.isfinite(nrm):
                    new[(v, d_out)] = old.copy()
                    flagged = True
                    continue
                mhat = mhat / nrm
                if float(np.dot(mhat, old)) < 0.0:
                    mhat = -mhat
                mnew = damping * old + (1.0 - damping) * mhat
                delta = max(delta, float(np.max(np.abs(mnew - old))))
                new[(v, d_out)] = mnew
        return new, delta, flagged

    def _bp_stage(self, tol, damping, budget):
        """One stage: restart from the init (R7) and sweep with `damping` until delta < tol or budget."""
        msgs = self._init_messages()
        n, delta = 0, float("inf")
        for _ in range(budget):
            msgs, delta, _ = self._bp_sweep(msgs, damping)
            n += 1
            if delta < tol:
                return 0, n, delta, msgs
        return 1, n, delta, msgs

    def bp_converge(self, tol, damping=0.0, max_sweeps=100, max_sweeps_damped=1000, damping2=None,
                    first_stage=0):
        """a14 until delta < tol or budget (R7).  Stage 0 undamped up to
        ``max_sweeps``; if not converged and damping > 0: restart from the init with that
        damping up to ``max_sweeps_damped`` (the paper's alpha-retry, L456); ``damping2`` adds a
        third stage with another alpha (the ladder of L451-L457: alpha = 0.5, then 0.8).
        Returns (status, sweeps, delta): status 0 converged, 1 budget exhausted.  The stage that
        ended the call is left in ``self.bp_stage``."""
        stages = [(0.0, max_sweeps), (damping, max_sweeps_damped)]
        if damping2 is not None:
            stages.append((damping2, max_sweeps_damped))
        sweeps, delta, status = 0, float("inf"), 1
        msgs = self._init_messages()
        for k, (d, budget) in enumerate(stages):
            if k < first_stage or (k >= 1 and not d > 0.0) or (k == 2 and d == damping):
                continue
            status, n, delta, msgs = self._bp_stage(tol, d, budget)
            sweeps += n
            self.bp_stage = k
            if status == 0:
                break
        self.msgs = msgs
        return status, sweeps, delta

    def observe(self, tol, damping, damping2=None, max_sweeps=100, max_sweeps_damped=1000):
        """BP + Bethe with the trap remediation procedure of PAPER L451-L457: a converged run with
        >= 30 sweeps is a trap candidate; it counts as a trap when |C| fell below half of the last
        accepted C(t) while gate_err did not double; then the next alpha is tried from the init.
        Returns (status, C, sweeps, stage): 0 accepted, 1 nothing converged (C = 0), 2 every converged
        stage looks trapped (C of the last one; L457: raise chi)."""
        if not hasattr(self, "obs_prev_C"):
            self.obs_prev_C, self.obs_prev_gerr = 1.0, 0.0            # C(0) = 1
        last = 2 if damping2 is not None else 1
        first, sweeps, C, have, trapped = 0, 0, 0.0, False, False
        status = 1
        while first <= last:
            status, n, _ = self.bp_converge(tol, damping, max_sweeps, max_sweeps_damped, damping2, first)
            sweeps += n
            if status != 0:
                break
            C = self.correlation()
            have = True
            candidate = sweeps >= 30
            dropped = abs(C) < 0.5 * abs(self.obs_prev_C)
            # "no corresponding increase in gate_err" (L454) needs a reference: none yet -> not a trap
            quiet = self.obs_prev_gerr > 0.0 and not self.gate_err > 2.0 * self.obs_prev_gerr
            if not (candidate and dropped and quiet):
                trapped = False
                break
            trapped = True
            first = self.bp_stage + 1
        out = status
        if have and trapped:
            out = 2
        if out == 0:
            self.obs_prev_C, self.obs_prev_gerr = C, self.gate_err
        return out, (C if have else 0.0), sweeps, getattr(self, "bp_stage", 0)

    # -- NEXT-1: norm-network BP with chi x chi matrix messages ---------------------------
    def _norm_site_contraction(self, v, skip_leg=None):
        """Double-layer contraction of site v with the incoming matrix messages on every leg except
        ``skip_leg``: returns the chi x chi matrix over (k, k') of that leg (SURVEY 8(f):
        Mhat[k,k'] = sum_p sum_{i,i'} psi[..i..,k,p] psi[..i'..,k',p] prod_u M_u[i_u,i'_u]), or the
        scalar f_v when no leg is skipped."""
        legs = self.lat.legs(v)
        psi = self.psi[v]
        B = psi
        for ax, d in enumerate(legs):
            if d == skip_leg:
                continue
            B = np.moveaxis(np.tensordot(B, self.Min[(v, d)], axes=([ax], [0])), -1, ax)   # i -> i'
        if skip_leg is None:
            return float(np.sum(B * psi))
        ax = legs.index(skip_leg)
        Bm = np.moveaxis(B, ax, 0).reshape(psi.shape[ax], -1)
        Pm = np.moveaxis(psi, ax, 0).reshape(psi.shape[ax], -1)
        return Bm @ Pm.T

    def norm_bp_init(self):
        """Initial messages = the stored diag(lambda_e) in both directions."""
        self.Min = {}
        for v in range(self.lat.n_sites):
            for d in self.lat.legs(v):
                self.Min[(v, d)] = np.diag(self.lam[self.lat.bond_id(v, d)])

    def norm_bp_sweep(self, damping):
        """One Jacobi sweep: every message recomputed from the previous sweep's; symmetrised, normalised
        to Frobenius norm 1 (matches sum lambda^2 = 1, eq. (12)), damped as eq. (19); delta as eq. (14)."""
        back = {"U": "D", "D": "U", "L": "R", "R": "L"}
        new, delta = {}, 0.0
        for v in range(self.lat.n_sites):
            for d in self.lat.legs(v):
                Mh = self._norm_site_contraction(v, skip_leg=d)        # leaves v through leg d
                Mh = 0.5 * (Mh + Mh.T)
                nrm = np.linalg.norm(Mh)
                u = self.lat.neighbour(v, d)
                old = self.Min[(u, back[d])]                           # it ARRIVES at the neighbour
                if nrm == 0.0 or not math.isfinite(nrm):
                    new[(u, back[d])] = old.copy()
                    continue
                Mn = damping * old + (1.0 - damping) * (Mh / nrm)
                delta = max(delta, float(np.max(np.abs(Mn - old))))
                new[(u, back[d])] = Mn
        self.Min = new
        return delta

    def norm_bp_converge(self, tol, damping=0.0, max_sweeps=100):
        """Sweeps from the CURRENT messages (norm_bp_init() first if there are none) until delta < tol.
        Returns (status, sweeps, delta)."""
        if self.Min is None:
            self.norm_bp_init()
        delta = float("inf")
        for n in range(1, max_sweeps + 1):
            delta = self.norm_bp_sweep(damping)
            if delta < tol:
                return 0, n, delta
        return 1, max_sweeps, delta

    def bethe_norm(self):
        """Bethe norm of Table 1: exp(sum_v log f_v - sum_e log Z_e), f_v the full
        double-layer site contraction, Z_e = sum_{kk'} M_{a->b}[k,k'] M_{b->a}[k,k']."""
        log_n = 0.0
        for v in range(self.lat.n_sites):
            log_n += math.log(self._norm_site_contraction(v))
        for e in range(self.lat.n_bonds):
            v1, d1, v2, d2 = self.lat.bond_sites(e)
            log_n -= math.log(float(np.sum(self.Min[(v1, d1)] * self.Min[(v2, d2)])))
        return math.exp(log_n)

    # -- a15: Bethe evaluation -----------------------------------------------------------
    def correlation(self):
        """eq. (7)-(9) PAPER L112-L128: C = prod vs_v / prod Z_e, evaluated in log space with
        explicit sign tracking.  R14: a zero vs_v gives C = 0; a zero Z_e is an error."""
        msgs = self.msgs
        log_num, sign = 0.0, 1.0
        for v in range(self.lat.n_sites):
            legs = self.lat.legs(v)
            t = self.pinned(v)
            for ax in reversed(range(len(legs))):
                t = np.tensordot(t, self._incoming(msgs, v, legs[ax]), axes=([ax], [0]))
            vs = float(t)
            if vs == 0.0:
                return 0.0
            log_num += math.log(abs(vs))
            sign *= math.copysign(1.0, vs)
        log_den = 0.0
        for e in range(self.lat.n_bonds):
            v1, d1, v2, d2 = self.lat.bond_sites(e)
            Ze = float(np.dot(msgs[(v1, d1)], msgs[(v2, d2)]))      # eq. (8)
            if Ze == 0.0:
                raise FloatingPointError("Z_e = 0")
            log_den += math.log(abs(Ze))
            sign *= math.copysign(1.0, Ze)
        return math.exp(log_num - log_den) * sign                   # eq. (9)

    # -- exact contraction of the pinned network (oracle-only, tiny grids) --------------
    def exact_contraction(self):
        """Brute-force contraction of prod_v T_v over all bonds (PAPER L112 step 1: 'summing
        over every shared bond index across the whole lattice').  Separates 'tensor update
        wrong' from 'BP approximate'.  Exponential cost: tiny grids only."""
        lat = self.lat
        operands = []
        for v in range(lat.n_sites):
            operands.append(self.pinned(v))
            operands.append([lat.bond_id(v, d) for d in lat.legs(v)])
        operands.append([])
        return float(np.einsum(*operands, optimize="greedy"))


def run_trajectory(Lx, Ly, cx, cy, J, h, dt, chi_max, n_steps, bp_tol, bp_damping=0.0,
                   eps_cut=1e-11, max_sweeps=100, max_sweeps_damped=1000, **kw):
    """C(t) after every step: trotter_step -> bp_converge -> correlation (PAPER Fig. 1)."""
    st = PEPOState(Lx, Ly, cx, cy, J, h, dt, chi_max, eps_cut=eps_cut, **kw)
    out = []
    for _ in range(n_steps):
        st.trotter_step()
        status, sweeps, delta = st.bp_converge(bp_tol, bp_damping, max_sweeps, max_sweeps_damped)
        out.append(dict(C=st.correlation(), status=status, sweeps=sweeps, delta=delta,
                        gate_err=st.gate_err, chi=st.bond_dims()))
    return st, out


# --------------------------------------------------------------------------------------
# a16: the paper's analytic memory model (eq. (15)-(17))
# --------------------------------------------------------------------------------------
def paper_memory_model_bytes(k: int, l: int, chi: int, D: int = 4, sizeof: int = 4):
    """(M_psi, M_mu, M_W) in bytes exactly as printed in eq. (15), (16), (17)."""
    M_psi = (4 * chi ** 2 + 2 * (k + l - 4) * chi ** 3 + (k - 2) * (l - 2) * chi ** 4) * D * sizeof
    M_mu = 2 * (k * (l - 1) + (k - 1) * l) * chi ** 2 * sizeof
    M_W = (4 * chi ** 3 * D * chi + 9 * (D * chi) ** 2 + 8 * chi ** 2) * sizeof
    return M_psi, M_mu, M_W
