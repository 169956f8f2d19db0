"""Thin ctypes binding of the C ABI in ``include/pepo.h`` (argument marshalling only: every
step of the hot path runs in the CUDA kernels of ``libpepo_b200.so``).

PyTorch supplies device memory (the arena, kernel-level tensors) and the stream.  There is no
CPU fallback: importing this module without the built library raises, and every call raises
``PepoError`` on a negative return code.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpepo_b200.so")


class PepoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pepo error %d: %s" % (code, msg))
        self.code = code


class PepoStats(C.Structure):
    _fields_ = [("gate_err", C.c_double), ("min_cut_gap", C.c_double),
                ("n_cholesky", C.c_longlong), ("n_householder", C.c_longlong),
                ("n_chol_failed", C.c_longlong), ("jacobi_sweeps", C.c_longlong),
                ("kernel_launches", C.c_longlong), ("last_bp_sweeps", C.c_int),
                ("last_bp_status", C.c_int), ("last_bp_delta", C.c_double),
                ("arena_high_water", C.c_size_t), ("arena_model_bytes", C.c_size_t),
                ("max_inflight_gates", C.c_int), ("chi_max_live", C.c_int), ("last_bp_trap", C.c_int),
                ("last_bp_stage", C.c_int), ("last_bp_flags", C.c_int)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            "libpepo_b200.so is not built (run `python -m paper_2606_30985_b200.build`); "
            "there is no CPU fallback for the hot path")
    lib = C.CDLL(LIB_PATH)
    vp, dp, ip, sz, ll, i, d = (C.c_void_p, C.c_void_p, C.POINTER(C.c_int), C.c_size_t,
                                C.c_longlong, C.c_int, C.c_double)
    sig = {
        "pepo_last_error": (C.c_char_p, []),
        "pepo_arena_bytes": (sz, [i, i, i]),
        "pepo_arena_bytes_ex": (sz, [i, i, i, i]),
        "pepo_init": (i, [C.POINTER(vp), i, i, i, i, d, d, d, i, d, d, vp, sz, vp]),
        "pepo_init_ex": (i, [C.POINTER(vp), i, i, i, i, d, d, d, i, d, d, vp, sz, vp, i, i, i, i]),
        "pepo_destroy": (i, [vp]),
        "pepo_set_option": (i, [vp, C.c_char_p, d]),
        "pepo_trotter_step": (i, [vp]),
        "pepo_apply_field": (i, [vp]),
        "pepo_apply_bond": (i, [vp, i]),
        "pepo_bp_converge": (i, [vp, ip, C.POINTER(d)]),
        "pepo_correlation": (i, [vp, C.POINTER(d)]),
        "pepo_observe": (i, [vp, C.POINTER(d), ip, ip]),
        "pepo_get_stats": (i, [vp, C.POINTER(PepoStats)]),
        "pepo_check_guards": (i, [vp]),
        "pepo_get_profile": (i, [vp, i, C.POINTER(d), C.POINTER(d), C.POINTER(d), C.POINTER(ll)]),
        "pepo_n_bonds": (i, [vp]),
        "pepo_get_bond_dims": (i, [vp, ip]),
        "pepo_set_bond_dims": (i, [vp, ip]),
        "pepo_site_size": (sz, [vp, i, i]),
        "pepo_get_site": (i, [vp, i, i, vp, sz]),
        "pepo_set_site": (i, [vp, i, i, vp, sz]),
        "pepo_set_site_async": (i, [vp, i, i, vp, sz]),
        "pepo_site_order": (i, [vp, vp, i]),
        "pepo_get_lambda": (i, [vp, i, vp, i]),
        "pepo_bond_entropy": (i, [vp, vp, i]),
        "pepo_get_message": (i, [vp, i, i, vp, i]),
        "pepo_site_weights": (i, [vp, vp, i, vp]),
        "pepo_norm_bp_converge": (i, [vp, d, d, i, ip, C.POINTER(d)]),
        "pepo_bethe_norm": (i, [vp, C.POINTER(d)]),
        "pepo_get_norm_message": (i, [vp, i, i, vp, i]),
        "pepo_set_lambda": (i, [vp, i, vp, i]),
        "pepo_site_ptr": (vp, [vp, i, i]),
        "pepo_permute": (i, [dp, dp, ip, ip, i, vp]),
        "pepo_permute_scaled": (i, [dp, dp, ip, ip, i, C.POINTER(vp), vp]),
        "pepo_gram_ws_bytes": (sz, [ll, i]),
        "pepo_gram": (i, [dp, ll, i, ll, dp, vp, sz, vp]),
        "pepo_static_scratch_bytes": (sz, []),
        "pepo_gram_static": (i, [dp, ll, i, ll, dp, vp]),
        "pepo_site_gram_ws_bytes": (sz, [ip, i, i]),
        "pepo_site_gram": (i, [dp, ip, i, i, C.POINTER(vp), dp, vp, sz, vp]),
        "pepo_site_apply": (i, [dp, ip, i, i, dp, i, dp, vp]),
        "pepo_dmma_peak": (i, [i, i, dp, C.POINTER(d), vp]),
        "pepo_cholqr_ws_bytes": (sz, [ll, i]),
        "pepo_cholqr": (i, [dp, ll, i, ll, dp, dp, vp, vp, sz, vp]),
        "pepo_householder_ws_bytes": (sz, [ll, i]),
        "pepo_householder_qr": (i, [dp, ll, i, ll, dp, dp, vp, sz, vp]),
        "pepo_svd_ws_bytes": (sz, [i, i]),
        "pepo_svd_jacobi": (i, [dp, i, i, i, dp, dp, dp, vp, vp, sz, vp]),
        "pepo_dgemm": (i, [i, i, ll, i, i, dp, ll, dp, ll, dp, ll, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    return lib, sorted(sig)


_lib, EXPORTED = _load()


def last_error() -> str:
    return _lib.pepo_last_error().decode()


def _check(rc):
    if rc < 0:
        raise PepoError(rc, last_error())
    return rc


def _stream(stream=None):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _iarr(v):
    return (C.c_int * len(v))(*[int(x) for x in v])


def _f64(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("%s must be a contiguous CUDA float64 tensor" % name)
    return C.c_void_p(t.data_ptr())


def arena_bytes(Lx, Ly, chi_max, max_inflight=0):
    return int(_lib.pepo_arena_bytes_ex(Lx, Ly, chi_max, max_inflight))


class Pepo:
    """Context of one simulation (see ``include/pepo.h``).  Owns the arena tensor."""

    def __init__(self, Lx, Ly, cx, cy, J, h, dt, chi_max, bp_tol, bp_damping=0.0, device="cuda:0",
                 max_inflight=0, bond_pauli=3, field_pauli=1, obs_pauli=3, arena=None):
        self.Lx, self.Ly, self.chi_max = Lx, Ly, chi_max
        self.device = torch.device(device)
        need = arena_bytes(Lx, Ly, chi_max, max_inflight)
        if need == 0:
            raise PepoError(-1, "bad grid / chi_max")
        with torch.cuda.device(self.device):
            self.arena = arena if arena is not None else torch.empty(need, dtype=torch.uint8, device=self.device)
            self.stream = torch.cuda.current_stream()
            h_ = C.c_void_p()
            _check(_lib.pepo_init_ex(C.byref(h_), Lx, Ly, cx, cy, J, h, dt, chi_max, bp_tol, bp_damping,
                                     C.c_void_p(self.arena.data_ptr()), self.arena.numel(),
                                     _stream(self.stream), max_inflight, bond_pauli, field_pauli, obs_pauli))
        self._h = h_
        self.n_bonds = _lib.pepo_n_bonds(self._h)

    def close(self):
        if getattr(self, "_h", None):
            _lib.pepo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        _check(_lib.pepo_set_option(self._h, key.encode(), float(value)))

    def trotter_step(self):
        _check(_lib.pepo_trotter_step(self._h))

    def apply_field(self):
        _check(_lib.pepo_apply_field(self._h))

    def apply_bond(self, bond):
        _check(_lib.pepo_apply_bond(self._h, int(bond)))

    def bp_converge(self):
        sw, de = C.c_int(0), C.c_double(0.0)
        status = _check(_lib.pepo_bp_converge(self._h, C.byref(sw), C.byref(de)))
        return status, sw.value, de.value

    def correlation(self):
        out = C.c_double(0.0)
        _check(_lib.pepo_correlation(self._h, C.byref(out)))
        return out.value

    def observe(self):
        """(status, C, sweeps, stage) of BP + Bethe with the alpha-retry / trap-verification procedure."""
        out, sw, stg = C.c_double(0.0), C.c_int(0), C.c_int(0)
        status = _check(_lib.pepo_observe(self._h, C.byref(out), C.byref(sw), C.byref(stg)))
        return status, out.value, sw.value, stg.value

    def check_guards(self):
        _check(_lib.pepo_check_guards(self._h))

    def stats(self):
        s = PepoStats()
        _check(_lib.pepo_get_stats(self._h, C.byref(s)))
        return {k: getattr(s, k) for k, _ in PepoStats._fields_}

    PROFILE_CLASSES = ("permute", "gram", "apply_gemm", "small_gemm", "cholesky", "householder",
                       "dress", "svd", "field", "bp")

    def profile(self):
        n = len(self.PROFILE_CLASSES)
        ms, fl, by = (C.c_double * n)(), (C.c_double * n)(), (C.c_double * n)()
        cnt = (C.c_longlong * n)()
        _check(_lib.pepo_get_profile(self._h, n, ms, fl, by, cnt))
        return {k: dict(ms=ms[i], flops=fl[i], bytes=by[i], count=cnt[i]) for i, k in enumerate(self.PROFILE_CLASSES)}

    def bond_dims(self):
        arr = (C.c_int * max(self.n_bonds, 1))()
        _check(_lib.pepo_get_bond_dims(self._h, arr))
        return [arr[i] for i in range(self.n_bonds)]

    def set_bond_dims(self, chi):
        assert len(chi) == self.n_bonds
        _check(_lib.pepo_set_bond_dims(self._h, _iarr(chi) if chi else (C.c_int * 1)()))

    def site_size(self, x, y):
        return int(_lib.pepo_site_size(self._h, x, y))

    def get_site(self, x, y):
        out = np.empty(self.site_size(x, y), dtype=np.float64)
        _check(_lib.pepo_get_site(self._h, x, y, out.ctypes.data_as(C.c_void_p), out.size))
        return out

    def set_site(self, x, y, flat):
        flat = np.ascontiguousarray(flat, dtype=np.float64).ravel()
        _check(_lib.pepo_set_site(self._h, x, y, flat.ctypes.data_as(C.c_void_p), flat.size))

    def set_site_async(self, x, y, flat):
        """flat: contiguous float64 array (pinned for a truly asynchronous copy) that the caller
        keeps alive and unchanged until trotter_step / bp_converge / correlation has returned."""
        if flat.dtype != np.float64 or not flat.flags["C_CONTIGUOUS"]:
            raise ValueError("set_site_async needs a contiguous float64 array")
        _check(_lib.pepo_set_site_async(self._h, x, y, flat.ctypes.data_as(C.c_void_p), flat.size))

    def site_order(self):
        """(x, y) of the sites in the order the next trotter_step first touches them."""
        n = self.Lx * self.Ly
        out = np.empty(n, dtype=np.int32)
        _check(_lib.pepo_site_order(self._h, out.ctypes.data_as(C.c_void_p), n))
        return [(int(v) % self.Lx, int(v) // self.Lx) for v in out]

    def bond_entropy(self):
        out = np.empty(self.n_bonds, dtype=np.float64)
        _check(_lib.pepo_bond_entropy(self._h, out.ctypes.data_as(C.c_void_p), self.n_bonds))
        return out

    def get_lambda(self, bond):
        n = self.bond_dims()[bond]
        out = np.empty(n, dtype=np.float64)
        _check(_lib.pepo_get_lambda(self._h, bond, out.ctypes.data_as(C.c_void_p), n))
        return out

    def site_weights(self):
        """(n(r) per site [y*Lx + x], (R_L1, R_L2, S_frac)) - PAPER.md section 6.4 / eq. (21)."""
        n = self.Lx * self.Ly
        out = np.empty(n, dtype=np.float64)
        spread = np.empty(3, dtype=np.float64)
        _check(_lib.pepo_site_weights(self._h, out.ctypes.data_as(C.c_void_p), n, spread.ctypes.data_as(C.c_void_p)))
        return out, tuple(spread)

    def norm_bp_converge(self, tol, damping=0.0, max_sweeps=100):
        sw, de = C.c_int(0), C.c_double(0.0)
        status = _check(_lib.pepo_norm_bp_converge(self._h, float(tol), float(damping), int(max_sweeps), C.byref(sw), C.byref(de)))
        return status, sw.value, de.value

    def bethe_norm(self):
        out = C.c_double(0.0)
        _check(_lib.pepo_bethe_norm(self._h, C.byref(out)))
        return out.value

    def get_norm_message(self, bond, from_v1=True):
        chi = self.bond_dims()[bond]
        out = np.empty(chi * chi, dtype=np.float64)
        _check(_lib.pepo_get_norm_message(self._h, bond, 1 if from_v1 else 0, out.ctypes.data_as(C.c_void_p), chi * chi))
        return out.reshape((chi, chi), order="F")

    def get_message(self, bond, from_v1=True):
        n = self.bond_dims()[bond]
        out = np.empty(n, dtype=np.float64)
        _check(_lib.pepo_get_message(self._h, bond, 1 if from_v1 else 0, out.ctypes.data_as(C.c_void_p), n))
        return out

    def set_lambda(self, bond, lam):
        lam = np.ascontiguousarray(lam, dtype=np.float64).ravel()
        _check(_lib.pepo_set_lambda(self._h, bond, lam.ctypes.data_as(C.c_void_p), lam.size))


# ---- kernel-level entry points (device tensors in, device tensors out) ------------------------
def permute(src, shape, perm, dst=None, scale=None):
    """``src``: flat CUDA f64 tensor holding a packed column-major tensor of dims ``shape``
    (first fastest).  Returns the packed column-major permuted tensor (flat)."""
    _f64(src, "src")
    if dst is None:
        dst = torch.empty_like(src)
    if scale is None:
        _check(_lib.pepo_permute(_f64(src, "src"), _f64(dst, "dst"), _iarr(shape), _iarr(perm), len(shape), _stream()))
    else:
        ptrs = (C.c_void_p * len(shape))(*[C.c_void_p(s.data_ptr()) if s is not None else C.c_void_p(0) for s in scale])
        _check(_lib.pepo_permute_scaled(_f64(src, "src"), _f64(dst, "dst"), _iarr(shape), _iarr(perm), len(shape),
                                        ptrs, _stream()))
    return dst


def _ws(nbytes, device):
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def gram(A_cm, m, n, ws=None):
    """A_cm: flat column-major m x n.  Returns C (n x n column-major, flat)."""
    Cm = torch.empty(n * n, dtype=torch.float64, device=A_cm.device)
    ws = ws if ws is not None else _ws(_lib.pepo_gram_ws_bytes(m, n), A_cm.device)
    _check(_lib.pepo_gram(_f64(A_cm, "A"), m, n, m, _f64(Cm, "C"), C.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return Cm


def static_scratch_bytes():
    return int(_lib.pepo_static_scratch_bytes())


def gram_static(A_cm, m, n, out):
    """pepo_gram_static: C = A^T A into the caller's `out` (n*n float64 on A's device) with the split-K
    scratch in the library's built-in device array: no allocation anywhere.  Raises PepoError(-2) when
    the plan needs more than static_scratch_bytes().  Calls on one device must not overlap on the GPU."""
    if out.numel() < n * n:
        raise PepoError(-1, "gram_static: out too small")
    _check(_lib.pepo_gram_static(_f64(A_cm, "A"), m, n, m, _f64(out, "out"), _stream()))
    return out


def site_gram(psi, dims, cut, w2=None):
    """psi: flat packed site tensor (dims + Pauli leg 4, column-major).  Returns the n x n Gram matrix
    (flat column-major, n = 4 dims[cut]) of the matrix view rows = other legs, cols = (cut, P), with the
    rows weighted by prod w2[leg][i_leg] (w2: list of CUDA vectors per leg, entry `cut` ignored)."""
    n = 4 * dims[cut] if 0 <= cut < len(dims) else 4
    Cm = torch.empty(n * n, dtype=torch.float64, device=psi.device)
    ws = _ws(_lib.pepo_site_gram_ws_bytes(_iarr(dims), len(dims), cut), psi.device)
    ptrs = None
    if w2 is not None:
        ptrs = (C.c_void_p * len(dims))(*[C.c_void_p(w.data_ptr()) if w is not None else C.c_void_p(0) for w in w2])
    _check(_lib.pepo_site_gram(_f64(psi, "psi"), _iarr(dims), len(dims), cut, ptrs, _f64(Cm, "C"),
                               C.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return Cm


def site_apply(psi, dims, cut, W, chi_new):
    """Returns the packed site tensor with dims[cut] -> chi_new: psi contracted over (cut, P) with W."""
    tot = 4 * chi_new
    for l, d in enumerate(dims):
        if l != cut:
            tot *= d
    out = torch.empty(tot, dtype=torch.float64, device=psi.device)
    _check(_lib.pepo_site_apply(_f64(psi, "psi"), _iarr(dims), len(dims), cut, _f64(W, "W"), chi_new,
                                _f64(out, "out"), _stream()))
    return out


def dmma_peak(iters, ctas_per_sm, sink):
    """Launch the register-only DMMA loop; returns the flops of the launch (time it with CUDA events)."""
    fl = C.c_double(0.0)
    _check(_lib.pepo_dmma_peak(int(iters), int(ctas_per_sm), _f64(sink, "sink"), C.byref(fl), _stream()))
    return fl.value


def cholqr(A_cm, m, n, Q=None, ws=None):
    Q = Q if Q is not None else torch.empty(m * n, dtype=torch.float64, device=A_cm.device)
    R = torch.empty(n * n, dtype=torch.float64, device=A_cm.device)
    info = torch.zeros(1, dtype=torch.int32, device=A_cm.device)
    ws = ws if ws is not None else _ws(_lib.pepo_cholqr_ws_bytes(m, n), A_cm.device)
    _check(_lib.pepo_cholqr(_f64(A_cm, "A"), m, n, m, _f64(Q, "Q"), _f64(R, "R"), C.c_void_p(info.data_ptr()),
                            C.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return Q, R, info


def householder_qr(A_cm, m, n):
    k = min(m, n)
    Q = torch.empty(m * k, dtype=torch.float64, device=A_cm.device)
    R = torch.empty(k * n, dtype=torch.float64, device=A_cm.device)
    ws = _ws(_lib.pepo_householder_ws_bytes(m, n), A_cm.device)
    _check(_lib.pepo_householder_qr(_f64(A_cm, "A"), m, n, m, _f64(Q, "Q"), _f64(R, "R"),
                                    C.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return Q, R


def svd_jacobi(A_cm, m, n):
    r = min(m, n)
    U = torch.empty(m * r, dtype=torch.float64, device=A_cm.device)
    s = torch.empty(r, dtype=torch.float64, device=A_cm.device)
    V = torch.empty(n * r, dtype=torch.float64, device=A_cm.device)
    sweeps = torch.zeros(1, dtype=torch.int32, device=A_cm.device)
    ws = _ws(_lib.pepo_svd_ws_bytes(m, n), A_cm.device)
    _check(_lib.pepo_svd_jacobi(_f64(A_cm, "A"), m, n, m, _f64(U, "U"), _f64(s, "s"), _f64(V, "V"),
                                C.c_void_p(sweeps.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(), _stream()))
    return U, s, V, sweeps


def dgemm(transA, transB, M, N, K, A, lda, B, ldb, Cout=None, ldc=None):
    ldc = ldc or M
    Cout = Cout if Cout is not None else torch.empty(ldc * N, dtype=torch.float64, device=A.device)
    _check(_lib.pepo_dgemm(int(transA), int(transB), M, N, K, _f64(A, "A"), lda, _f64(B, "B"), ldb,
                           _f64(Cout, "C"), ldc, _stream()))
    return Cout
