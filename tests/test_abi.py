"""Host-only checks of the C-ABI boundary (no GPU needed): the shared library loads, exports
every symbol include/pepo.h declares, the Python binding covers them, and the analytic memory
model (pepo_arena_bytes) agrees with a closed form written out here from DESIGN.md section 5."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pepo.h")
LIB = os.path.join(ROOT, "paper_2606_30985_b200", "libpepo_b200.so")


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pepo_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(LIB):
        import __graft_entry__
        __graft_entry__.build()
    return ctypes.CDLL(LIB)


def test_header_declares_the_contract_calls():
    syms = declared_symbols()
    for must in ("pepo_init", "pepo_trotter_step", "pepo_bp_converge", "pepo_correlation", "pepo_arena_bytes",
                 "pepo_permute", "pepo_cholqr", "pepo_householder_qr", "pepo_svd_jacobi", "pepo_gram"):
        assert must in syms


def test_library_exports_every_declared_symbol(lib):
    missing = [s for s in declared_symbols() if not hasattr(lib, s)]
    assert not missing, missing


def test_binding_covers_every_declared_symbol():
    from paper_2606_30985_b200 import binding
    assert sorted(binding.EXPORTED) == declared_symbols()


def test_bad_arguments_do_not_need_a_gpu(lib):
    lib.pepo_arena_bytes.restype = ctypes.c_size_t
    assert lib.pepo_arena_bytes(0, 3, 8) == 0
    assert lib.pepo_arena_bytes(3, 3, 0) == 0
    lib.pepo_last_error.restype = ctypes.c_char_p
    assert lib.pepo_trotter_step(None) == -1
    assert b"NULL" in lib.pepo_last_error()


def gram_splits(m, n, bound=False):
    """Split-K factor of the Gram kernel, restated from DESIGN.md section 5 (independent of the library):
    upper-triangle tiles of 80 (n % 80 == 0), 64 (n <= 64) or 128; enough splits to fill 2 resident CTAs on
    148 SMs (two whole waves for the 80-tile), at least 256 rows per split, chunks rounded up to 16 rows.
    bound=True: the count before the chunk rounding = the largest count any m' <= m can get (the rounded
    count is not monotone in m; the per-lane workspace of a run is sized with the bound)."""
    if n % 80 == 0:
        bt, target, cap, whole = 80, 148 * 2 * 2, 200, True
    elif n <= 64:
        bt, target, cap, whole = 64, 148 * 4, 1024, False
    else:
        bt, target, cap, whole = 128, 148 * 2, 128, False
    tn = -(-n // bt)
    upper = tn * (tn + 1) // 2
    ks = max(1, target // upper) if whole else -(-target // upper)
    ks = max(1, min(ks, (m + 255) // 256, cap))
    if bound:
        return ks
    kc = -(-m // ks)
    kc = -(-kc // 16) * 16
    return -(-m // kc)


def closed_form_bytes(Lx, Ly, chi, B):
    """DESIGN.md section 5, term by term, written out here independently of the library: site slots +
    BP partials + B lanes x 2 site slots (explicit work matrix cv, one spare site slot per site class -
    the largest doubling as the Householder work matrix -, split-K partials, small dense buffers) +
    per-lane core / SVD buffers.  Dominant terms only (the O(n_bonds chi) vectors are left out)."""
    n, N = 4 * chi, 4 * chi
    doubles = 0
    degs = set()
    for y in range(Ly):
        for x in range(Lx):
            hU, hD, hL, hR = y > 0, y < Ly - 1, x > 0, x < Lx - 1
            deg = hU + hD + hL + hR
            degs.add(deg)
            doubles += 4 * chi ** deg                                                  # psi_v
            # BP partials: per-chunk vectors for the first two legs that exist, slice scalars for the others
            doubles += (chi ** ((deg >= 1) + (deg >= 3) + (deg >= 4)) + chi ** ((deg >= 2) + (deg >= 3) + (deg >= 4))
                        + chi ** ((deg >= 3) + (deg >= 4)))
            doubles += 64 * 4 + 4                                                      # n(r,t) partials
    n_bonds = Ly * (Lx - 1) + (Ly - 1) * Lx
    doubles += 8 * n_bonds * chi * chi + 22 * chi * chi      # matrix messages (2 sets, sqrt, inverse sqrt) + their workspace
    degmax = max(degs)
    m_max = chi ** max(degmax - 1, 0)
    ld = (m_max + 1) // 2 * 2
    part = max(gram_splits(m_max, 4 * c, bound=True) * (4 * c) ** 2 for c in range(1, chi + 1))
    spares = sum(4 * chi ** d for d in degs if 1 <= d < degmax) + max(ld * n, 4 * chi ** degmax)
    slot = ld * n + spares + part + n * n + 2 * N * N + n * n + 4 * n * N + N * chi + n * 4 * chi + 4 * n * chi
    lane = 2 * slot + 4 * N * N + 2 * N * chi
    doubles += B * lane
    # every sub-buffer starts on a 256-byte boundary and is followed by 64 guard bytes (pepo_check_guards):
    # 4 buffers per site, 34 global ones, 14 + one per site class per lane slot, 8 per lane
    n_buffers = 4 * Lx * Ly + 34 + B * (2 * (14 + len([d for d in degs if d >= 1])) + 8)
    return 8 * doubles + n_buffers * (128 + 64)


@pytest.mark.parametrize("Lx,Ly,chi", [(3, 3, 8), (4, 4, 60), (8, 8, 60), (10, 10, 95)])
def test_memory_model_matches_closed_form(lib, Lx, Ly, chi):
    lib.pepo_arena_bytes_ex.restype = ctypes.c_size_t
    for B in (1, 4):
        got = lib.pepo_arena_bytes_ex(Lx, Ly, chi, B)
        want = closed_form_bytes(Lx, Ly, chi, B)
        assert abs(got - want) <= 0.02 * want, (got, want)


def test_split_k_workspace_covers_every_smaller_row_count(lib):
    """The per-lane split-K workspace is shared by all the sites a lane meets, with every row count m <= m_max
    (mixed bond dimensions during growth).  pepo_gram_ws_bytes(m, n) is not monotone in m (62400 x 160 needs
    195 splits, 64000 x 160 only 191: seen as an overwritten arena guard at 4x4 chi 40, step 11), so the
    layout's bound must cover all of them."""
    lib.pepo_gram_ws_bytes.restype = ctypes.c_size_t
    lib.pepo_gram_ws_bytes.argtypes = [ctypes.c_longlong, ctypes.c_int]
    assert lib.pepo_gram_ws_bytes(62400, 160) > lib.pepo_gram_ws_bytes(64000, 160)
    rng = np.random.default_rng(3)
    for chi in (40, 60):
        m_max = chi ** 3
        cap = 8 * max(gram_splits(m_max, 4 * c, bound=True) * (4 * c) ** 2 for c in range(1, chi + 1))
        dims = list(range(max(1, chi - 12), chi + 1))
        for _ in range(4000):
            a, b, c3, cc = rng.choice(dims, 4)
            assert lib.pepo_gram_ws_bytes(int(a * b * c3), int(4 * cc)) <= cap + 256, (a, b, c3, cc)


def test_config5_sized_to_fit_180GB(lib):
    """BASELINE config 5: chi_max = 100 does not fit 180 GB in fp64 (sites alone are 205 GB);
    the model says which chi_max does."""
    lib.pepo_arena_bytes_ex.restype = ctypes.c_size_t
    assert lib.pepo_arena_bytes_ex(10, 10, 100, 1) > 180e9
    fits = [c for c in range(80, 101) if lib.pepo_arena_bytes_ex(10, 10, c, 1) <= 180e9]
    assert fits and 90 <= max(fits) <= 97
