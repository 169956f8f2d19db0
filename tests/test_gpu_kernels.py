"""GPU parity of the kernel-level C-ABI entry points against the CPU oracle (oracle/), element
by element on seeded inputs.  -m gpu.  Integer / copy work is bit-exact; floating point is
within the tolerances of BASELINE.json's north_star (1e-12 relative Frobenius for QR / SVD
reconstructions)."""
import itertools

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_30985_b200 import binding
    return torch, binding


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


# ------------------------------------------------------------------ permutation (a4 / a11) ---
@pytest.mark.parametrize("shape", [(5, 3, 4, 2, 4), (7, 6, 5, 3, 4), (33, 4, 9, 2, 4), (70, 3, 67, 1, 4)])
def test_permute_all_perms_bit_exact(gpu, shape):
    """Every axis permutation of a small ragged rank-5 tensor vs Listing 1."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    src = inputs.normal_tensor(shape, seed=1)
    d_src = _dev(torch, src)
    for perm in itertools.permutations(range(5)):
        want = po.permute_listing1(src, shape, perm)
        got = B.permute(d_src, shape, perm).cpu().numpy()
        assert np.array_equal(got.view(np.int64), want.view(np.int64)), (shape, perm)


@pytest.mark.parametrize("rank", [1, 2, 3, 4, 6])
def test_permute_other_ranks(gpu, rank):
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    shape = [9, 5, 34, 3, 2, 6][:rank]
    src = inputs.normal_tensor(shape, seed=2)
    d_src = _dev(torch, src)
    perms = list(itertools.permutations(range(rank)))
    for perm in perms[:: max(1, len(perms) // 40)]:
        want = po.permute_listing1(src, shape, perm)
        got = B.permute(d_src, shape, perm).cpu().numpy()
        assert np.array_equal(got.view(np.int64), want.view(np.int64)), (shape, perm)


def test_permute_in_method_cases_chi40(gpu):
    """The permutations Algorithm 1 itself uses: cut-leg-to-last on a rank-5
    site tensor with chi = 40 (several tiles + ragged tail), checked bit-exactly on all elements."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    chi = 40
    shape = (chi, chi, chi, chi, 4)
    src = inputs.normal_tensor(shape, seed=1)
    d_src = _dev(torch, src)
    for perm in [(1, 2, 3, 0, 4), (0, 2, 3, 1, 4), (0, 1, 3, 2, 4), (3, 0, 1, 2, 4), (4, 0, 1, 2, 3), (4, 3, 2, 1, 0)]:
        want = po.permute_listing1(src, shape, perm)
        got = B.permute(d_src, shape, perm).cpu().numpy()
        assert np.array_equal(got.view(np.int64), want.view(np.int64)), perm
        # permutation composed with its inverse is the identity (pin P9)
        inv = np.argsort(perm)
        shp2 = [shape[p] for p in perm]
        back = B.permute(_dev(torch, got), shp2, inv).cpu().numpy()
        assert np.array_equal(back.view(np.int64), src.view(np.int64))


def test_permute_scaled_matches_absorb(gpu):
    """a3 + a4 fused: scale by sqrt(lambda) on the env legs then permute."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    shape = (6, 35, 7, 5, 4)
    rng = np.random.default_rng(5)
    src = inputs.normal_tensor(shape, seed=3)
    scales = [rng.uniform(0.1, 1.0, s) for s in shape[:3]] + [None, None]
    t = src.reshape(shape, order="F").copy()
    for ax, s in enumerate(scales):
        if s is not None:
            shp = [1] * 5
            shp[ax] = shape[ax]
            t = t * s.reshape(shp)
    perm = (0, 1, 2, 3, 4)
    for perm in [(0, 1, 2, 3, 4), (1, 2, 0, 3, 4), (2, 0, 1, 3, 4), (4, 1, 0, 2, 3)]:
        want = po.permute_listing1(t.flatten(order="F"), shape, perm)
        d_scales = [None if s is None else _dev(torch, s) for s in scales]
        got = B.permute(_dev(torch, src), shape, perm, scale=d_scales).cpu().numpy()
        assert np.allclose(got, want, rtol=2e-15, atol=0), perm   # 3 multiplies, order free


def test_permute_empty_and_errors(gpu):
    torch, B = gpu
    d = torch.zeros(0, dtype=torch.float64, device="cuda")
    out = B.permute(d, (3, 0, 2), (2, 0, 1))
    assert out.numel() == 0
    with pytest.raises(B.PepoError):
        B.permute(torch.zeros(6, dtype=torch.float64, device="cuda"), (3, 2), (0, 0))


# ------------------------------------------------------------------ DGEMM / Gram (a5, a10) ---
@pytest.mark.parametrize("ta,tb", [(0, 0), (1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (37, 29, 53), (300, 130, 77), (1000, 96, 240), (129, 257, 16)])
def test_dgemm_vs_oracle_matmul(gpu, ta, tb, M, N, K):
    torch, B = gpu
    rng = np.random.default_rng(M * 7 + N * 3 + K)
    A = rng.standard_normal((K, M) if ta else (M, K))
    Bm = rng.standard_normal((N, K) if tb else (K, N))
    want = (A.T if ta else A) @ (Bm.T if tb else Bm)
    got = B.dgemm(ta, tb, M, N, K, _dev(torch, A.flatten(order="F")), A.shape[0],
                  _dev(torch, Bm.flatten(order="F")), Bm.shape[0]).cpu().numpy().reshape((M, N), order="F")
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want) + 1e-300


@pytest.mark.parametrize("m,n", [(1000, 40), (4099, 160), (7777, 33), (513, 240), (64, 64), (3, 5)])
def test_gram_vs_definition(gpu, m, n):
    """eq. (10): C = A^T A; symmetric to the bit; split-K deterministic."""
    torch, B = gpu
    A = np.random.default_rng(m + n).standard_normal((m, n))
    dA = _dev(torch, A.flatten(order="F"))
    got = B.gram(dA, m, n).cpu().numpy().reshape((n, n), order="F")
    want = A.T @ A
    assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want)
    assert np.array_equal(got, got.T)
    again = B.gram(dA, m, n).cpu().numpy().reshape((n, n), order="F")
    assert np.array_equal(got, again)


# ------------------------------------------------------------------ QR (a5 / a6) -------------
@pytest.mark.parametrize("m,n", [(2000, 40), (5001, 160), (999, 97), (400, 100)])
def test_cholqr_vs_oracle(gpu, m, n):
    torch, B = gpu
    from oracle import pepo_oracle as po
    A = np.random.default_rng(m * 3 + n).standard_normal((m, n))
    Q, R, info = B.cholqr(_dev(torch, A.flatten(order="F")), m, n)
    assert int(info.item()) == 0
    Q = Q.cpu().numpy().reshape((m, n), order="F")
    R = R.cpu().numpy().reshape((n, n), order="F")
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    assert np.all(np.diag(R) > 0)
    assert np.linalg.norm(A - Q @ R) <= 1e-12 * np.linalg.norm(A)
    assert np.linalg.norm(Q.T @ Q - np.eye(n)) <= 1e-11
    Qo, Ro = po.cholesky_qr(A)
    assert np.linalg.norm(R - Ro) <= 1e-11 * np.linalg.norm(Ro)
    assert np.linalg.norm(Q - Qo) <= 1e-11 * np.linalg.norm(Qo)
    # against Householder after sign normalisation (uniqueness of QR with positive diagonal)
    Qh, Rh = po.householder_qr(A)
    sg = np.sign(np.diag(Rh))
    assert np.linalg.norm(R - sg[:, None] * Rh) <= 1e-10 * np.linalg.norm(Rh)


def test_cholqr_reports_indefinite(gpu):
    """potrf_info != 0 on a rank-deficient matrix."""
    torch, B = gpu
    A = np.random.default_rng(0).standard_normal((500, 24))
    A[:, 7] = 0.0
    _, _, info = B.cholqr(_dev(torch, A.flatten(order="F")), 500, 24)
    assert int(info.item()) == 8


@pytest.mark.parametrize("m,n,kind", [(300, 40, "full"), (64, 256, "wide"), (1, 12, "row"), (500, 32, "deficient"),
                                       (9000, 48, "big"), (700, 400, "bigsq"), (40, 40, "zero")])
def test_householder_qr_vs_oracle(gpu, m, n, kind):
    torch, B = gpu
    from oracle import pepo_oracle as po
    rng = np.random.default_rng(m + 13 * n)
    A = rng.standard_normal((m, n))
    if kind == "deficient":
        A[:, 5] = 0.0
        A[:, 9] = A[:, 3] * 2.0
        A[:, 20:] = A[:, :12] @ rng.standard_normal((12, 12))
    if kind == "zero":
        A[:] = 0.0
    Q, R = B.householder_qr(_dev(torch, A.flatten(order="F")), m, n)
    k = min(m, n)
    Q = Q.cpu().numpy().reshape((m, k), order="F")
    R = R.cpu().numpy().reshape((k, n), order="F")
    assert np.array_equal(np.tril(R, -1), np.zeros_like(R))
    assert np.linalg.norm(A - Q @ R) <= 1e-12 * max(np.linalg.norm(A), 1e-300) + (0 if kind != "zero" else 1e-300)
    assert np.linalg.norm(Q.T @ Q - np.eye(k)) <= 1e-12 * np.sqrt(k) * 10
    if kind in ("full", "big", "bigsq"):
        Qo, Ro = po.householder_qr(A)
        s1, s2 = np.sign(np.diag(R)), np.sign(np.diag(Ro))
        assert np.linalg.norm(s1[:, None] * R - s2[:, None] * Ro) <= 1e-11 * np.linalg.norm(Ro)


# ------------------------------------------------------------------ Jacobi SVD (a9) ----------
@pytest.mark.parametrize("m,n,kind", [(32, 32, "full"), (96, 40, "tall"), (24, 80, "wide"), (64, 64, "lowrank"),
                                       (130, 130, "graded"), (1, 1, "one"), (16, 16, "zero")])
def test_svd_jacobi_vs_oracle(gpu, m, n, kind):
    torch, B = gpu
    rng = np.random.default_rng(m * 5 + n)
    A = rng.standard_normal((m, n))
    if kind == "lowrank":
        A = rng.standard_normal((m, 7)) @ rng.standard_normal((7, n))
    if kind == "graded":
        u, _ = np.linalg.qr(rng.standard_normal((m, m)))
        v, _ = np.linalg.qr(rng.standard_normal((n, n)))
        A = (u * 10.0 ** (-12.0 * np.arange(n) / n)) @ v.T
    if kind == "zero":
        A[:] = 0
    U, s, V, sweeps = B.svd_jacobi(_dev(torch, A.flatten(order="F")), m, n)
    r = min(m, n)
    U = U.cpu().numpy().reshape((m, r), order="F")
    V = V.cpu().numpy().reshape((n, r), order="F")
    s = s.cpu().numpy()
    so = np.linalg.svd(A, compute_uv=False)
    assert np.all(np.diff(s) <= 0) and np.all(s >= 0)
    assert np.allclose(s, so, rtol=0, atol=1e-13 * max(so[0], 1e-300))
    assert np.linalg.norm(A - (U * s) @ V.T) <= 1e-12 * max(np.linalg.norm(A), 1e-300)
    if kind in ("full", "tall", "wide"):
        assert np.linalg.norm(U.T @ U - np.eye(r)) <= 1e-12 * r
        assert np.linalg.norm(V.T @ V - np.eye(r)) <= 1e-12 * r
    if kind == "lowrank":
        assert np.all(s[7:] <= 1e-13 * s[0])


# ------------------------------------------------- permute-on-load contractions (a3-a5, a10-a13) ---
SITE_CASES = [
    # dims of the bond legs (Pauli leg 4 implicit), several tiles + ragged tails, even and odd extents
    (12, 10, 14, 8), (7, 5, 9, 3), (20, 18), (9, 11, 6), (1, 6, 5, 4), (16,), (6, 1, 1, 8), (24, 24, 24, 24),
]


@pytest.mark.parametrize("dims", SITE_CASES, ids=["x".join(map(str, d)) for d in SITE_CASES])
def test_site_gram_and_apply_match_the_explicit_path(gpu, dims):
    """pepo_site_gram / pepo_site_apply read the packed site tensor in place.  Reference = the oracle's
    explicit path on the same seeded tensor: absorb sqrt(lambda) on the environment legs (a3), permute
    the cut leg last with Listing 1 (a4), C = cv^T cv (eq. (10)); out = cv W, inverse permutation (a11),
    de-absorb (a12).  Every cut leg of every shape; tolerance 1e-13 relative Frobenius (a DMMA dot product
    of m <= 3.3e5 terms)."""
    torch, B = gpu
    from oracle import pepo_oracle as po
    from paper_2606_30985_b200 import inputs
    nl = len(dims)
    shape = list(dims) + [4]
    rng = np.random.default_rng(5)
    psi = inputs.normal_tensor(shape, seed=3)
    t = psi.reshape(shape, order="F")
    lam = [np.sort(rng.random(d) + 1e-3)[::-1].copy() for d in dims]        # positive, graded weights
    d_psi = _dev(torch, psi)
    d_lam = [_dev(torch, l) for l in lam]
    for cut in range(nl):
        # ---- oracle: a3 + a4 ----
        ta = t.copy()
        for ax in range(nl):
            if ax != cut:
                shp = [1] * (nl + 1); shp[ax] = dims[ax]
                ta = ta * np.sqrt(lam[ax]).reshape(shp)
        env = [ax for ax in range(nl) if ax != cut]
        perm = env + [cut, nl]
        m = int(np.prod([dims[a] for a in env])) if env else 1
        n = 4 * dims[cut]
        cv = po.permute_listing1(ta.flatten(order="F"), shape, perm).reshape((m, n), order="F")
        C_o = cv.T @ cv
        C_g = B.site_gram(d_psi, list(dims), cut, d_lam).cpu().numpy().reshape((n, n), order="F")
        assert np.linalg.norm(C_g - C_o) <= 1e-13 * np.linalg.norm(C_o), (dims, cut)
        assert np.array_equal(C_g, C_g.T)
        # unweighted variant
        cv0 = po.permute_listing1(psi, shape, perm).reshape((m, n), order="F")
        C_g0 = B.site_gram(d_psi, list(dims), cut, None).cpu().numpy().reshape((n, n), order="F")
        assert np.linalg.norm(C_g0 - cv0.T @ cv0) <= 1e-13 * np.linalg.norm(cv0.T @ cv0)
        # ---- a10-a12: out = deabsorb(inverse-permute(cv W)) = psi contracted with W ----
        for chi_new in sorted({1, 3, dims[cut], min(2 * dims[cut] + 1, 40)}):
            W = rng.standard_normal((n, 4 * chi_new))
            out_cv = cv @ W
            shape_perm = [dims[a] for a in env] + [chi_new, 4]
            inv = [0] * (nl + 1)
            for j, pj in enumerate(perm):
                inv[pj] = j
            flat = po.permute_listing1(out_cv.flatten(order="F"), shape_perm, inv)
            shape_new = [shape_perm[inv[j]] for j in range(nl + 1)]
            want = flat.reshape(shape_new, order="F")
            for ax in range(nl):
                if ax != cut:
                    shp = [1] * (nl + 1); shp[ax] = dims[ax]
                    want = want / np.sqrt(lam[ax]).reshape(shp)
            got = B.site_apply(d_psi, list(dims), cut, _dev(torch, W.flatten(order="F")), chi_new).cpu().numpy()
            got = got.reshape(shape_new, order="F")
            assert np.linalg.norm(got - want) <= 1e-13 * np.linalg.norm(want), (dims, cut, chi_new)


def test_site_contractions_reject_bad_arguments(gpu):
    torch, B = gpu
    psi = torch.zeros(4 * 6 * 6, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PepoError) as e:
        B.site_gram(psi, [6, 6], 2)
    assert e.value.code == -1
    with pytest.raises(B.PepoError) as e:
        B.site_gram(psi, [6, 300], 0)
    assert e.value.code == -1
