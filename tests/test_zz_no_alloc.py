"""pepo_gram_static: the Gram kernel with its split-K scratch in the library's built-in device array, for
callers that may not allocate device memory.  Collected last (file name) so that a failure here hides no
other test under `pytest -x`.  Checks, on two calls in a row that SHARE the array (a large plan first, then
a smaller one with a different n, so the second call finds the first one's partial sums in the scratch):
the output against the existing path pepo_gram (same kernels and plan: equal bits, asserted within the
1e-13 relative tolerance the Gram tests use) and against the definition A^T A; that no device memory is
allocated during the calls; and the rejection of a plan beyond the array."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_30985_b200 import binding
    return torch, binding


def test_gram_static_matches_gram_on_two_calls_in_a_row(gpu):
    torch, B = gpu
    assert B.static_scratch_bytes() == 8 << 20
    cases = [(256000, 40), (4099, 160)]         # BASELINE configs[2]'s narrow Gram (7.6 MB of partials), then a ragged one
    inputs, outs, wants = [], [], []
    for m, n in cases:
        A = np.random.default_rng(m + n).standard_normal((m, n))
        inputs.append(torch.from_numpy(A.flatten(order="F")).cuda())
        outs.append(torch.full((n * n,), float("nan"), dtype=torch.float64, device="cuda"))
        wants.append(A.T @ A)
    ref = [B.gram(dA, m, n).cpu().numpy() for dA, (m, n) in zip(inputs, cases)]     # existing path, own workspace
    # first use on this device: the address look-up (and, with lazy module loading, the load of the array itself)
    tiny = torch.ones(15, dtype=torch.float64, device="cuda")
    B.gram_static(tiny, 3, 5, torch.empty(25, dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for dA, (m, n), out in zip(inputs, cases, outs):                                # two calls in a row, one stream
        B.gram_static(dA, m, n, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == before                                   # nothing was allocated
    for (m, n), out, r, want in zip(cases, outs, ref, wants):
        got = out.cpu().numpy()
        assert np.linalg.norm(got - r) <= 1e-13 * np.linalg.norm(r)
        assert np.array_equal(got, r)                                               # same kernels, same plan
        g = got.reshape((n, n), order="F")
        assert np.linalg.norm(g - want) <= 1e-13 * np.linalg.norm(want)
        assert np.array_equal(g, g.T)
    # and once more in the other order: the scratch now holds the small plan's partial sums
    for idx in (1, 0):
        m, n = cases[idx]
        outs[idx].fill_(float("nan"))
        B.gram_static(inputs[idx], m, n, outs[idx])
        assert np.array_equal(outs[idx].cpu().numpy(), ref[idx])


def test_gram_static_rejects_a_plan_beyond_the_array(gpu):
    torch, B = gpu
    m, n = 256000, 160                                                               # 40 MB of partial sums
    dA = torch.zeros(m * n, dtype=torch.float64, device="cuda")
    out = torch.zeros(n * n, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PepoError) as ei:
        B.gram_static(dA, m, n, out)
    assert ei.value.code == -2 and "built-in array holds 8388608" in str(ei.value)
    with pytest.raises(B.PepoError):
        B.gram_static(dA, 0, n, out)
