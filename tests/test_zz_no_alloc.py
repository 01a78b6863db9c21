"""ks_zgemm_hn_static: the allocation-free variant of the split-K product C = A^H B (include/kspw.h).  Its split-K
partial tiles live in a file-scope device array of the library (8 MiB) instead of a cudaMalloc'ed workspace.  Checked
against the existing path (ks_zgemm_hn) and the definition (numpy), on two calls in a row: the second call is smaller and
has a different split count, so anything read from the array that the call itself did not write would show.
This file sorts last on purpose (the run uses pytest -x)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MAX_ELEMS = (8 << 20) // 16        # M * N limit stated in include/kspw.h


@pytest.fixture(scope="module")
def ks():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2501_08697_b200 import kspw
    return kspw


def _t(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _pair(M, N, K, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((M, K)) + 1j * rng.standard_normal((M, K))
    B = rng.standard_normal((N, K)) + 1j * rng.standard_normal((N, K))
    return A, B


def _check(ks, M, N, K, seed):
    import torch
    A, B = _pair(M, N, K, seed)
    At, Bt = _t(A), _t(B)
    out = torch.full((N, M), complex(float("nan"), float("nan")), dtype=torch.complex128, device="cuda")
    ks.ks_zgemm_hn_static(At, Bt, out)
    got = out.cpu().numpy()
    old = ks.ks_zgemm_hn(At, Bt).cpu().numpy()                  # the existing (allocating) path
    ref = (A.conj() @ B.T).T                                     # C[m][n] = sum_k conj(A[m][k]) B[n][k]
    tol = 1e-13 * max(1, K) ** 0.5 * (np.abs(ref).max() + 1)     # the tolerance of test_zgemm_hn
    assert np.isfinite(got.view(np.float64)).all()
    assert np.abs(got - old).max() <= tol
    assert np.abs(got - ref).max() <= tol
    return out


def test_static_scratch_product_two_calls_in_a_row(ks):
    import torch
    # call 1: a Gram-matrix-like product with many splits (160 x 160 x 37 073, cfg 1's V^H W shape)
    _check(ks, 160, 160, 37073, 1)
    # call 2, straight after: smaller output, ragged tiles, fewer k-tiles -> other split count, the array still holds call 1's partials
    _check(ks, 70, 37, 4099, 2)
    # and the shapes whose partial tiles come closest to the limit / have a single split / no K at all
    _check(ks, 724, 724, 300, 3)
    _check(ks, 5, 3, 0, 4)
    _check(ks, 1, 1, 1, 5)
    # repeatable bit for bit (fixed split count and summation order, no atomics)
    A, B = _pair(96, 200, 8459, 6)
    At, Bt = _t(A), _t(B)
    o1 = torch.empty((200, 96), dtype=torch.complex128, device="cuda")
    o2 = torch.empty_like(o1)
    ks.ks_zgemm_hn_static(At, Bt, o1)
    ks.ks_zgemm_hn_static(At, Bt, o2)
    assert bool((o1 == o2).all())


def test_static_scratch_rejects_sizes_beyond_the_array(ks):
    import torch
    M, N, K = 1024, 513, 16                                      # M * N = 525 312 > 524 288
    assert M * N > MAX_ELEMS
    A = torch.zeros((M, K), dtype=torch.complex128, device="cuda")
    B = torch.zeros((N, K), dtype=torch.complex128, device="cuda")
    out = torch.zeros((N, M), dtype=torch.complex128, device="cuda")
    with pytest.raises(ks.KsError) as ei:
        ks.ks_zgemm_hn_static(A, B, out)
    assert ei.value.rc == -1 and "static scratch" in str(ei.value) and "524288" in str(ei.value)
    # exactly at the limit it runs
    M, N = 1024, 512
    out = torch.empty((N, M), dtype=torch.complex128, device="cuda")
    ks.ks_zgemm_hn_static(A, B[:N].contiguous(), out)
    assert float(out.abs().max()) == 0.0
