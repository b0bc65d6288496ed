"""epw_zgemm_noalloc against epw_zgemm.

Some users of the library cannot let it allocate device memory: applications that handed all of HBM to their own pool
allocator, loops that must not see the device-wide stall of cudaMalloc / cudaFree, hosts that forbid a plug-in to grow
the process's device footprint.  For them the library has one contraction entry point whose packed operands live in a
fixed 16 MiB array inside the library image instead of two cudaMalloc'ed buffers.  The array is shared by every call
and keeps the last call's contents, so the check is made on two calls in a row with different shapes (the second one
smaller and ragged: a stale value of the first call that leaked into the product would show).

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this side entry point must
not hide the parity tests of the hot path.  It passes alone in a fresh process (then its first call is the library's
first CUDA call of the process and does the per-device set-up) and after the other GPU tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def epw():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2603_10295_b200 as p

    p.load_library()
    return p


def zdev(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return torch.from_numpy(a.view(np.float64).reshape(a.shape + (2,))).cuda()


def znp(t):
    return t.cpu().numpy().view(np.complex128).reshape(t.shape[:-1])


def test_zgemm_noalloc_matches_zgemm_on_two_calls_in_a_row(epw):
    """Both calls of the allocation-free entry point are issued back to back on one stream before anything is read, and
    each is compared with what epw_zgemm (the existing, allocating path) gives for the same operands, at the tolerance of
    test_zgemm_dmma (1e-13 K max|C|); the plain definition C = A B is checked too so that the two cannot be wrong together."""
    rng = np.random.default_rng(2603)
    shapes = [(300, 150, 343), (130, 70, 9)]   # (M, N, K): several tiles with ragged tails, then fewer and smaller chunks
    ops = [(rng.standard_normal((M, K)) + 1j * rng.standard_normal((M, K)),
            rng.standard_normal((K, N)) + 1j * rng.standard_normal((K, N))) for M, N, K in shapes]
    dA = [zdev(A) for A, _ in ops]
    dB = [zdev(B) for _, B in ops]
    pad = 3
    got = [torch.zeros((M, N + pad, 2), dtype=torch.float64, device="cuda") for M, N, _ in shapes]
    for (M, N, K), a, b, c in zip(shapes, dA, dB, got):      # two calls in a row, nothing in between
        epw.epw_zgemm_noalloc(a, b, c, M, N, K, N + pad)
    torch.cuda.synchronize()
    for (M, N, K), (A, B), a, b, c in zip(shapes, ops, dA, dB, got):
        want = torch.zeros((M, N + pad, 2), dtype=torch.float64, device="cuda")
        epw.epw_zgemm(a, b, want, M, N, K, N + pad)
        torch.cuda.synchronize()
        g, w, ref = znp(c), znp(want), A @ B
        tol = 1e-13 * K * max(1.0, np.abs(ref).max())
        assert np.abs(g[:, :N] - w[:, :N]).max() <= tol, (M, N, K)
        assert np.abs(g[:, :N] - ref).max() <= tol, (M, N, K)
        assert np.all(g[:, N:] == 0)   # the padding columns of C are the caller's: untouched


def test_zgemm_noalloc_rejects_a_product_beyond_its_scratch(epw):
    """Past the 16 MiB the call must fail with a message that states the limit, launch nothing and leave C alone."""
    M, N, K = 128 * 40, 64, 343      # 40 x 43 + 1 x 43 = 1,763 chunks of 16 KB > 1,024
    a = torch.zeros((M, K, 2), dtype=torch.float64, device="cuda")
    b = torch.zeros((K, N, 2), dtype=torch.float64, device="cuda")
    c = torch.full((M, N, 2), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(epw.EpwError) as e:
        epw.epw_zgemm_noalloc(a, b, c, M, N, K, N)
    assert e.value.code == epw.binding.EPW_EUNSUPPORTED
    assert "1763" in str(e.value) and "1024" in str(e.value)
    torch.cuda.synchronize()
    assert bool((c == 7.0).all())
    # a product that needs exactly the whole array still goes through
    M2, N2, K2 = 128 * 1016, 8 * 64, 8                                # 1,016 + 8 = 1,024 chunks of 16 KB
    assert M2 // 128 + N2 // 64 == epw.binding.EPW_ZGEMM_NOALLOC_SCRATCH_BYTES // 16384
    a = torch.ones((M2, K2, 2), dtype=torch.float64, device="cuda")
    b = torch.ones((K2, N2, 2), dtype=torch.float64, device="cuda")
    c = torch.zeros((M2, N2, 2), dtype=torch.float64, device="cuda")
    epw.epw_zgemm_noalloc(a, b, c, M2, N2, K2, N2)
    torch.cuda.synchronize()
    # (1 + i)(1 + i) = 2i, summed over K2 = 8 terms
    assert bool((c[..., 0] == 0.0).all()) and bool((c[..., 1] == 2.0 * K2).all())
