"""GPU parity tests: every CUDA stage and the whole path against the CPU oracle, through the C ABI.

Run on the B200 box with `python -m pytest tests -m gpu`.  Inputs are the seeded synthetic workloads of synth/
(DESIGN.md "Input recipe"); expected values always come from oracle/.
"""
import numpy as np
import pytest

import oracle
import synth
from parity import assert_path_close, eig_close

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def epw():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2603_10295_b200 as p

    p.load_library()
    return p


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def zdev(a):
    """complex128 numpy -> float64 device tensor of interleaved (re, im)."""
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return torch.from_numpy(a.view(np.float64).reshape(a.shape + (2,))).cuda()


def znp(t):
    return t.cpu().numpy().view(np.complex128).reshape(t.shape[:-1])


rng = np.random.default_rng(7)


def crandn(*s):
    return rng.standard_normal(s) + 1j * rng.standard_normal(s)


# ---------------------------------------------------------------------------------------------------------
# stage-level parity
# ---------------------------------------------------------------------------------------------------------
def test_phase_table(epw):
    w = synth.make_config(1)
    x = np.concatenate([w.q_list[:50], w.k_list[1000:1037], [[0, 0, 0], [0.5, 0.5, 0.5], [3.25, -7.5, 11.0]]])
    wt = rng.random(w.ne) + 0.5
    P = torch.empty((len(x), w.ne, 2), dtype=torch.float64, device="cuda")
    epw.epw_phase_table(dev(x), len(x), dev(w.Re), dev(wt), w.ne, P)
    got = znp(P)
    ref = np.array([[wt[ir] * np.exp(1j * oracle.phase(xx, w.Re[ir])) for ir in range(w.ne)] for xx in x])
    assert np.abs(got - ref).max() < 2e-14


@pytest.mark.parametrize("nq", [1, 3, 8])
def test_rp_to_q_eq9(epw, nq):
    w = synth.make_config(0)
    g = w.g_full()
    q = w.q_list[[5, 17, 63, 1, 2, 3, 40, 41][:nq]] + 0.013
    Pq = torch.empty((nq, w.np_, 2), dtype=torch.float64, device="cuda")
    epw.epw_phase_table(dev(q), nq, dev(w.Rp), dev(w.w_p), w.np_, Pq)
    g1 = torch.empty((nq, w.slab_elems, 2), dtype=torch.float64, device="cuda")
    epw.epw_rp_to_q(zdev(g), w.slab_elems, w.np_, Pq, nq, g1)
    got = znp(g1)
    for i in range(nq):
        ref = oracle.rp_to_q(g, w.Rp, w.w_p, q[i]).ravel()
        assert np.abs(got[i] - ref).max() <= 1e-13 * np.abs(ref).max()


def test_rp_to_q_ragged_rows_and_many_rp(epw):
    """rows not a multiple of the CTA size, Np not a multiple of the unroll."""
    nb, nm, ne, np_ = 3, 2, 5, 37
    R = rng.integers(-4, 5, size=(np_, 3)).astype(np.int32)
    wp = rng.random(np_) + 0.5
    g = crandn(np_, nm, ne, nb, nb)
    q = rng.random((2, 3))
    Pq = torch.empty((2, np_, 2), dtype=torch.float64, device="cuda")
    epw.epw_phase_table(dev(q), 2, dev(R), dev(wp), np_, Pq)
    rows = nb * nb * ne * nm
    g1 = torch.empty((2, rows, 2), dtype=torch.float64, device="cuda")
    epw.epw_rp_to_q(zdev(g), rows, np_, Pq, 2, g1)
    for i in range(2):
        ref = oracle.rp_to_q(g, R, wp, q[i]).ravel()
        assert np.abs(znp(g1)[i] - ref).max() <= 1e-13 * np.abs(ref).max()


def test_interp_operator_Dq(epw):
    w = synth.make_config(2)
    q = w.q_list[:9]
    P = torch.empty((9, w.np_, 2), dtype=torch.float64, device="cuda")
    epw.epw_phase_table(dev(q), 9, dev(w.Rp), dev(w.w_p), w.np_, P)
    out = torch.empty((9, w.nmodes, w.nmodes, 2), dtype=torch.float64, device="cuda")
    epw.epw_interp_operator(zdev(w.D_R), w.nmodes, w.np_, P, 9, out)
    got = znp(out)
    for i in range(9):
        ref = oracle.interp_operator(w.D_R, w.Rp, w.w_p, q[i])
        assert np.abs(got[i] - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("n", [1, 2, 3, 6, 8, 9, 11, 16, 31, 32, 33, 48, 97, 192, 288])
def test_eigh_batched(epw, n):
    batch = 37 if n <= 32 else (5 if n < 100 else 3)
    A = crandn(batch, n, n)
    A = 0.5 * (A + np.conj(np.swapaxes(A, 1, 2)))
    A[1] = np.diag(np.arange(n, 0, -1)).astype(np.complex128)  # already diagonal, descending
    if n >= 4:  # exactly degenerate spectrum
        Q, _ = np.linalg.qr(crandn(n, n))
        lam = np.repeat(np.arange(n // 2 + 1), 2)[:n].astype(float)
        M = (Q * lam) @ Q.conj().T
        A[2] = 0.5 * (M + M.conj().T)
    A_cm = np.ascontiguousarray(np.swapaxes(A, 1, 2))  # column-major storage
    ev = torch.empty((batch, n), dtype=torch.float64, device="cuda")
    V = torch.empty((batch, n, n, 2), dtype=torch.float64, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    epw.epw_eigh_batched(zdev(A_cm), n * n, n, batch, ev, V, 0, status)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    ev, Vm = ev.cpu().numpy(), np.swapaxes(znp(V), 1, 2)  # Vm[b] = matrix with eigenvector columns
    for b in range(batch):
        ref_ev, _, sweeps = oracle.eigh_jacobi(A_cm[b])
        assert sweeps >= 0
        e, ok = eig_close(ev[b], ref_ev)
        assert ok, (n, b, e)
        nrm = max(np.linalg.norm(A[b]), 1e-300)
        assert np.linalg.norm(A[b] @ Vm[b] - Vm[b] * ev[b][None, :]) <= 1e-13 * nrm * n
        assert np.linalg.norm(Vm[b].conj().T @ Vm[b] - np.eye(n)) <= 1e-13 * n


@pytest.mark.parametrize("n,batch", [(2, 70), (3, 33), (5, 64), (6, 100), (7, 31), (8, 37), (8, 4099),
                                     (9, 37), (10, 64), (11, 70), (11, 2100), (12, 33), (13, 31), (14, 40), (15, 65), (16, 37)])
def test_eigh_thread_per_matrix(epw, n, batch):
    """The register-resident solvers of the per-pair H(k+q) solves (EPW_EIGH_THREAD for n <= 8, EPW_EIGH_COLS for
    9 <= n <= 16): ragged batches (not a multiple of the 32 matrices of a CTA), diagonal, zero and exactly degenerate
    inputs, every matrix against the defining invariants and a sample against the oracle's Jacobi."""
    algo = epw.EPW_EIGH_THREAD if n <= 8 else epw.EPW_EIGH_COLS
    A = crandn(batch, n, n)
    A = 0.5 * (A + np.conj(np.swapaxes(A, 1, 2)))
    A[1] = np.diag(np.arange(n, 0, -1)).astype(np.complex128)
    if n >= 4:
        Q, _ = np.linalg.qr(crandn(n, n))
        lam = np.repeat(np.arange(n // 2 + 1), 2)[:n].astype(float)
        M = (Q * lam) @ Q.conj().T
        A[2] = 0.5 * (M + M.conj().T)
    A[3] = 0.0  # zero matrix
    A_cm = np.ascontiguousarray(np.swapaxes(A, 1, 2))
    ev = torch.empty((batch, n), dtype=torch.float64, device="cuda")
    V = torch.empty((batch, n, n, 2), dtype=torch.float64, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    epw.epw_eigh_batched_algo(zdev(A_cm), n * n, n, batch, ev, V, 0, status, algo)
    torch.cuda.synchronize()
    assert int(status.item()) == 0
    ev, Vm = ev.cpu().numpy(), np.swapaxes(znp(V), 1, 2)
    for b in range(batch):
        nrm = max(np.linalg.norm(A[b]), 1e-300)
        assert np.all(np.diff(ev[b]) >= 0)
        assert np.linalg.norm(A[b] @ Vm[b] - Vm[b] * ev[b][None, :]) <= 1e-13 * nrm * n
        assert np.linalg.norm(Vm[b].conj().T @ Vm[b] - np.eye(n)) <= 1e-13 * n
    assert np.all(ev[3] == 0.0)
    for b in [0, 1, 2, 4, 5, 6, 7, batch // 2, batch - 1]:
        ref_ev, _, _ = oracle.eigh_jacobi(A_cm[b])
        e, ok = eig_close(ev[b], ref_ev)
        assert ok, (n, b, e)
    bad_n, bad_algo = (9, epw.EPW_EIGH_THREAD) if n <= 8 else (8, epw.EPW_EIGH_COLS)
    with pytest.raises(epw.EpwError):
        epw.epw_eigh_batched_algo(zdev(A_cm), n * n, bad_n, 1, torch.empty((1, 16), dtype=torch.float64, device="cuda"),
                                  torch.empty((1, 16, 16, 2), dtype=torch.float64, device="cuda"), 0, status, bad_algo)


@pytest.mark.parametrize("n,batch", [(192, 150), (40, 300), (288, 9)])
def test_eigh_cluster_many_matrices(epw, n, batch):
    """The cluster eigensolver in its throughput configuration (more matrices than clusters: smallest cluster that holds
    the matrix, several matrices per cluster): a few matrices against the oracle's Jacobi, all of them against the
    defining invariants (residual, unitarity, ascending order)."""
    A = crandn(batch, n, n)
    A = 0.5 * (A + np.conj(np.swapaxes(A, 1, 2)))
    A_cm = np.ascontiguousarray(np.swapaxes(A, 1, 2))
    ev = torch.empty((batch, n), dtype=torch.float64, device="cuda")
    V = torch.empty((batch, n, n, 2), dtype=torch.float64, device="cuda")
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    dA = zdev(A_cm)
    epw.epw_eigh_batched(dA, n * n, n, batch, ev, V, 0, status)
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    epw.epw_eigh_batched(dA, n * n, n, batch, ev, V, 0, status)
    t1.record()
    torch.cuda.synchronize()
    print(f"eigh n={n} batch={batch}: {t0.elapsed_time(t1):.2f} ms")
    assert int(status.item()) == 0
    ev, Vm = ev.cpu().numpy(), np.swapaxes(znp(V), 1, 2)
    for b in range(batch):
        nrm = np.linalg.norm(A[b])
        assert np.all(np.diff(ev[b]) >= 0)
        assert np.linalg.norm(A[b] @ Vm[b] - Vm[b] * ev[b][None, :]) <= 1e-13 * nrm * n
        assert np.linalg.norm(Vm[b].conj().T @ Vm[b] - np.eye(n)) <= 1e-13 * n
    for b in (0, batch // 2, batch - 1):
        ref_ev, _, _ = oracle.eigh_jacobi(A_cm[b])
        e, ok = eig_close(ev[b], ref_ev)
        assert ok, (n, b, e)


def test_eigh_strided_input_sqrt_mode_and_hermitian_part(epw):
    """Matrices embedded in wider rows (as the H(k+q) block of the contraction output), omega = sqrt(lambda),
    and only the Hermitian part of a slightly non-Hermitian input is used."""
    n, batch, stride = 6, 11, 100
    A = crandn(batch, n, n)
    A = A @ np.conj(np.swapaxes(A, 1, 2)) + 0.1 * np.eye(n)  # positive definite
    noise = 1e-3 * crandn(batch, n, n)
    buf = np.zeros((batch, stride), dtype=np.complex128)
    buf[:, 7:7 + n * n] = np.swapaxes(A + noise - np.conj(np.swapaxes(noise, 1, 2)), 1, 2).reshape(batch, -1)
    d = zdev(buf)
    om = torch.empty((batch, n), dtype=torch.float64, device="cuda")
    V = torch.empty((batch, n, n, 2), dtype=torch.float64, device="cuda")
    epw.load_library().epw_eigh_batched(d.data_ptr() + 7 * 16, stride, n, batch, om.data_ptr(), V.data_ptr(), 1, None,
                                        torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    for b in range(batch):
        ref, _, _ = oracle.eigh_jacobi(np.ascontiguousarray(A[b].T))
        e, ok = eig_close(om[b].cpu().numpy(), oracle.omega_from_lambda(ref))
        assert ok, e


@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (130, 70, 9), (300, 150, 37), (128, 64, 8), (257, 449, 343), (1000, 7, 5)])
def test_zgemm_dmma(epw, M, N, K):
    """The DMMA contraction kernel against the plain definition C = A B (several tiles + ragged tails)."""
    A, B = crandn(M, K), crandn(K, N)
    C = torch.zeros((M, N + 3, 2), dtype=torch.float64, device="cuda")
    epw.epw_zgemm(zdev(A), zdev(B), C, M, N, K, N + 3)
    got = znp(C)
    ref = A @ B
    assert np.abs(got[:, :N] - ref).max() <= 1e-13 * K * max(1.0, np.abs(ref).max())
    assert np.all(got[:, N:] == 0)  # padding columns untouched


def test_zgemm_matches_oracle_re_to_k(epw):
    """S2 as the paper defines it: sum_Re g(Re,q) e^{ik.Re} for a batch of k (oracle.re_to_k per k)."""
    w = synth.make_custom("t", 3, 4, (2, 1, 1), 1.0, 0.1, 1.0, (5, 3, 2), ("random", 1, 3), seed=3)
    g1 = oracle.rp_to_q(w.g_full(), w.Rp, w.w_p, w.q_list[0])  # [nm][ne][nb][nb]
    nk, nbb = w.nk, 9
    P = torch.empty((nk, w.ne, 2), dtype=torch.float64, device="cuda")
    epw.epw_phase_table(dev(w.k_list), nk, dev(w.Re), dev(w.w_e), w.ne, P)
    B = np.ascontiguousarray(np.moveaxis(g1.reshape(w.nmodes, w.ne, nbb), 1, 0).reshape(w.ne, -1))  # [ie][ka*nbb+el]
    C = torch.empty((nk, w.nmodes * nbb, 2), dtype=torch.float64, device="cuda")
    epw.epw_zgemm(P, zdev(B), C, nk, w.nmodes * nbb, w.ne, w.nmodes * nbb)
    got = znp(C)
    for ik in range(nk):
        ref = oracle.re_to_k(g1, w.Re, w.w_e, w.k_list[ik]).ravel()
        assert np.abs(got[ik] - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("nb,nm,nk", [(8, 6, 19), (11, 9, 19), (3, 2, 19), (1, 1, 19), (16, 3, 19), (5, 7, 6), (7, 3, 33),
                                      (13, 20, 9), (16, 48, 5), (8, 6, 9509), (11, 9, 4801)])
def test_rotate_g2(epw, nb, nm, nk):
    """S4b on the FP64 tensor path: every Nb tile shape (K and column padding, ragged row tiles), 1 / 2 / 4 warps per
    pair (staging-buffer size), more pairs than one pass of the grid, with and without the k+q gather."""
    gt = crandn(nk, nm, nb, nb)
    nu_ = min(nk, 64)  # distinct unitaries (QR on the host is slow); pairs reuse them cyclically
    Ub = np.stack([np.linalg.qr(crandn(nb, nb))[0].T for _ in range(nu_)])  # column-major storage
    Uk = np.ascontiguousarray(Ub[np.arange(nk) % nu_])
    Ukq = np.ascontiguousarray(Ub[(np.arange(nk) * 7 + 3) % nu_])
    idx = rng.permutation(nk).astype(np.int32)
    g2 = torch.empty((nk, nm, nb, nb), dtype=torch.float64, device="cuda")
    sample = range(nk) if nk <= 40 else sorted(set([0, 1, nk // 2, nk - 2, nk - 1]) | set(rng.integers(0, nk, 24).tolist()))
    for kq_idx in (None, idx):
        g2.fill_(-1.0)
        epw.epw_rotate_g2(zdev(gt), nm * nb * nb, zdev(Uk), zdev(Ukq), None if kq_idx is None else dev(kq_idx), nb, nm,
                          nk, g2)
        got = g2.cpu().numpy()
        assert got.min() >= 0.0  # every element written
        for ik in sample:
            u = Ukq[ik] if kq_idx is None else Ukq[kq_idx[ik]]
            ref = np.abs(oracle.band_rotate(gt[ik], u, Uk[ik])) ** 2
            assert np.abs(got[ik] - ref).max() <= 1e-12 * ref.max()


@pytest.mark.parametrize("case", ["plain", "blocked", "blocked_ragged", "colmajor_c", "batched_gather_conj_abs2"])
def test_zgemm_strided(epw, case):
    """The in-place-A DMMA contraction of the large-Nb path against the plain definition, in every addressing mode the
    path uses: blocked rows (a_rb < tile), several row blocks per tile, ragged M / N / K, transposed store, batches with
    gathered conjugated B and the |.|^2 epilogue."""
    if case == "plain":            # S4a-like: A[row][r] at r*M + row ; C row-major
        M, N, K, batch = 300, 70, 21, 1
        A = crandn(K, M); B = crandn(K, N)
        ref = np.einsum("rm,rn->mn", A, B)
        C = torch.zeros((M, N, 2), dtype=torch.float64, device="cuda")
        epw.epw_zgemm_strided(zdev(A), M, 0, M, 0, zdev(B), N, 1, 0, 0, None, 1, C, M, 0, N, 1, 0, 0, M, N, K, 1)
        got = znp(C)
    elif case in ("blocked", "blocked_ragged"):   # S4b-like: row = (nu, x), A at nu*nbb + r*nb + x
        nb, nm = (192, 3) if case == "blocked" else (13, 37)
        M, N, K = nm * nb, nb, nb
        G = crandn(nm, nb, nb)      # [nu][r][x]
        U = crandn(nb, nb)          # column-major storage: U[n][r] <-> B[r][n]
        ref = np.einsum("vrx,nr->vxn", G, U).reshape(M, N)
        C = torch.zeros((M, N, 2), dtype=torch.float64, device="cuda")
        epw.epw_zgemm_strided(zdev(G), nb, nb * nb, nb, 0, zdev(U), 1, nb, 0, 0, None, 1, C, M, 0, N, 1, 0, 0, M, N, K, 1)
        got = znp(C)
    elif case == "colmajor_c":     # S2-like: C[c][k] stored at k*M + c, N not a multiple of the tile
        M, N, K = 1000, 70, 17
        A = crandn(K, M); P = crandn(N, K)     # B[r][n] = P[n][r]
        ref = np.einsum("rm,nr->mn", A, P)
        C = torch.zeros((N, M, 2), dtype=torch.float64, device="cuda")
        epw.epw_zgemm_strided(zdev(A), M, 0, M, 0, zdev(P), 1, K, 0, 0, None, 1, C, M, 0, 1, M, 0, 0, M, N, K, 1)
        got = znp(C).T
    else:
        nb, nm, batch = 20, 9, 5
        M, N, K = nm * nb, nb, nb
        T = crandn(batch, nm, nb, nb)   # [b][nu][r][x]
        U = crandn(7, nb, nb)           # 7 matrices, column-major: U[i][m][r]
        idx = np.array([6, 0, 3, 3, 1], dtype=np.int32)
        ref = np.abs(np.einsum("bvrx,bmr->bvxm", T, U[idx].conj())) ** 2
        C = torch.zeros((batch, M, N), dtype=torch.float64, device="cuda")
        epw.epw_zgemm_strided(zdev(T), nb, nb * nb, nb, nm * nb * nb, zdev(U), 1, nb, nb * nb, 1, dev(idx), 7, C, M, 0, N,
                              1, M * N, 1, M, N, K, batch)
        got = C.cpu().numpy().reshape(ref.shape)
    torch.cuda.synchronize()
    assert np.abs(got.reshape(ref.shape) - ref).max() <= 1e-13 * K * max(1.0, np.abs(ref).max())


def test_rotate_g2_large(epw):
    """S4b beyond the shared-memory kernel (Nb = 48): two in-place DMMA contractions, against oracle.band_rotate."""
    nb, nm, nk = 48, 7, 5
    gt = crandn(nk, nm, nb, nb)
    Uk = np.stack([np.linalg.qr(crandn(nb, nb))[0].T for _ in range(nk)])
    Ukq = np.stack([np.linalg.qr(crandn(nb, nb))[0].T for _ in range(nk)])
    idx = rng.permutation(nk).astype(np.int32)
    g2 = torch.empty((nk, nm, nb, nb), dtype=torch.float64, device="cuda")
    for kq_idx in (None, idx):
        epw.epw_rotate_g2(zdev(gt), nm * nb * nb, zdev(Uk), zdev(Ukq), None if kq_idx is None else dev(kq_idx), nb, nm,
                          nk, g2)
        got = g2.cpu().numpy()
        for ik in range(nk):
            u = Ukq[ik] if kq_idx is None else Ukq[kq_idx[ik]]
            ref = np.abs(oracle.band_rotate(gt[ik], u, Uk[ik])) ** 2
            assert np.abs(got[ik] - ref).max() <= 1e-12 * ref.max()


@pytest.mark.parametrize("nb,nmodes,L,cnt,slab,nbatch,extra", [
    (8, 6, 7, 40, 5, 1, 0),      # configs[1]: K = 14 real exactly 4 k-steps, ten quads
    (8, 2, 9, 13, 3, 2, 64),     # L = 9 (configs[3]): five of eight k-steps, ragged last quad, two blocks, padded rows
    (11, 3, 13, 10, 2, 3, 0),    # Nb = 11 (configs[2]): 121 columns per group, ragged column tile
    (8, 3, 17, 9, 1, 1, 0),      # L = 17 (the ribbon's lattice-vector list): nine k-steps
    (3, 5, 2, 5, 4, 2, 9),       # tiny shapes
])
def test_axis_pass_dmma(epw, nb, nmodes, L, cnt, slab, nbatch, extra):
    """One axis of the factorised Re -> k sum as the DMMA product (pass-only variant of grid_fused_kernel, batched) against
    the plain definition out[b][j][c][col] = sum_n P[n][j] T[b][n][c][col]."""
    ncols = nb * nb * nmodes
    stride = ncols + extra
    T = crandn(nbatch, L, slab, ncols)
    P = crandn(L, cnt)
    out = torch.zeros((nbatch, cnt, slab, stride, 2), dtype=torch.float64, device="cuda")
    epw.epw_axis_pass_dmma(zdev(T), slab, ncols, L, zdev(P), cnt, nb, out, stride, nbatch, L * slab * ncols,
                           cnt * slab * stride)
    torch.cuda.synchronize()
    got = znp(out)
    ref = np.einsum("nj,bncx->bjcx", P, T)
    assert np.abs(got[..., :ncols] - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.abs(got[..., ncols:]).max() == 0.0 if extra else True   # nothing written beyond the columns of a row


# ---------------------------------------------------------------------------------------------------------
# whole path
# ---------------------------------------------------------------------------------------------------------
def run_gpu(epw, w, k_list, q_list, kq_map=None, q_batch=0, host_api=False, path=0, workspace_bytes=0, grid=None,
            shift=None, flags=0):
    """grid = (N1, N2, N3): call the uniform-grid entry point (k_list is then only used for its length);
    flags = EPW_FLAG_GRID_UNFUSED keeps the last axis pass and the rotation as two kernels."""
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, q_batch=q_batch, path=path, workspace_bytes=workspace_bytes,
                      flags=flags)
    try:
        h.set_operators_from_host(w)
        if host_api:
            nk, nq = len(k_list), len(q_list)
            eps_k = np.empty((nk, w.nbnd))
            eps_kq = np.empty((nq, nk, w.nbnd))
            om = np.empty((nq, w.nmodes))
            g2 = np.empty((nq, nk, w.nmodes, w.nbnd, w.nbnd))
            if grid is not None:
                epw.epw_interp_interpolate_grid_host(h.h, grid, shift, np.ascontiguousarray(q_list), nq, kq_map, eps_k,
                                                     eps_kq, om, g2)
            else:
                epw.epw_interp_interpolate_host(h.h, np.ascontiguousarray(k_list), nk, np.ascontiguousarray(q_list), nq,
                                                kq_map, eps_k, eps_kq, om, g2)
            return eps_k, eps_kq, om, g2
        if grid is not None:
            out = h.interpolate_grid(grid, dev(q_list), k_shift=shift, kq_map=None if kq_map is None else dev(kq_map))
            fused = flags == 2 or (flags == 0 and w.nbnd <= 8)
            want = "list" if path == 2 or w.nbnd > 16 else ("grid-fused" if fused else "grid")
            assert epw.epw_interp_last_plan(h.h)["k_mode"] == want
        else:
            out = h.interpolate(dev(k_list), dev(q_list), None if kq_map is None else dev(kq_map))
        epw.epw_interp_sync(h.h)
        return [None if t is None else t.cpu().numpy() for t in out]
    finally:
        h.close()


def test_config0_full_both_kq_modes(epw):
    """BASELINE.json configs[0], all 4,096 pairs: grid-folded k+q (kq_map) and per-pair H(k+q) eigensolves."""
    w = synth.make_config(0)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    worst = assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, w.kq_map), ref)
    worst2 = assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, None), ref)
    print(f"config 0 worst |g|^2 error: {worst:.3f} / {worst2:.3f} of tolerance")


def test_config0_host_api_and_q_batches(epw):
    w = synth.make_config(0)
    ql = w.q_list[:7] + [0.01, 0.02, 0.03]
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, ql)
    for qb in (1, 3, 8):
        assert_path_close(run_gpu(epw, w, w.k_list, ql, None, q_batch=qb), ref)
    assert_path_close(run_gpu(epw, w, w.k_list, ql, None, host_api=True), ref)


@pytest.mark.parametrize("shape", ["si", "mos2", "odd"])
def test_reduced_shapes(epw, shape):
    """Reduced-size versions of configs 1-3 (same generators, fewer lattice vectors and k): several M tiles,
    ragged tails, odd Nb/Nm (11, 9), 2-D lattices."""
    if shape == "si":
        w = synth.make_custom("si-r", 8, 6, (2, 2, 2), 1.5, 0.1, 1.5, (7, 6, 5), ("random", 3, 3), seed=11)
    elif shape == "mos2":
        w = synth.make_custom("mos2-r", 11, 9, (3, 3, 0), 2.0, 0.1, 2.0, (15, 13, 1), ("random", 3, 2), seed=12)
    else:
        w = synth.make_custom("odd", 5, 3, (1, 2, 0), 1.0, 0.1, 1.0, (9, 1, 17), ("random", 2, 3), seed=13)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list), ref)


# ---- uniform-grid entry point (factorised S2, csrc/re_to_k_grid.cu) ----------------------------------------
def test_grid_config0_both_kq_modes_and_host_api(epw):
    """configs[0] through epw_interp_interpolate_grid: all 4,096 pairs with kq_map, per-pair H(k+q), host buffers."""
    w = synth.make_config(0)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    for flags in (0, 2):
        assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, w.kq_map, grid=w.k_grid, flags=flags), ref)
        assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, None, grid=w.k_grid, flags=flags), ref)
    ql = w.q_list[:5] + [0.01, 0.02, 0.03]
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, ql)
    assert_path_close(run_gpu(epw, w, w.k_list, ql, None, grid=w.k_grid, host_api=True, q_batch=3), ref)


@pytest.mark.parametrize("flags", [0, 1, 2])
@pytest.mark.parametrize("shape", ["si", "mos2", "odd", "chunks", "large-forced", "modes-split"])
def test_grid_reduced_shapes(epw, shape, flags):
    """Reduced configs 1-3 through the grid entry point: ragged tiles in every axis pass, 2-D and skewed lattices,
    several i1-plane chunks (workspace cap), and the large-Nb family (which expands the grid to a list)."""
    ws, path = 0, 0
    if shape == "si":
        w = synth.make_custom("si-r", 8, 6, (2, 2, 2), 1.5, 0.1, 1.5, (7, 6, 5), ("random", 3, 3), seed=11)
    elif shape == "mos2":
        w = synth.make_custom("mos2-r", 11, 9, (3, 3, 0), 2.0, 0.1, 2.0, (15, 13, 1), ("random", 3, 2), seed=12)
    elif shape == "odd":
        w = synth.make_custom("odd", 5, 3, (1, 2, 0), 1.0, 0.1, 1.0, (9, 1, 17), ("random", 2, 3), seed=13)
    elif shape == "chunks":
        w = synth.make_custom("chunks", 4, 3, (1, 1, 1), 1.0, 0.1, 1.0, (11, 3, 4), ("random", 2, 3), seed=14)
        # three i1 planes (12 k each) of per-k workspace per chunk -> 4 chunks, ragged last
        ws = (16 * 12 * ((16 * 3 if flags != 2 else 0) + 16 + 16 + 4) + 16) * 3 + 100
    elif shape == "modes-split":
        # Nb = 13, Nm = 12, L1 = 7: the fused kernel cannot hold all modes of a cell in shared memory -> mode groups
        w = synth.make_custom("modes", 13, 12, (3, 1, 0), 1.0, 0.1, 1.0, (10, 3, 1), ("random", 2, 2), seed=15)
    else:
        w = synth.make_custom("mos2-l", 11, 9, (2, 2, 0), 2.0, 0.1, 2.0, (13, 11, 1), ("random", 2, 2), seed=23)
        path = 2
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, grid=w.k_grid, workspace_bytes=ws, path=path, flags=flags), ref)


def test_grid_shifted_and_sparse_lattice_list(epw):
    """A shifted grid k = (i + s)/N and an Re list that is NOT a full box (vectors removed, order shuffled, non-unit
    Wigner-Seitz weights): the box scatter must leave zeros where the list has no vector."""
    w = synth.make_custom("sparse", 4, 3, (2, 1, 1), 1.0, 0.1, 1.0, (6, 5, 4), ("random", 2, 3), seed=31)
    rng = np.random.default_rng(3)
    keep = rng.permutation(w.ne)[: w.ne - 11]
    g = np.ascontiguousarray(w.g_full()[:, :, keep])

    class Sub:
        nbnd, nmodes, ne, np_ = w.nbnd, w.nmodes, len(keep), w.np_
        H_R, D_R = np.ascontiguousarray(w.H_R[keep]), w.D_R
        Re, Rp, w_p = np.ascontiguousarray(w.Re[keep]), w.Rp, w.w_p
        w_e = rng.uniform(0.3, 1.0, size=len(keep))
        slab_elems = w.nbnd * w.nbnd * len(keep) * w.nmodes

        @staticmethod
        def g_slabs(ip, cnt):
            return np.ascontiguousarray(g[ip:ip + cnt])

    shift = (0.5, 0.25, 0.125)
    k_list = (np.stack(np.meshgrid(*[np.arange(n) for n in w.k_grid], indexing="ij"), -1).reshape(-1, 3)
              + np.array(shift)) / np.array(w.k_grid)
    ref = oracle.interpolate(Sub.H_R, Sub.D_R, g, Sub.Re, Sub.w_e, Sub.Rp, Sub.w_p, k_list, w.q_list)
    assert_path_close(run_gpu(epw, Sub, k_list, w.q_list, grid=w.k_grid, shift=shift), ref)
    assert_path_close(run_gpu(epw, Sub, k_list, w.q_list, grid=w.k_grid, shift=shift, flags=2), ref)
    # and the same k-points as a list through the dense contraction
    assert_path_close(run_gpu(epw, Sub, k_list, w.q_list), ref)


def test_large_path_forced_on_config0(epw):
    """The large-Nb kernels (S4a, S2, S4b as in-place DMMA contractions) on configs[0], where the small-Nb path and the
    oracle are both available: grid-folded k+q and per-pair H(k+q)."""
    w = synth.make_config(0)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list[:9])
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list[:9], w.kq_map[:9], path=2), ref)
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list[:9], None, path=2, q_batch=3), ref)


@pytest.mark.parametrize("shape", ["zsnr-r", "zsnr-r-offgrid", "mos2-r-large"])
def test_large_path_reduced_shapes(epw, shape):
    """Reduced configs[4]-like ribbon (1-D lattice, Nb > 16 so the large path is chosen, Nb > 32 so the CTA-per-matrix
    eigensolver runs, ragged tiles everywhere), with k+q on the grid and off it; and an odd 2-D shape forced large."""
    if shape == "zsnr-r":
        w = synth.make_custom("zsnr-r", 36, 15, (3, 0, 0), 1.0, 0.05, 2.0, (70, 1, 1), ("grid", (10, 1, 1)), seed=21)
        kq, path = w.kq_map, 0
    elif shape == "zsnr-r-offgrid":
        w = synth.make_custom("zsnr-o", 20, 12, (2, 0, 0), 1.0, 0.05, 2.0, (9, 1, 1), ("random", 3, 1), seed=22)
        kq, path = None, 0
    else:
        w = synth.make_custom("mos2-l", 11, 9, (2, 2, 0), 2.0, 0.1, 2.0, (13, 11, 1), ("random", 2, 2), seed=23)
        kq, path = None, 2
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, kq, path=path), ref)


def test_large_path_k_chunks(epw):
    """A workspace cap that forces several 64-k chunks (and a ragged last one) through S2 / S4b of the large path."""
    w = synth.make_custom("zsnr-c", 18, 6, (2, 0, 0), 1.0, 0.05, 2.0, (150, 1, 1), ("grid", (3, 1, 1)), seed=24)
    E = w.nbnd * w.nbnd * w.nmodes
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    assert_path_close(run_gpu(epw, w, w.k_list, w.q_list, w.kq_map, workspace_bytes=2 * 16 * E * 64 + 1000), ref)


def test_debug_intermediates_config0(epw):
    """g(Re,q), H(k), e_q and g~ of the last q against the oracle's stage functions."""
    w = synth.make_config(0)
    g = w.g_full()
    q = w.q_list[9:10] + 0.004
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
    try:
        h.set_operators_from_host(w)
        h.interpolate(dev(w.k_list), dev(q))
        g1 = np.empty((w.nmodes, w.ne, w.nbnd, w.nbnd), dtype=np.complex128)
        epw.epw_interp_debug_get(h.h, epw.EPW_DBG_G_REQ, g1)
        ref1 = oracle.rp_to_q(g, w.Rp, w.w_p, q[0])
        assert np.abs(g1 - ref1).max() <= 1e-13 * np.abs(ref1).max()
        Hk = np.empty((w.nk, w.nbnd, w.nbnd), dtype=np.complex128)
        epw.epw_interp_debug_get(h.h, epw.EPW_DBG_H_K, Hk)
        for ik in (0, 13, 63):
            refH = oracle.interp_operator(w.H_R, w.Re, w.w_e, w.k_list[ik])
            assert np.abs(Hk[ik] - refH).max() <= 1e-13 * np.abs(refH).max()
        gt = np.empty((w.nk, w.nmodes, w.nbnd, w.nbnd), dtype=np.complex128)
        epw.epw_interp_debug_get(h.h, epw.EPW_DBG_G_TILDE, gt)
        e_ref, om_ref = oracle.phonon(w.D_R, w.Rp, w.w_p, q[0])
        # gauge-free check of the mode-rotated g~: sum_nu 2 omega_nu |g~_nu|^2 = sum_ka |g~_ka|^2 per (m',n')
        for ik in (0, 31):
            raw = oracle.re_to_k(ref1, w.Re, w.w_e, w.k_list[ik])
            lhs = (2 * om_ref[:, None, None] * np.abs(gt[ik]) ** 2).sum(axis=0)
            rhs = (np.abs(raw) ** 2).sum(axis=0)
            assert np.abs(lhs - rhs).max() <= 1e-11 * rhs.max()
    finally:
        h.close()


def test_errors_are_reported(epw):
    with pytest.raises(epw.EpwError):
        epw.epw_interp_create(0, 6, 27, 27)
    h = epw.EpwInterp(2, 3, 5, 5)
    try:
        k = torch.zeros((4, 3), dtype=torch.float64, device="cuda")
        with pytest.raises(epw.EpwError) as ei:
            h.interpolate(k, k)
        assert "operators not set" in str(ei.value)
    finally:
        h.close()


# ---------------------------------------------------------------------------------------------------------
# full-size configurations, in the launch configuration bench.py times: sampled pairs against the oracle
# ---------------------------------------------------------------------------------------------------------
def check_sampled_pairs(epw, w, q_idx, k_idx, q_batch=0, grid=False, flags=0):
    """Run the library on ALL k of workload w and the q-points q_idx (one interpolate call, as bench.py does), then
    compare eps_k, omega_q, eps_kq and |g|^2 on the sampled (q, k) pairs with the oracle computed pair by pair."""
    g = w.g_full()
    ql = np.ascontiguousarray(w.q_list[q_idx])
    kq_map = None if w.kq_map is None else np.ascontiguousarray(w.kq_map[q_idx])
    eps_k, eps_kq, om, g2 = run_gpu(epw, w, w.k_list, ql, kq_map, q_batch=q_batch, grid=w.k_grid if grid else None,
                                    flags=flags)
    worst = 0.0
    for jq in range(len(q_idx)):
        e_ref, om_ref = oracle.phonon(w.D_R, w.Rp, w.w_p, ql[jq])
        err, ok = eig_close(om[jq], om_ref)
        assert ok, f"omega mismatch at q {q_idx[jq]}: {err:.3e}"
        g1 = oracle.rp_to_q(g, w.Rp, w.w_p, ql[jq])
        for ik in k_idx:
            r_g2, r_ek, r_ekq = oracle.pair(g1, w.H_R, w.Re, w.w_e, e_ref, om_ref, w.k_list[ik], ql[jq])
            err, ok = eig_close(eps_k[ik], r_ek)
            assert ok, f"eps_k mismatch at k {ik}: {err:.3e}"
            err, ok = eig_close(eps_kq[jq, ik], r_ekq)
            assert ok, f"eps_kq mismatch at (q {q_idx[jq]}, k {ik}): {err:.3e}"
            from parity import g2_pair_close

            wst, ok = g2_pair_close(g2[jq, ik], r_g2, r_ekq, r_ek, om_ref)
            assert ok, f"|g|^2 mismatch at (q {q_idx[jq]}, k {ik}): {wst:.3f} x tolerance"
            worst = max(worst, wst)
    return worst


def sample_k(nk, n=24, seed=5):
    """first / last rows, the rows around the 128-row tile edges and a few random ones"""
    r = np.random.default_rng(seed)
    fixed = [0, 1, 127, 128, nk // 2, nk - 129, nk - 128, nk - 1]
    return sorted(set(int(x) for x in fixed if 0 <= x < nk) | set(int(x) for x in r.integers(0, nk, size=n)))


def test_config1_full_size_sampled(epw):
    """BASELINE.json configs[1] on the k-list route: all 64,000 k, 8 q per call (one S1 batch of 8, the default q_batch;
    the grid route at the bench's 96 q per call is test_grid_full_size_sampled)."""
    w = synth.make_config(1)
    q_idx = [0, 1, 2, 3, 500, 501, 998, 999]
    worst = check_sampled_pairs(epw, w, q_idx, sample_k(w.nk))
    print(f"config 1 full size: worst |g|^2 deviation {worst:.3f} x tolerance")


# q-points per interpolate call of the default bench.py step of each config (bench.NQ_STEP)
BENCH_NQ_STEP = {1: 96, 2: 32, 3: 13}


@pytest.mark.parametrize("cfg,flags", [(1, 0), (1, 1), (2, 0), (2, 2), (3, 0)])
def test_grid_full_size_sampled(epw, cfg, flags):
    """configs[1..3] at full size through the uniform-grid entry point in the launch configuration bench.py times: all k,
    the bench's number of q-points per call (96 / 32 / 13), default kernel choice (flags 0: one-kernel form for Nb = 8,
    two-kernel form for Nb = 11) and the other form.  The outputs stay on the device (19 GB for configs[1]); sampled
    (q, k) pairs -- the S1 batch edges, first / last q, i1-plane and chunk edges in k -- are compared with the oracle."""
    from parity import g2_pair_close

    w = synth.make_config(cfg)
    nq = BENCH_NQ_STEP[cfg]
    rng_q = np.random.default_rng(100 + cfg)
    q_idx = np.sort(rng_q.choice(w.nq, size=nq, replace=False))
    ql = np.ascontiguousarray(w.q_list[q_idx])
    check_q = sorted({0, 7, 8, nq // 2, nq - 1}) if cfg == 1 else [0, nq - 1]
    k_idx = sample_k(w.nk, 12 if cfg != 1 else 6)
    slab = w.k_grid[1] * w.k_grid[2]
    k_idx = sorted(set(k_idx) | {slab - 1, slab, 63 * slab + 5 if 63 * slab + 5 < w.nk else 0,
                                 64 * slab if 64 * slab < w.nk else 0})  # i1-plane and chunk edges
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, flags=flags)
    try:
        h.set_operators_from_host(w)
        eps_k, eps_kq, om, g2 = h.interpolate_grid(w.k_grid, dev(ql))
        epw.epw_interp_sync(h.h)
        want = "grid-fused" if (flags == 2 or (flags == 0 and w.nbnd <= 8)) else "grid"
        assert epw.epw_interp_last_plan(h.h)["k_mode"] == want
        kt = torch.tensor(k_idx, device="cuda")
        eps_k_s = eps_k[kt].cpu().numpy()
        om = om.cpu().numpy()
        g = w.g_full()
        worst = 0.0
        for jq in check_q:
            eps_kq_s = eps_kq[jq][kt].cpu().numpy()
            g2_s = g2[jq][kt].cpu().numpy()
            e_ref, om_ref = oracle.phonon(w.D_R, w.Rp, w.w_p, ql[jq])
            err, ok = eig_close(om[jq], om_ref)
            assert ok, f"omega mismatch at q {jq}: {err:.3e}"
            g1 = oracle.rp_to_q(g, w.Rp, w.w_p, ql[jq])
            for i, ik in enumerate(k_idx):
                r_g2, r_ek, r_ekq = oracle.pair(g1, w.H_R, w.Re, w.w_e, e_ref, om_ref, w.k_list[ik], ql[jq])
                err, ok = eig_close(eps_k_s[i], r_ek)
                assert ok, f"eps_k mismatch at k {ik}: {err:.3e}"
                err, ok = eig_close(eps_kq_s[i], r_ekq)
                assert ok, f"eps_kq mismatch at (q {jq}, k {ik}): {err:.3e}"
                wst, ok = g2_pair_close(g2_s[i], r_g2, r_ekq, r_ek, om_ref)
                assert ok, f"|g|^2 mismatch at (q {jq}, k {ik}): {wst:.3f} x tolerance"
                worst = max(worst, wst)
    finally:
        h.close()
    print(f"config {cfg} full size (grid, flags {flags}, {nq} q per call): worst |g|^2 deviation {worst:.3f} x tolerance")


def test_config2_full_size_sampled(epw):
    """BASELINE.json configs[2] (MoS2-like, Nb=11, Nm=9, 2-D): all 14,400 k, 3 q."""
    w = synth.make_config(2)
    worst = check_sampled_pairs(epw, w, [0, 1000, 1999], sample_k(w.nk, 16))
    print(f"config 2 full size: worst |g|^2 deviation {worst:.3f} x tolerance")


def test_config3_full_size_sampled(epw):
    """BASELINE.json configs[3] (10^6 k streamed through a reused g~ buffer, Ne=Np=729): 2 q, sampled k."""
    w = synth.make_config(3)
    worst = check_sampled_pairs(epw, w, [0, 255], sample_k(w.nk, 16))
    print(f"config 3 full size: worst |g|^2 deviation {worst:.3f} x tolerance")


def test_config4_full_size_sampled(epw):
    """BASELINE.json configs[4] (stanene-nanoribbon-like: Nb=192, Nm=288, Ne=Np=17, g(Re,Rp) = 49 GB streamed to the GPU
    in Rp slabs) in the launch configuration bench.py times: the 200-point grid through epw_interp_interpolate_grid,
    TWO q of the grid per call (bench.NQ_STEP[4]; k+q folded through kq_map, 34 GB of |g|^2).
    The oracle gets g(Re,q) of both q from the same slabs, one Rp at a time (Eq. 9 is a sum over Rp), and one sampled pair
    per q (a pair costs the oracle's plain loops the better part of a minute)."""
    from parity import g2_pair_close

    w = synth.make_config(4)
    iqs = [37, 121]
    k_of = {37: 0, 121: 133}
    qs = np.ascontiguousarray(w.q_list[iqs])
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
    try:
        epw.epw_interp_set_wannier_operators(h.h, w.H_R, w.D_R, None, w.Re, w.w_e, w.Rp, w.w_p, 0)
        g1_ref = [np.zeros((w.nmodes, w.ne, w.nbnd, w.nbnd), dtype=np.complex128) for _ in iqs]
        for ip in range(w.np_):
            slab = w.g_slabs(ip, 1)
            epw.epw_interp_set_g_slabs(h.h, ip, 1, slab, 0)
            for j in range(len(iqs)):
                g1_ref[j] += oracle.rp_to_q(slab, w.Rp[ip:ip + 1], w.w_p[ip:ip + 1], qs[j])
            del slab
        kq_map = np.ascontiguousarray(w.kq_map[iqs])
        eps_k, eps_kq, om, g2 = h.interpolate_grid(w.k_grid, dev(qs), kq_map=dev(kq_map))
        epw.epw_interp_sync(h.h)
        assert epw.epw_interp_last_plan(h.h)["path"] == "large"
        eps_k, eps_kq, om = eps_k.cpu().numpy(), eps_kq.cpu().numpy(), om.cpu().numpy()
        for j, iq in enumerate(iqs):
            e_ref, om_ref = oracle.phonon(w.D_R, w.Rp, w.w_p, qs[j])
            err, ok = eig_close(om[j], om_ref)
            assert ok, f"omega mismatch at q {iq}: {err:.3e}"
            ik = k_of[iq]
            r_g2, r_ek, r_ekq = oracle.pair(g1_ref[j], w.H_R, w.Re, w.w_e, e_ref, om_ref, w.k_list[ik], qs[j])
            err, ok = eig_close(eps_k[ik], r_ek)
            assert ok, f"eps_k mismatch at k {ik}: {err:.3e}"
            err, ok = eig_close(eps_kq[j, ik], r_ekq)
            assert ok, f"eps_kq mismatch at q {iq}, k {ik}: {err:.3e}"
            wst, ok = g2_pair_close(g2[j, ik].cpu().numpy(), r_g2, r_ekq, r_ek, om_ref)
            assert ok, f"|g|^2 mismatch at q {iq}, k {ik}: {wst:.3f} x tolerance"
            print(f"config 4 full size, q {iq}, k {ik}: worst |g|^2 deviation {wst:.3f} x tolerance")
    finally:
        h.close()


# ---------------------------------------------------------------------------------------------------------
# NEXT-1: g(Re,Rp) split by Rp over ranks.  One GPU here: the two "ranks" are two handles run
# one after the other (no kernel waits on another), their partial g(Re,q) summed explicitly where NCCL would.
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("large", [False, True])
def test_rp_sharded_two_handles(epw, large):
    from paper_2603_10295_b200 import shard

    if large:
        w = synth.make_custom("zsnr-s", 18, 6, (3, 0, 0), 1.0, 0.05, 2.0, (40, 1, 1), ("random", 3, 1), seed=51)
    else:
        w = synth.make_custom("si-s", 8, 6, (1, 2, 1), 1.5, 0.1, 1.5, (6, 5, 4), ("random", 5, 3), seed=52)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    world = 2
    rows = w.nbnd * w.nbnd * w.nmodes * w.ne
    handles = []
    try:
        for r, (a, b) in enumerate(shard.rp_ranges(w.np_, world)):
            h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, q_batch=2)
            h.set_operators_from_host(w, rp_range=(a, b))
            handles.append(h)
        # a sharded handle refuses the unsharded call
        with pytest.raises(epw.EpwError):
            handles[0].interpolate(dev(w.k_list), dev(w.q_list))
        q_d = dev(w.q_list)
        partial = []
        for h in handles:
            g1 = torch.empty((w.nq, rows, 2), dtype=torch.float64, device="cuda")
            epw.epw_interp_rp_to_q_partial(h.h, q_d, w.nq, g1)
            partial.append(g1)
        total = partial[0] + partial[1]          # what dist.all_reduce(SUM) leaves on every rank
        g1_ref = np.stack([oracle.rp_to_q(w.g_full(), w.Rp, w.w_p, q) for q in w.q_list]).reshape(w.nq, rows)
        assert np.abs(znp(total) - g1_ref).max() <= 1e-13 * np.abs(g1_ref).max()
        # each rank: the rest of the path on its own share of the k-points, through the helper bench / users call
        outs = []
        for r, (ka, kb) in enumerate(shard.k_ranges(w.nk, world)):
            res = {}

            def rest(h=handles[r], ka=ka, kb=kb):
                res["out"] = h.interpolate(dev(w.k_list[ka:kb]), q_d)

            shard.interpolate_rp_sharded(epw, handles[r].h, q_d, w.nq, rows, rest, reduce_fn=lambda t: total)
            epw.epw_interp_sync(handles[r].h)
            outs.append([t.cpu().numpy() for t in res["out"]])
        eps_k = np.concatenate([o[0] for o in outs], axis=0)
        eps_kq = np.concatenate([o[1] for o in outs], axis=1)
        g2 = np.concatenate([o[3] for o in outs], axis=1)
        assert_path_close((eps_k, eps_kq, outs[0][2], g2), ref)
        np.testing.assert_array_equal(outs[0][2], outs[1][2])  # omega_q identical on both ranks
    finally:
        for h in handles:
            h.close()


def test_rp_sharded_fused_scatter_add(epw):
    """NEXT-1 with the exchange step fused into the S1 kernel (epw_interp_rp_to_q_scatter_add): two Rp-shard handles, each
    on its own stream at the same time, add their partial g(Re,q) straight into the buffers of the q-points' owners (here
    both 'owners' live on this GPU; across GPUs the pointers are peer mappings and the adds cross NVLink).  No kernel
    waits on another.  The summed g(Re,q) against the oracle's Eq. 9, then the rest of the path on it."""
    from paper_2603_10295_b200 import shard

    # 12 q: two S1 batches of 8 and 4 -> the bulk-TMA kernel (NQ = 8) and the register-staged one (NQ = 4)
    w = synth.make_custom("si-f", 8, 6, (2, 2, 2), 1.5, 0.1, 1.5, (6, 5, 4), ("random", 12, 3), seed=53)
    g = w.g_full()
    rows = w.nbnd * w.nbnd * w.nmodes * w.ne
    world = 2
    handles, streams = [], [torch.cuda.Stream() for _ in range(world)]
    try:
        for a, b in shard.rp_ranges(w.np_, world):
            h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
            h.set_operators_from_host(w, rp_range=(a, b))
            handles.append(h)
        q_d = dev(w.q_list)
        # owner of q-point iq = rank iq % 2; every owner zeroes its own buffers
        own = [torch.zeros((w.nq, rows, 2), dtype=torch.float64, device="cuda") for _ in range(world)]
        dst = [own[iq % world][iq] for iq in range(w.nq)]
        torch.cuda.synchronize()
        for r in range(world):
            with torch.cuda.stream(streams[r]):
                epw.epw_interp_rp_to_q_scatter_add(handles[r].h, q_d, w.nq, dst)
        torch.cuda.synchronize()   # (the barrier between the ranks)
        total = torch.stack(dst)
        g1_ref = np.stack([oracle.rp_to_q(g, w.Rp, w.w_p, q) for q in w.q_list]).reshape(w.nq, rows)
        assert np.abs(znp(total) - g1_ref).max() <= 1e-13 * np.abs(g1_ref).max()
        # the rest of the path on the summed g(Re,q)
        ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
        epw.epw_interp_set_gq(handles[0].h, total)
        out = handles[0].interpolate_grid(w.k_grid, q_d)
        epw.epw_interp_sync(handles[0].h)
        epw.epw_interp_set_gq(handles[0].h, None)
        assert_path_close([t_.cpu().numpy() for t_ in out], ref)
    finally:
        for h in handles:
            h.close()


# ---------------------------------------------------------------------------------------------------------
# NEXT-3: energy-window pre-screening of the pairs
# ---------------------------------------------------------------------------------------------------------
def pick_window(eps_all, frac_lo=0.48, frac_hi=0.52, margin=1e-6):
    """A window whose edges are at least `margin` away from every eigenvalue, so that the keep / skip decision is the
    same on both sides although their eigenvalues differ in the last digits (floats deciding an integer)."""
    v = np.sort(np.asarray(eps_all).ravel())
    lo, hi = v[int(frac_lo * len(v))], v[int(frac_hi * len(v))]
    for edge in ("lo", "hi"):
        x = lo if edge == "lo" else hi
        while np.abs(v - x).min() < margin:
            x += 3.3 * margin
        lo, hi = (x, hi) if edge == "lo" else (lo, x)
    return float(lo), float(hi)


@pytest.mark.parametrize("mode", ["grid-fused", "grid-unfused", "list", "list-kqmap", "large"])
def test_energy_window_screening(epw, mode):
    fl = {"grid-fused": 2, "grid-unfused": 1}.get(mode, 0)
    if mode == "large":
        w = synth.make_custom("zsnr-w", 18, 5, (2, 0, 0), 1.0, 0.05, 2.0, (30, 1, 1), ("random", 3, 1), seed=61)
    else:
        w = synth.make_config(0)
    ql = w.q_list[:6] if mode == "list-kqmap" else (w.q_list[:6] + ([0.013, 0.007, 0.021] if mode != "large" else 0.0))
    kq_map = np.ascontiguousarray(w.kq_map[:6]) if mode == "list-kqmap" else None
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, ql)
    emin, emax = pick_window(np.concatenate([ref[0].ravel(), ref[1].ravel()]))
    mask_ref = oracle.window_mask(ref[0], ref[1], emin, emax)
    assert 0.02 < mask_ref.mean() < 0.95      # the window really screens, and really keeps
    g2_ref = ref[3] * mask_ref[:, :, None, None, None]
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, q_batch=4, flags=fl)
    try:
        h.set_operators_from_host(w)
        mask_d = torch.full((len(ql), w.nk), 7, dtype=torch.uint8, device="cuda")
        epw.epw_interp_set_energy_window(h.h, True, emin, emax, mask_d)
        if mode.startswith("grid"):
            out = h.interpolate_grid(w.k_grid, dev(ql))
        else:
            out = h.interpolate(dev(w.k_list), dev(ql), None if kq_map is None else dev(kq_map))
        epw.epw_interp_sync(h.h)
        eps_k, eps_kq, om, g2 = [t.cpu().numpy() for t in out]
        np.testing.assert_array_equal(mask_d.cpu().numpy(), mask_ref)        # integer decision: bit-exact
        assert (g2[mask_ref == 0] == 0.0).all()                              # skipped pairs report exact zeros
        kept = [(iq, ik) for iq in range(len(ql)) for ik in range(w.nk) if mask_ref[iq, ik]]
        assert_path_close((eps_k, eps_kq, om, g2), (ref[0], ref[1], ref[2], g2_ref), pairs=kept)
        # switching the window off restores the full result (no internal mask buffer this time)
        epw.epw_interp_set_energy_window(h.h, False)
        out = h.interpolate_grid(w.k_grid, dev(ql)) if mode.startswith("grid") else \
            h.interpolate(dev(w.k_list), dev(ql), None if kq_map is None else dev(kq_map))
        epw.epw_interp_sync(h.h)
        assert_path_close([t.cpu().numpy() for t in out], ref, pairs=kept[:50] + [(0, 0), (len(ql) - 1, w.nk - 1)])
        # internal mask buffer (mask_out = NULL)
        epw.epw_interp_set_energy_window(h.h, True, emin, emax, None)
        out = h.interpolate_grid(w.k_grid, dev(ql)) if mode.startswith("grid") else \
            h.interpolate(dev(w.k_list), dev(ql), None if kq_map is None else dev(kq_map))
        epw.epw_interp_sync(h.h)
        g2b = out[3].cpu().numpy()
        assert (g2b[mask_ref == 0] == 0.0).all() and np.array_equal(g2b != 0, g2 != 0)
    finally:
        h.close()


# ---------------------------------------------------------------------------------------------------------
# degenerate cases of the method
# ---------------------------------------------------------------------------------------------------------
class _Wl:
    """Minimal workload object for EpwInterp.set_operators_from_host built from explicit arrays."""

    def __init__(self, H_R, D_R, g, Re, Rp, w_e=None, w_p=None):
        self.H_R, self.D_R, self._g, self.Re, self.Rp = H_R, D_R, np.ascontiguousarray(g), Re, Rp
        self.nbnd, self.nmodes, self.ne, self.np_ = H_R.shape[1], D_R.shape[1], len(Re), len(Rp)
        self.w_e = np.ones(self.ne) if w_e is None else w_e
        self.w_p = np.ones(self.np_) if w_p is None else w_p
        self.slab_elems = self.nbnd * self.nbnd * self.ne * self.nmodes

    def g_slabs(self, ip, cnt):
        return np.ascontiguousarray(self._g[ip:ip + cnt])

    def g_full(self):
        return self._g


@pytest.mark.parametrize("route", ["list", "grid", "large"])
def test_exactly_degenerate_bands_and_modes(epw, route):
    """H(R) = 1_2 (x) h(R) and D(R) = 1_2 (x) d(R): every band and every mode is exactly two-fold degenerate at every k, q,
    so individual |g_mn nu|^2 are not unique (reading G10) -- compare sums over the degenerate blocks."""
    base = synth.make_custom("deg", 3, 2, (1, 1, 0), 1.0, 0.1, 1.0, (5, 4, 1), ("random", 3, 2), seed=71)
    H = np.stack([np.kron(np.eye(2), base.H_R[i].T).T for i in range(base.ne)])   # column-major storage [j][i]
    D = np.stack([np.kron(np.eye(2), base.D_R[i].T).T for i in range(base.np_)])
    nb, nm = 6, 4
    g = 0.1 * crandn(base.np_, nm, base.ne, nb, nb) * np.exp(-np.linalg.norm(base.Re, axis=1))[None, None, :, None, None]
    w = _Wl(np.ascontiguousarray(H), np.ascontiguousarray(D), g, base.Re, base.Rp)
    ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, base.k_list, base.q_list)
    assert np.abs(ref[0][:, 0] - ref[0][:, 1]).max() < 1e-9        # the spectrum really is pairwise degenerate
    kw = dict(path=2) if route == "large" else (dict(grid=base.k_grid) if route == "grid" else {})
    assert_path_close(run_gpu(epw, w, base.k_list, base.q_list, **kw), ref)


@pytest.mark.parametrize("route", ["list", "grid", "large"])
def test_omega_min_cutoff_and_tiny_lists(epw, route):
    """Modes with omega <= omega_min report |g|^2 = 0 exactly (reading G12); one k and one q; nq not a multiple of the S1
    batch."""
    w = synth.make_custom("cut", 4, 5, (1, 1, 1), 1.0, 0.1, 1.0, (3, 2, 2), ("random", 11, 3), seed=72)
    g = w.g_full()
    om = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list[:1], w.q_list)[2]
    omega_min = float(np.sort(om.ravel())[len(om.ravel()) // 3]) + 1e-7     # cuts about a third of the modes
    ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list, omega_min=omega_min)
    assert (ref[3] == 0).any() and (ref[3] != 0).any()
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, omega_min=omega_min, path=2 if route == "large" else 0, q_batch=4)
    try:
        h.set_operators_from_host(w)
        out = h.interpolate_grid(w.k_grid, dev(w.q_list)) if route == "grid" else h.interpolate(dev(w.k_list), dev(w.q_list))
        epw.epw_interp_sync(h.h)
        got = [t.cpu().numpy() for t in out]
        assert_path_close(got, ref)
        assert np.array_equal(got[3] == 0, ref[3] == 0)
        # one k, one q
        k1, q1 = w.k_list[5:6], w.q_list[3:4]
        ref1 = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, k1, q1, omega_min=omega_min)
        out = h.interpolate(dev(k1), dev(q1))
        epw.epw_interp_sync(h.h)
        assert_path_close([t.cpu().numpy() for t in out], ref1)
        if route == "grid":   # a 1 x 1 x 1 "grid" with a shift = the single point k1
            out = h.interpolate_grid((1, 1, 1), dev(q1), k_shift=tuple(k1[0]))
            epw.epw_interp_sync(h.h)
            assert_path_close([t.cpu().numpy() for t in out], ref1)
    finally:
        h.close()


# ---------------------------------------------------------------------------------------------------------
# NEXT-4: a consumer of |g|^2 on the device (Im Sigma_nk accumulator, reading G18)
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["grid-fused-nog2", "grid-fused", "grid-fused-kqmap-nog2", "grid-fused-nb13-nog2",
                                  "grid-unfused", "list", "list-kqmap-nog2", "large", "large-nog2"])
def test_selfenergy_consumer(epw, mode):
    """NEXT-4 consumer against oracle.selfenergy_accumulate in every kernel route.  grid-fused*: the reduction runs in the
    epilogue of the one-kernel grid form (nb13: Nb = 13, Nm = 12, modes split over several tiles -> atomic adds); the other
    routes reduce a one-q |g|^2 slab with a second kernel.  Tolerance per entry: 1e-8 relative + 1e-10 of the largest entry
    (reading G18: sums of up to Nq Nb Nm non-negative products of |g|^2, itself within 1e-9, and Gaussian weights
    evaluated in FP64 on both sides; the absolute term covers entries made only of terms below the kernels' e^-50 cut-off)."""
    if "nb13" in mode:
        w = synth.make_custom("modes", 13, 12, (3, 1, 0), 1.0, 0.1, 1.0, (10, 3, 1), ("random", 5, 2), seed=15)
        ql, kq_map = w.q_list, None
    elif mode.startswith("large"):
        w = synth.make_custom("zsnr-se", 18, 5, (2, 0, 0), 1.0, 0.05, 2.0, (24, 1, 1), ("random", 5, 1), seed=81)
        ql, kq_map = w.q_list, None
    else:
        w = synth.make_config(0)
        ql = w.q_list[:6] if "kqmap" in mode else w.q_list[:6] + [0.013, 0.007, 0.021]
        kq_map = np.ascontiguousarray(w.kq_map[:6]) if "kqmap" in mode else None
    nq = len(ql)
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, ql)
    mu = float(np.median(ref[0]))
    kT, sigma = 0.05, 0.08
    wq = np.random.default_rng(5).uniform(0.5, 1.5, size=nq)
    want = oracle.selfenergy_accumulate(ref[3], ref[0], ref[1], ref[2], wq, mu, kT, sigma)
    want2 = oracle.selfenergy_accumulate(ref[3][:2], ref[0], ref[1][:2], ref[2][:2], None, mu, kT, sigma, out=want.copy())
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, q_batch=4, path=2 if mode.startswith("large") else 0,
                      flags=2 if mode.startswith("grid-fused") else (1 if mode == "grid-unfused" else 0))
    try:
        h.set_operators_from_host(w)
        acc = torch.zeros((w.nk, w.nbnd), dtype=torch.float64, device="cuda")
        wq_d = dev(wq)
        epw.epw_interp_set_selfenergy_consumer(h.h, True, mu, kT, sigma, wq_d, acc)
        nog2 = mode.endswith("nog2")
        eps_k = torch.empty((w.nk, w.nbnd), dtype=torch.float64, device="cuda")
        om = torch.empty((nq, w.nmodes), dtype=torch.float64, device="cuda")
        g2 = None if nog2 else torch.empty((nq, w.nk, w.nmodes, w.nbnd, w.nbnd), dtype=torch.float64, device="cuda")
        q_d, k_d = dev(ql), dev(w.k_list)
        map_d = None if kq_map is None else dev(kq_map)

        def call(nq_call, eps_kq):
            if mode.startswith("grid"):
                epw.epw_interp_interpolate_grid(h.h, w.k_grid, None, q_d, nq_call, map_d, eps_k, eps_kq, om, g2)
            else:
                epw.epw_interp_interpolate(h.h, k_d, w.nk, q_d, nq_call, map_d, eps_k, eps_kq, om, g2)
            epw.epw_interp_sync(h.h)

        call(nq, None)   # eps_kq = NULL: the consumer reads the library's own eigenvalues
        got = acc.cpu().numpy()
        assert np.all(np.abs(got - want) <= 1e-8 * np.abs(want) + 1e-10 * np.abs(want).max())
        if g2 is not None:   # |g|^2 is still delivered when the caller asks for it
            assert_path_close((eps_k.cpu().numpy(), ref[1], om.cpu().numpy(), g2.cpu().numpy()), ref,   # eps_kq not requested
                              pairs=[(0, 0), (nq - 1, w.nk - 1), (2, 7)])
        # a second call accumulates (first two q again, unit weights)
        epw.epw_interp_set_selfenergy_consumer(h.h, True, mu, kT, sigma, None, acc)
        eps_kq = torch.empty((2, w.nk, w.nbnd), dtype=torch.float64, device="cuda")
        call(2, eps_kq)
        got2 = acc.cpu().numpy()
        assert np.all(np.abs(got2 - want2) <= 1e-8 * np.abs(want2) + 1e-10 * np.abs(want2).max())
        # g2 = NULL without a consumer is an error
        epw.epw_interp_set_selfenergy_consumer(h.h, False)
        if nog2:
            with pytest.raises(epw.EpwError):
                call(2, eps_kq)
    finally:
        h.close()


@pytest.mark.parametrize("delta", [3e-7, 1e-4])
@pytest.mark.parametrize("route", ["list", "grid"])
def test_nearly_degenerate_bands(epw, route, delta):
    """Bands split by delta: 3e-7 eV (inside the 1e-6 eV degeneracy window: compared as block sums) and 1e-4 eV (resolved
    individually: the eigenvectors must then be accurate to ~ eps / delta)."""
    base = synth.make_custom("ndeg", 3, 3, (1, 1, 0), 1.0, 0.1, 1.0, (5, 4, 1), ("random", 3, 2), seed=73)
    H = np.stack([np.kron(np.eye(2), base.H_R[i].T).T for i in range(base.ne)])
    i0 = [i for i, r in enumerate(base.Re) if not r.any()][0]
    H[i0] += np.diag([0, 0, 0, delta, delta, delta])
    nb, nm = 6, 3
    g = 0.1 * crandn(base.np_, nm, base.ne, nb, nb) * np.exp(-np.linalg.norm(base.Re, axis=1))[None, None, :, None, None]
    w = _Wl(np.ascontiguousarray(H), base.D_R, g, base.Re, base.Rp)
    ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, base.k_list, base.q_list)
    gaps = np.diff(ref[0], axis=1)
    assert np.abs(gaps - delta).min() < 1e-9            # the splitting is really there
    kw = dict(grid=base.k_grid) if route == "grid" else {}
    assert_path_close(run_gpu(epw, w, base.k_list, base.q_list, **kw), ref)


def test_many_lattice_vectors_clamp_the_s1_batch(epw):
    """Np = 2,197 (a 13^3 Wigner-Seitz box): the [Np][8] phase table of the default S1 batch does not fit shared memory,
    so the library lowers the batch (6 q per pass here) instead of failing; 9 q = one full and one ragged pass."""
    w = synth.make_custom("many-R", 1, 1, (6, 6, 6), 2.0, 0.1, 2.0, (2, 3, 1), ("random", 9, 3), seed=41)
    assert w.np_ == 2197
    ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
    try:
        h.set_operators_from_host(w)
        out = h.interpolate(dev(w.k_list), dev(w.q_list))
        epw.epw_interp_sync(h.h)
        assert epw.epw_interp_last_plan(h.h)["q_batch"] == 6
        assert_path_close([t.cpu().numpy() for t in out], ref)
        out = h.interpolate_grid(w.k_grid, dev(w.q_list))
        epw.epw_interp_sync(h.h)
        assert_path_close([t.cpu().numpy() for t in out], ref)
    finally:
        h.close()


def test_two_handles_from_two_threads_count_their_own_rotations(epw):
    """include/epw_interp.h: distinct handles are independent.  Two handles with stage timing on, driven from two host
    threads on two streams at the same time, must report the rotation counts (and results) of their serial runs."""
    import threading

    ws = [synth.make_custom("si-a", 8, 6, (1, 1, 1), 1.5, 0.1, 1.5, (12, 12, 16), ("random", 3, 3), seed=51),
          synth.make_custom("si-b", 6, 3, (1, 1, 1), 1.0, 0.1, 1.0, (16, 12, 12), ("random", 2, 3), seed=52)]

    def run(w, stream, out):
        with torch.cuda.stream(stream):
            h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
            try:
                h.set_operators_from_host(w)
                epw.epw_interp_enable_stage_timing(h.h, True)
                for _ in range(3):
                    res = h.interpolate_grid(w.k_grid, dev(w.q_list))
                epw.epw_interp_sync(h.h)
                out["rot"] = epw.epw_interp_get_eigh_rotations(h.h)
                out["g2"] = res[3].cpu().numpy()
            finally:
                h.close()

    serial = [dict(), dict()]
    for w, o in zip(ws, serial):
        run(w, torch.cuda.Stream(), o)
    par = [dict(), dict()]
    th = [threading.Thread(target=run, args=(w, torch.cuda.Stream(), o)) for w, o in zip(ws, par)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for s, p in zip(serial, par):
        assert s["rot"]["Hkq"] > 0 and s["rot"] == p["rot"]
        assert np.array_equal(s["g2"], p["g2"])


def test_large_path_k_side_cache_and_its_invalidation(epw):
    """Large-Nb family on a uniform grid: the k side (phases, H(k), U_k, eps_k) is kept between calls on the same grid.
    Second call on the same grid (cache hit: fewer launches, same results), a call with k+q off the grid after one with
    kq_map (the packed conj U_k is overwritten), a SHIFTED grid (k changes: miss), and new operators (miss) are each
    checked against the oracle."""
    w = synth.make_custom("zsnr-c", 20, 12, (2, 0, 0), 1.0, 0.05, 2.0, (10, 1, 1), ("grid", (10, 1, 1)), seed=24)
    g = w.g_full()
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
    try:
        h.set_operators_from_host(w)

        def call(q, kq, shift=None):
            out = h.interpolate_grid(w.k_grid, dev(q), k_shift=shift, kq_map=None if kq is None else dev(kq))
            epw.epw_interp_sync(h.h)
            return [t.cpu().numpy() for t in out], epw.epw_interp_last_launch_count(h.h)

        qa, qb = w.q_list[:3], w.q_list[3:6]
        ref_a = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, qa)
        ref_b = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, qb)
        out1, n1 = call(qa, w.kq_map[:3])
        assert_path_close(out1, ref_a)
        out2, n2 = call(qb, w.kq_map[3:6])            # same grid: cache hit
        assert n2 < n1
        assert_path_close(out2, ref_b)
        q_off = qa + 0.013
        ref_off = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, q_off)
        out3, _ = call(q_off, None)                   # per-pair H(k+q): overwrites the packed conj(U_k)
        assert_path_close(out3, ref_off)
        out4, n4 = call(qa, w.kq_map[:3])             # must rebuild it
        assert_path_close(out4, ref_a)
        shift = np.array([0.25, 0.0, 0.0])
        k_sh = w.k_list + shift / np.array(w.k_grid)
        ref_sh = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, k_sh, q_off)
        out5, n5 = call(q_off, None, shift=shift)     # k changed between calls: miss
        assert_path_close(out5, ref_sh)
        w2 = synth.make_custom("zsnr-c2", 20, 12, (2, 0, 0), 1.0, 0.05, 2.0, (10, 1, 1), ("grid", (10, 1, 1)), seed=25)
        h.set_operators_from_host(w2)                 # new operators, same grid: miss
        ref_w2 = oracle.interpolate(w2.H_R, w2.D_R, w2.g_full(), w2.Re, w2.w_e, w2.Rp, w2.w_p, k_sh, q_off)
        out6, _ = call(q_off, None, shift=shift)
        assert_path_close(out6, ref_w2)
    finally:
        h.close()


@pytest.mark.parametrize("flags", [0, 1])
def test_small_path_k_side_cache_on_a_grid(epw, flags):
    """Small-Nb family on a uniform grid: U_k and eps_k are kept between calls on the same grid (second call: fewer launches,
    same results); a shifted grid, a k-list call in between and new operators each invalidate the cache."""
    w = synth.make_custom("si-k", 8, 6, (1, 1, 1), 1.5, 0.1, 1.5, (6, 5, 4), ("random", 6, 3), seed=61)
    g = w.g_full()
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_, flags=flags)
    try:
        h.set_operators_from_host(w)

        def call(q, shift=None):
            out = h.interpolate_grid(w.k_grid, dev(q), k_shift=shift)
            epw.epw_interp_sync(h.h)
            return [t.cpu().numpy() for t in out], epw.epw_interp_last_launch_count(h.h)

        qa, qb = w.q_list[:3], w.q_list[3:]
        ref_a = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, qa)
        ref_b = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, qb)
        out1, n1 = call(qa)
        assert_path_close(out1, ref_a)
        out2, n2 = call(qb)                           # same grid: cache hit
        assert n2 < n1
        assert_path_close(out2, ref_b)
        shift = np.array([0.5, 0.25, 0.0])
        k_sh = w.k_list + shift / np.array(w.k_grid)
        ref_sh = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, k_sh, qa)
        out3, n3 = call(qa, shift=shift)              # k changed: miss
        assert n3 == n1
        assert_path_close(out3, ref_sh)
        outl = h.interpolate(dev(w.k_list), dev(qa))  # a k-list call overwrites U_k
        epw.epw_interp_sync(h.h)
        assert_path_close([t.cpu().numpy() for t in outl], ref_a)
        out4, n4 = call(qa, shift=shift)              # ... so the grid call after it recomputes
        assert n4 == n1
        assert_path_close(out4, ref_sh)
        w2 = synth.make_custom("si-k2", 8, 6, (1, 1, 1), 1.5, 0.1, 1.5, (6, 5, 4), ("random", 6, 3), seed=62)
        h.set_operators_from_host(w2)                 # new operators, same grid: miss
        ref_w2 = oracle.interpolate(w2.H_R, w2.D_R, w2.g_full(), w2.Re, w2.w_e, w2.Rp, w2.w_p, k_sh, w2.q_list[:3])
        out5, _ = call(w2.q_list[:3], shift=shift)
        assert_path_close(out5, ref_w2)
    finally:
        h.close()


def test_k_side_cache_dropped_when_an_eigensolve_did_not_converge(epw):
    """An H(k) solve that hits the sweep limit (here: a NaN in H(R), so no rotation ever converges) is reported by
    epw_interp_sync, and the k side it belongs to must not stay cached: with a kq_map the H(k) solves are the only band
    solves of a call, so the SECOND call on the same grid raises the flag again only if it solved H(k) again."""
    w = synth.make_custom("si-nan", 8, 6, (1, 1, 1), 1.5, 0.1, 1.5, (4, 4, 4), ("grid", (4, 4, 4)), seed=63)
    assert w.kq_map is not None
    ie0 = int(np.flatnonzero((w.Re == 0).all(axis=1))[0])
    H_bad = w.H_R.copy()
    H_bad.reshape(w.ne, w.nbnd, w.nbnd)[ie0, 0, 0] = np.nan
    h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
    try:
        epw.epw_interp_set_wannier_operators(h.h, H_bad, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, 0)
        for _ in range(2):
            h.interpolate_grid(w.k_grid, dev(w.q_list[:3]), kq_map=dev(w.kq_map[:3]))
            with pytest.raises(epw.EpwError) as e:
                epw.epw_interp_sync(h.h)
            assert e.value.code == epw.binding.EPW_ENOTCONVERGED
        # healthy operators afterwards: the handle is usable and right again
        h.set_operators_from_host(w)
        out = h.interpolate_grid(w.k_grid, dev(w.q_list[:3]), kq_map=dev(w.kq_map[:3]))
        epw.epw_interp_sync(h.h)
        ref = oracle.interpolate(w.H_R, w.D_R, w.g_full(), w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list[:3])
        assert_path_close([t.cpu().numpy() for t in out], ref)
    finally:
        h.close()
