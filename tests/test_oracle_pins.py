"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Nothing here comes from the CUDA path.  Each test states which part of
oracle/epw_oracle.c it pins and by what: a library routine (numpy.fft,
numpy.linalg.eigh), a closed form, an invariant, brute force, or a number the
paper prints (tests/golden/).
"""
import os

import numpy as np
import pytest

import oracle
from oracle import cm

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(20260310295)


def crandn(*shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def random_unitary_cm(n):
    """Random unitary from numpy QR, returned in the oracle's column-major storage [col][row]."""
    q, _ = np.linalg.qr(crandn(n, n))
    return np.ascontiguousarray(q.T)


def residue_vectors(N, shift):
    """One integer representative per residue class of Z^3 / (N1,N2,N3), shifted to include negatives."""
    ax = [np.arange(n) - s for n, s in zip(N, shift)]
    return np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.int32)


def grid(N):
    ax = [np.arange(n) / n for n in N]
    return np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)


# ---------------------------------------------------------------------------------------------
# Fourier sums (Eq. 9 and the FT part of Eq. 10): signs, weights, layouts.
# ---------------------------------------------------------------------------------------------
def _wannier_from_bloch_fft(G, Nk, Nq, Re, Rp):
    """Eq. 6 (U = u = 1) through numpy.fft: the forward DFT over the k' and q' grid
    indices, read off at (R mod N).  G [q1,q2,q3,k1,k2,k3,Nm,Nb,Nb] -> g_RR [Np][Nm][Ne][Nb][Nb]."""
    F = np.fft.fftn(G, axes=(0, 1, 2, 3, 4, 5), norm="forward")  # sum exp(-2 pi i n.m/N) / prod(N)
    out = np.empty((len(Rp), G.shape[6], len(Re)) + G.shape[7:], dtype=np.complex128)
    for ip, rp in enumerate(Rp):
        for ie, re in enumerate(Re):
            out[ip, :, ie] = F[rp[0] % Nq[0], rp[1] % Nq[1], rp[2] % Nq[2], re[0] % Nk[0], re[1] % Nk[1], re[2] % Nk[2]]
    return out


def test_roundtrip_against_numpy_fft():
    """Pin (library routine): g(Re,Rp) built from an arbitrary coarse-grid G(k',q') with numpy.fft is
    interpolated back by the oracle's Eq. 9 + Eq. 10-FT to G at every coarse point (PAPER.md:L78-84:
    Eqs. 6 and 7 are inverse generalized Fourier transforms)."""
    Nk, Nq, nb, nm = (3, 2, 4), (2, 3, 1), 2, 3
    Re = residue_vectors(Nk, (1, 1, 2))
    Rp = residue_vectors(Nq, (1, 1, 0))
    G = crandn(*Nq, *Nk, nm, nb, nb)
    g_RR = _wannier_from_bloch_fft(G, Nk, Nq, Re, Rp)
    kc, qc = grid(Nk), grid(Nq)
    w_e, w_p = np.ones(len(Re)), np.ones(len(Rp))
    Gf = G.reshape(len(qc), len(kc), nm, nb, nb)
    for iq, q in enumerate(qc):
        g1 = oracle.rp_to_q(g_RR, Rp, w_p, q)
        for ik, k in enumerate(kc):
            gt = oracle.re_to_k(g1, Re, w_e, k)
            np.testing.assert_allclose(gt, Gf[iq, ik], rtol=0, atol=1e-13 * np.abs(G).max())


def test_eq6_helper_matches_numpy_fft():
    """The test-only Eq. 6 helper agrees with numpy.fft (so it can feed other tests)."""
    Nk, Nq, nb, nm = (2, 3, 1), (2, 1, 2), 2, 2
    Re, Rp = residue_vectors(Nk, (0, 1, 0)), residue_vectors(Nq, (1, 0, 1))
    G = crandn(*Nq, *Nk, nm, nb, nb)
    ref = _wannier_from_bloch_fft(G, Nk, Nq, Re, Rp)
    got = oracle.eq6_wannier_from_bloch(G.reshape(4, 6, nm, nb, nb), grid(Nk), grid(Nq), Re, Rp)
    np.testing.assert_allclose(got, ref, rtol=0, atol=1e-14)


def test_weights_multiply_each_R_term():
    """Wigner-Seitz weights: splitting one R into two entries of weight 1/2 changes nothing [reading G7]."""
    nb, nm = 2, 2
    Re = np.array([[0, 0, 0], [1, 0, 0], [1, 0, 0], [-1, 2, 0]], dtype=np.int32)
    Rp = np.array([[0, 0, 0], [0, 1, 0], [0, 1, 0]], dtype=np.int32)
    g = crandn(3, nm, 4, nb, nb)
    g[:, :, 2] = g[:, :, 1]
    g[2] = g[1]
    w_e, w_p = np.array([1, 0.5, 0.5, 1.0]), np.array([1, 0.5, 0.5])
    q, k = np.array([0.3, 0.7, 0.1]), np.array([0.15, 0.4, 0.9])
    a = oracle.re_to_k(oracle.rp_to_q(g, Rp, w_p, q), Re, w_e, k)
    sel_e, sel_p = [0, 1, 3], [0, 1]
    b = oracle.re_to_k(oracle.rp_to_q(g[sel_p][:, :, sel_e], Rp[sel_p], np.ones(2), q), Re[sel_e], np.ones(3), k)
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-14)


def test_single_R0_term_is_k_q_independent():
    """Pin (special case): only R = 0 => g~(k,q) = g(0,0) for every k, q."""
    nb, nm = 3, 2
    R = np.zeros((1, 3), dtype=np.int32)
    g = crandn(1, nm, 1, nb, nb)
    for _ in range(4):
        k, q = rng.random(3), rng.random(3)
        gt = oracle.re_to_k(oracle.rp_to_q(g, R, np.ones(1), q), R, np.ones(1), k)
        np.testing.assert_allclose(gt, g[0, :, 0], rtol=0, atol=1e-15)


def test_periodicity_in_k_and_q():
    """Pin (invariant): k -> k + integer, q -> q + integer leave everything unchanged (R integer)."""
    nb, nm = 2, 2
    Re, Rp = residue_vectors((3, 3, 2), (1, 1, 1)), residue_vectors((2, 2, 2), (1, 1, 1))
    g = crandn(len(Rp), nm, len(Re), nb, nb)
    k, q = np.array([0.21, 0.43, 0.87]), np.array([0.05, 0.55, 0.31])
    a = oracle.re_to_k(oracle.rp_to_q(g, Rp, np.ones(len(Rp)), q), Re, np.ones(len(Re)), k)
    b = oracle.re_to_k(oracle.rp_to_q(g, Rp, np.ones(len(Rp)), q + [1, -2, 3]), Re, np.ones(len(Re)), k + [-1, 2, 1])
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-13)


def test_phase_sign_is_plus_i():
    """Pin (closed form): one term at R=(1,0,0), q=(1/4,0,0) gives the factor exp(+i pi/2) = +i
    (Eq. 9 carries e^{+i q.Rp}; L114, Eq. 10 carries e^{+i k.Re})."""
    R0 = np.array([[1, 0, 0]], dtype=np.int32)
    Z = np.zeros((1, 3), dtype=np.int32)
    g = np.ones((1, 1, 1, 1, 1), dtype=np.complex128)
    g1 = oracle.rp_to_q(g, R0, np.ones(1), [0.25, 0, 0])
    assert abs(g1.ravel()[0] - 1j) < 1e-15
    gt = oracle.re_to_k(oracle.rp_to_q(g, Z, np.ones(1), [0.25, 0, 0]), R0, np.ones(1), [0.25, 0, 0])
    assert abs(gt.ravel()[0] - 1j) < 1e-15
    assert abs(oracle.phase([0.75, 0.5, 0.0], [-1, 1, 5]) - 2 * np.pi * 0.75) < 1e-14


# ---------------------------------------------------------------------------------------------
# Operator interpolation + eigenvalues: closed forms.
# ---------------------------------------------------------------------------------------------
def test_chain_closed_form_dispersion():
    """Pin (closed form): 1-D chain Nb = Nm = 1, H(0) = e0, H(+-1) = t  =>  eps(k) = e0 + 2 t cos(2 pi k);
    D likewise => omega(q) = sqrt(d0 + 2 d1 cos(2 pi q)); |g|^2 = |sum g(Re,Rp) e^{i(..)}|^2 / (2 omega)."""
    R = np.array([[-1, 0, 0], [0, 0, 0], [1, 0, 0]], dtype=np.int32)
    e0, t, d0, d1 = 0.3, -0.7, 2.5, 0.4
    H_R = np.array([t, e0, t], dtype=np.complex128).reshape(3, 1, 1)
    D_R = np.array([d1, d0, d1], dtype=np.complex128).reshape(3, 1, 1)
    g = crandn(3, 1, 3, 1, 1)
    w = np.ones(3)
    for k, q in [(0.0, 0.0), (0.1, 0.37), (0.5, 0.25), (0.83, 0.9)]:
        kv, qv = np.array([k, 0, 0]), np.array([q, 0, 0])
        eps_k, eps_kq, om, g2 = oracle.interpolate(H_R, D_R, g, R, w, R, w, kv, qv)
        assert abs(eps_k[0, 0] - (e0 + 2 * t * np.cos(2 * np.pi * k))) < 1e-14
        assert abs(eps_kq[0, 0, 0] - (e0 + 2 * t * np.cos(2 * np.pi * (k + q)))) < 1e-14
        w_ref = np.sqrt(d0 + 2 * d1 * np.cos(2 * np.pi * q))
        assert abs(om[0, 0] - w_ref) < 1e-14
        amp = sum(g[ip, 0, ie, 0, 0] * np.exp(2j * np.pi * (q * R[ip, 0] + k * R[ie, 0])) for ip in range(3) for ie in range(3))
        assert abs(g2.ravel()[0] - abs(amp) ** 2 / (2 * w_ref)) < 1e-13 * abs(amp) ** 2


def test_hermitian_family_gives_hermitian_Hk_and_real_eigenvalues():
    """Pin (invariant): H(-R) = H(R)^dagger  =>  H(k) Hermitian (before the symmetrisation step)."""
    nb = 4
    R = residue_vectors((3, 3, 1), (1, 1, 0))
    H_R = np.empty((len(R), nb, nb), dtype=np.complex128)
    for i in range(len(R)):
        j = len(R) - 1 - i
        if i <= j:
            m = crandn(nb, nb)
            H_R[i] = m if i != j else 0.5 * (m + m.conj().T)
            H_R[j] = H_R[i].conj().T
    k = np.array([0.123, 0.456, 0.0])
    ph = np.exp(2j * np.pi * (R @ k))
    raw = np.einsum("r,rji->ij", ph, H_R)  # un-symmetrised definition
    assert np.abs(raw - raw.conj().T).max() < 1e-13
    Hk = cm(oracle.interp_operator(H_R, R, np.ones(len(R)), k))
    np.testing.assert_allclose(Hk, raw, rtol=0, atol=1e-13)
    ev, V, sw = oracle.eigh_jacobi(oracle.interp_operator(H_R, R, np.ones(len(R)), k))
    np.testing.assert_allclose(ev, np.linalg.eigvalsh(raw), rtol=0, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# Jacobi eigensolver.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 6, 8, 11, 24])
def test_jacobi_residual_unitarity_and_eigh(n):
    """Pins (invariants + library routine): ||A V - V lambda|| <= 1e-13 ||A||, ||V^dagger V - I|| <= 1e-13,
    eigenvalues ascending and equal to numpy.linalg.eigh's."""
    for _ in range(5):
        M = crandn(n, n)
        A = 0.5 * (M + M.conj().T)
        ev, Vcm, sweeps = oracle.eigh_jacobi(np.ascontiguousarray(A.T))
        assert 0 <= sweeps <= 20
        V = cm(Vcm)
        nrm = np.linalg.norm(A)
        assert np.linalg.norm(A @ V - V * ev[None, :]) <= 1e-13 * max(nrm, 1e-300)
        assert np.linalg.norm(V.conj().T @ V - np.eye(n)) <= 1e-13
        assert np.all(np.diff(ev) >= 0)
        np.testing.assert_allclose(ev, np.linalg.eigvalsh(A), rtol=0, atol=1e-13 * nrm)


def test_jacobi_2x2_closed_form():
    """Pin (closed form): [[a, b],[b*, d]] has lambda = (a+d)/2 -+ sqrt(((a-d)/2)^2 + |b|^2)."""
    a, d, b = 0.7, -1.3, 0.4 - 0.9j
    A = np.array([[a, b], [np.conj(b), d]])
    ev, Vcm, _ = oracle.eigh_jacobi(np.ascontiguousarray(A.T))
    r = np.sqrt(((a - d) / 2) ** 2 + abs(b) ** 2)
    np.testing.assert_allclose(ev, [(a + d) / 2 - r, (a + d) / 2 + r], rtol=0, atol=1e-15)
    V = cm(Vcm)
    # eigenvector of lambda_-: (b, lambda_- - a) up to normalisation and phase
    v = np.array([b, ev[0] - a])
    v /= np.linalg.norm(v)
    assert abs(abs(np.vdot(v, V[:, 0])) - 1) < 1e-14


def test_jacobi_degenerate_and_diagonal():
    """Special cases: already diagonal (unsorted) input; exactly degenerate spectrum."""
    d = np.array([3.0, -1.0, 2.0, -1.0])
    ev, Vcm, sw = oracle.eigh_jacobi(np.diag(d).astype(np.complex128))
    assert sw == 0
    np.testing.assert_array_equal(ev, np.sort(d))
    V = cm(Vcm)
    np.testing.assert_allclose(np.diag(d) @ V, V * ev[None, :], atol=0)
    Q = cm(random_unitary_cm(5))
    lam = np.array([1.0, 1.0, 1.0, 2.0, 2.0])
    A = (Q * lam) @ Q.conj().T
    A = 0.5 * (A + A.conj().T)
    ev, Vcm, sw = oracle.eigh_jacobi(np.ascontiguousarray(A.T))
    np.testing.assert_allclose(ev, lam, atol=1e-14)
    V = cm(Vcm)
    assert np.linalg.norm(A @ V - V * ev) < 1e-13


def test_omega_is_sqrt_of_lambda_with_sign():
    lam = np.array([-4.0, 0.0, 9.0])
    np.testing.assert_array_equal(oracle.omega_from_lambda(lam), [-2.0, -0.0, 3.0])


# ---------------------------------------------------------------------------------------------
# Rotations, amplitude, index placement.
# ---------------------------------------------------------------------------------------------
def test_diagonal_operators_reduce_to_amplitude_only():
    """Pin (special case chained onto the FFT round trip): H(R) = delta_R0 diag(distinct ascending),
    D(R) = delta_R0 diag(distinct ascending) => U = e = 1 => |g_mn nu|^2 = |G_mn nu(k',q')|^2 / (2 omega_nu)
    with omega_nu = sqrt(D_nu nu) -- pins the 1/sqrt(2 omega) amplitude and omega = sqrt(lambda)."""
    Nk, Nq, nb, nm = (2, 2, 1), (2, 1, 1), 3, 2
    Re, Rp = residue_vectors(Nk, (1, 0, 0)), residue_vectors(Nq, (0, 0, 0))
    G = crandn(*Nq, *Nk, nm, nb, nb)
    g_RR = _wannier_from_bloch_fft(G, Nk, Nq, Re, Rp)
    hd, dd = np.array([-1.0, 0.5, 2.0]), np.array([1.5, 4.0])
    H_R = np.zeros((len(Re), nb, nb), dtype=np.complex128)
    H_R[[i for i, r in enumerate(Re) if not r.any()][0]] = np.diag(hd)
    D_R = np.zeros((len(Rp), nm, nm), dtype=np.complex128)
    D_R[[i for i, r in enumerate(Rp) if not r.any()][0]] = np.diag(dd)
    kc, qc = grid(Nk), grid(Nq)
    eps_k, eps_kq, om, g2 = oracle.interpolate(H_R, D_R, g_RR, Re, np.ones(len(Re)), Rp, np.ones(len(Rp)), kc, qc)
    np.testing.assert_allclose(eps_k, np.tile(hd, (len(kc), 1)), atol=1e-15)
    np.testing.assert_allclose(om, np.tile(np.sqrt(dd), (len(qc), 1)), atol=1e-15)
    ref = np.abs(G.reshape(len(qc), len(kc), nm, nb, nb)) ** 2 / (2 * np.sqrt(dd))[None, None, :, None, None]
    np.testing.assert_allclose(g2, ref, rtol=1e-12, atol=1e-14)


def test_permutation_case_pins_which_index_goes_with_k_and_kq():
    """Pin (closed form): diagonal H(R) with band crossings. eps_i(k) = d_i + 2 t_i cos(2 pi k), U_k is the
    permutation that sorts them, so g2[nu][n][m] = |g~[nu][pi_k(n)][pi_kq(m)]|^2 / (2 omega): the first
    Wannier index m' (fastest) is rotated by k+q, the second n' by k [reading G5], eigenvalues ascending."""
    nb, nm = 3, 1
    R = np.array([[-1, 0, 0], [0, 0, 0], [1, 0, 0]], dtype=np.int32)
    d, t = np.array([0.0, 0.1, -0.2]), np.array([0.5, -0.4, 0.3])
    H_R = np.stack([np.diag(t), np.diag(d), np.diag(t)]).astype(np.complex128)
    D_R = np.array([0.0, 2.0, 0.0], dtype=np.complex128).reshape(3, 1, 1)
    g = np.zeros((3, nm, 3, nb, nb), dtype=np.complex128)
    gt0 = crandn(nm, nb, nb)  # only Re = Rp = 0 => g~(k,q) = gt0, stored [nu][n'][m']
    g[1, :, 1] = gt0
    differing = 0
    for k, q in [(0.05, 0.2), (0.3, 0.45), (0.6, 0.15), (0.02, 0.5)]:
        ek = d + 2 * t * np.cos(2 * np.pi * k)
        ekq = d + 2 * t * np.cos(2 * np.pi * (k + q))
        pk, pkq = np.argsort(ek), np.argsort(ekq)
        differing += not np.array_equal(pk, pkq)
        eps_k, eps_kq, om, g2 = oracle.interpolate(H_R, D_R, g, R, np.ones(3), R, np.ones(3), [k, 0, 0], [q, 0, 0])
        np.testing.assert_allclose(eps_k[0], ek[pk], atol=1e-15)
        np.testing.assert_allclose(eps_kq[0, 0], ekq[pkq], atol=1e-15)
        ref = np.abs(gt0[:, pk][:, :, pkq]) ** 2 / (2 * np.sqrt(2.0))
        np.testing.assert_allclose(g2[0, 0], ref, rtol=1e-13)
    assert differing >= 2  # the band order at k and k+q really differs, so m <-> n mix-ups would show


def test_two_band_closed_form_eigenvectors_pin_conjugation():
    """Pin (closed form): Nb = 2, H(k) = [[0, h],[h*, 0]], h = t e^{2 pi i k}: eigenvalues -+|t| with
    eigenvectors (1, -+e^{-i theta_k})/sqrt(2), theta_k = arg t + 2 pi k.  g = V_{k+q}^dagger g~ V_k is then
    known in closed form; using U^T, swapping k <-> k+q or m' <-> n' changes |g|^2."""
    t = 0.8 * np.exp(0.6j)
    R = np.array([[-1, 0, 0], [0, 0, 0], [1, 0, 0]], dtype=np.int32)
    H_R = np.zeros((3, 2, 2), dtype=np.complex128)  # [ir][j][i]
    H_R[2][1][0] = t  # H(R=+1)[i=0, j=1] = t
    H_R[0][0][1] = np.conj(t)  # H(R=-1) = H(+1)^dagger
    D_R = np.array([0.0, 3.0, 0.0], dtype=np.complex128).reshape(3, 1, 1)
    gt0 = crandn(1, 2, 2)  # [nu][n'][m']
    g = np.zeros((3, 1, 3, 2, 2), dtype=np.complex128)
    g[1, :, 1] = gt0

    def V(kk):
        th = np.angle(t) + 2 * np.pi * kk
        return np.array([[1, 1], [-np.exp(-1j * th), np.exp(-1j * th)]]) / np.sqrt(2)

    for k, q in [(0.13, 0.29), (0.7, 0.55)]:
        eps_k, eps_kq, om, g2 = oracle.interpolate(H_R, D_R, g, R, np.ones(3), R, np.ones(3), [k, 0, 0], [q, 0, 0])
        np.testing.assert_allclose(eps_k[0], [-abs(t), abs(t)], atol=1e-15)
        Gm = gt0[0].T  # mathematical matrix [m', n']
        ref = V(k + q).conj().T @ Gm @ V(k) / np.sqrt(2 * np.sqrt(3.0))  # [m, n]
        np.testing.assert_allclose(g2[0, 0, 0], (np.abs(ref) ** 2).T, rtol=1e-12)
        wrong = V(k).conj().T @ Gm @ V(k + q) / np.sqrt(2 * np.sqrt(3.0))
        assert np.abs(np.abs(wrong) ** 2 - np.abs(ref) ** 2).max() > 1e-3


def test_mode_rotation_closed_form_two_modes():
    """Pin (closed form): Nm = 2, D(q) = [[a, b e^{2 pi i q}],[c.c., a]]: omega^2 = a -+ |b|, eigenvectors
    (1, -+e^{-i theta_q})/sqrt(2); g^_nu = sum_ka g~_ka e[ka,nu]/sqrt(2 omega_nu) (no conjugate on e)."""
    a, b = 5.0, 1.2 * np.exp(-0.4j)
    R = np.array([[-1, 0, 0], [0, 0, 0], [1, 0, 0]], dtype=np.int32)
    D_R = np.zeros((3, 2, 2), dtype=np.complex128)
    D_R[1] = a * np.eye(2)
    D_R[2][1][0] = b
    D_R[0][0][1] = np.conj(b)
    H_R = np.array([0.0, 1.0, 0.0], dtype=np.complex128).reshape(3, 1, 1)
    gt0 = crandn(2, 1, 1)
    g = np.zeros((3, 2, 3, 1, 1), dtype=np.complex128)
    g[1, :, 1] = gt0
    for q in (0.21, 0.66):
        th = np.angle(b) + 2 * np.pi * q
        e = np.array([[1, 1], [-np.exp(-1j * th), np.exp(-1j * th)]]) / np.sqrt(2)  # [ka, nu]
        om_ref = np.sqrt([a - abs(b), a + abs(b)])
        _, _, om, g2 = oracle.interpolate(H_R, D_R, g, R, np.ones(3), R, np.ones(3), [0.3, 0, 0], [q, 0, 0])
        np.testing.assert_allclose(om[0], om_ref, atol=1e-14)
        ref = np.abs(gt0[:, 0, 0] @ e) ** 2 / (2 * om_ref)
        np.testing.assert_allclose(g2[0, 0, :, 0, 0], ref, rtol=1e-12)


def test_unitarity_sum_rules():
    """Pins (invariants): sum_mn |g_mn nu|^2 = sum_m'n' |g^_m'n' nu|^2 (U unitary) and
    sum_nu 2 omega_nu |g_mn nu|^2 = sum_ka |(U^dagger g~ U)_mn ka|^2 (e unitary)."""
    nb, nm = 4, 3
    gt = crandn(nm, nb, nb)
    Uk, Ukq, e = random_unitary_cm(nb), random_unitary_cm(nb), random_unitary_cm(nm)
    om = np.array([0.5, 1.0, 2.5])
    gh = oracle.mode_rotate(gt, e, om)
    g = oracle.band_rotate(gh, Ukq, Uk)
    np.testing.assert_allclose((np.abs(g) ** 2).sum(axis=(1, 2)), (np.abs(gh) ** 2).sum(axis=(1, 2)), rtol=1e-13)
    rot_only = oracle.band_rotate(gt, Ukq, Uk)
    lhs = (2 * om[:, None, None] * np.abs(g) ** 2).sum(axis=0)
    np.testing.assert_allclose(lhs, (np.abs(rot_only) ** 2).sum(axis=0), rtol=1e-13)


def test_omega_min_cutoff_zeroes_modes():
    gt = crandn(2, 2, 2)
    gh = oracle.mode_rotate(gt, np.eye(2, dtype=np.complex128), np.array([1e-9, 1.0]), omega_min=1e-6)
    assert np.all(gh[0] == 0) and np.all(gh[1] != 0)


def test_bruteforce_eq7_equals_nested_loops():
    """Pin (brute force: single-loop Eq. 7 == nested Eqs. 9 + 10) on a tiny input,
    with U, e random unitaries that do not come from the oracle's eigensolver."""
    nb, nm = 2, 3
    Re = np.array([[0, 0, 0], [1, 0, -1], [-1, 2, 0], [0, -1, 1], [2, 1, 1]], dtype=np.int32)
    Rp = np.array([[0, 0, 0], [-1, 0, 0], [0, 1, 1], [1, -1, 0], [0, 0, 2]], dtype=np.int32)
    w_e, w_p = rng.random(5) + 0.5, rng.random(5) + 0.5
    g = crandn(5, nm, 5, nb, nb)
    Uk, Ukq, e = random_unitary_cm(nb), random_unitary_cm(nb), random_unitary_cm(nm)
    om = np.array([0.7, 1.1, 1.9])
    k, q = np.array([0.11, 0.52, 0.93]), np.array([0.37, 0.08, 0.61])
    direct = oracle.eq7_direct(g, Re, w_e, Rp, w_p, Ukq, Uk, e, om, k, q)
    gt = oracle.re_to_k(oracle.rp_to_q(g, Rp, w_p, q), Re, w_e, k)
    nested = oracle.band_rotate(oracle.mode_rotate(gt, e, om), Ukq, Uk)
    np.testing.assert_allclose(nested, direct, rtol=0, atol=1e-13 * np.abs(direct).max())


def test_gauge_invariance_of_block_sums():
    """Pin (invariant, [reading G10]): column phases and a unitary mixing inside a degenerate pair leave the
    block-summed |g|^2 unchanged."""
    nb, nm = 4, 3
    gt = crandn(nm, nb, nb)
    Uk, Ukq, e = random_unitary_cm(nb), random_unitary_cm(nb), random_unitary_cm(nm)
    om = np.array([0.5, 1.0, 1.0])  # modes 1,2 degenerate
    eps_k = np.array([-1.0, 0.2, 0.2, 3.0])  # bands 1,2 degenerate at k
    eps_kq = np.array([-2.0, -1.0, 0.0, 1.0])
    g2a = np.abs(oracle.band_rotate(oracle.mode_rotate(gt, e, om), Ukq, Uk)) ** 2
    ph = np.exp(2j * np.pi * rng.random(nb))
    Uk2 = Uk * ph[:, None]  # column-major storage [col][row]: scale each column
    W = cm(random_unitary_cm(2))
    Uk2m = cm(Uk2).copy()
    Uk2m[:, 1:3] = Uk2m[:, 1:3] @ W
    e2m = cm(e).copy()
    e2m[:, 1:3] = e2m[:, 1:3] @ cm(random_unitary_cm(2))
    Ukq2 = Ukq * np.exp(2j * np.pi * rng.random(nb))[:, None]
    g2b = np.abs(oracle.band_rotate(oracle.mode_rotate(gt, np.ascontiguousarray(e2m.T), om), Ukq2,
                                    np.ascontiguousarray(Uk2m.T))) ** 2
    assert np.abs(g2a - g2b).max() > 1e-3  # individual elements do change
    sa = oracle.block_sum_g2(g2a, eps_kq, eps_k, om)
    sb = oracle.block_sum_g2(g2b, eps_kq, eps_k, om)
    assert sa.shape == (2, 3, 4)
    np.testing.assert_allclose(sa, sb, rtol=1e-12)


def test_degenerate_repeated_block_through_whole_path():
    """A deliberately degenerate H (two identical 2x2 blocks): eigenvalues come in exact pairs, and the
    block-summed |g|^2 is invariant under a basis change inside the repeated block."""
    R = np.array([[-1, 0, 0], [0, 0, 0], [1, 0, 0]], dtype=np.int32)
    blk0 = np.array([[0.2, 0.5 + 0.1j], [0.5 - 0.1j, -0.3]])
    blk1 = 0.3 * crandn(2, 2)
    Z = np.zeros((2, 2))
    H0 = np.block([[blk0, Z], [Z, blk0]])
    H1 = np.block([[blk1, Z], [Z, blk1]])
    H_R = np.stack([H1.conj().T.T, H0.T, H1.T]).astype(np.complex128)  # storage [j][i] = transpose
    H_R[0] = np.ascontiguousarray(H1.conj().T.T)
    D_R = np.array([0.1, 2.0, 0.1], dtype=np.complex128).reshape(3, 1, 1)
    g = 0.3 * crandn(3, 1, 3, 4, 4)
    k, q = [0.17, 0, 0], [0.41, 0, 0]
    eps_k, eps_kq, om, g2 = oracle.interpolate(H_R, D_R, g, R, np.ones(3), R, np.ones(3), k, q)
    assert abs(eps_k[0, 0] - eps_k[0, 1]) < 1e-13 and abs(eps_k[0, 2] - eps_k[0, 3]) < 1e-13
    # same physics in a rotated Wannier basis that mixes the two copies: W = Q (x) 1_2
    Q = cm(random_unitary_cm(2))
    W = np.kron(Q, np.eye(2))
    Hm = cm(H_R)
    H_R2 = np.ascontiguousarray(cm(W.conj().T @ Hm @ W))
    gm = cm(g)  # [..., m', n']
    g_rot = np.ascontiguousarray(cm(W.conj().T @ gm @ W))
    _, _, _, g2r = oracle.interpolate(H_R2, D_R, g_rot, R, np.ones(3), R, np.ones(3), k, q)
    sa = oracle.block_sum_g2(g2[0, 0], eps_kq[0, 0], eps_k[0], om[0])
    sb = oracle.block_sum_g2(g2r[0, 0], eps_kq[0, 0], eps_k[0], om[0])
    assert sa.shape == (1, 2, 2)
    np.testing.assert_allclose(sa, sb, rtol=1e-11)


def test_linearity_in_g():
    """Pin (invariant): g_RR -> alpha g_RR  =>  |g|^2 -> |alpha|^2 |g|^2."""
    import synth

    w = synth.make_custom("t", 3, 3, (1, 0, 0), 1.0, 0.1, 1.0, (2, 1, 1), ("grid", (2, 1, 1)), seed=5)
    g = w.g_full()
    a = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    alpha = 0.3 - 1.7j
    b = oracle.interpolate(w.H_R, w.D_R, alpha * g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    np.testing.assert_allclose(b[3], abs(alpha) ** 2 * a[3], rtol=1e-12)
    np.testing.assert_array_equal(a[0], b[0])


def test_interpolate_list_driver_matches_stagewise_calls():
    """The list driver (C-ABI mirror) is the stage functions chained in the paper's nested order."""
    import synth

    w = synth.make_custom("t", 3, 3, (1, 1, 0), 1.0, 0.1, 1.0, (2, 2, 1), ("random", 2, 3), seed=9)
    g = w.g_full()
    eps_k, eps_kq, om, g2 = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
    for iq, q in enumerate(w.q_list):
        e, omega = oracle.phonon(w.D_R, w.Rp, w.w_p, q)
        np.testing.assert_array_equal(omega, om[iq])
        g1 = oracle.rp_to_q(g, w.Rp, w.w_p, q)
        for ik, k in enumerate(w.k_list):
            p = oracle.pair(g1, w.H_R, w.Re, w.w_e, e, omega, k, q)
            np.testing.assert_array_equal(p[0], g2[iq, ik])
            np.testing.assert_array_equal(p[1], eps_k[ik])
            np.testing.assert_array_equal(p[2], eps_kq[iq, ik])


def test_synthetic_Dq_is_positive_definite_and_kq_fold_is_harmless():
    """Config-0 style inputs: D(q) > 0 (diagonal shift), and folding k+q onto the grid changes nothing [G9]."""
    import synth

    w = synth.make_config(0)
    for q in w.q_list[::7]:
        _, om = oracle.phonon(w.D_R, w.Rp, w.w_p, q)
        assert om.min() > 0.5
    k, q = w.k_list[37], w.q_list[50]
    a = oracle.interp_operator(w.H_R, w.Re, w.w_e, k + q)
    b = oracle.interp_operator(w.H_R, w.Re, w.w_e, w.k_list[w.kq_map[50, 37]])
    np.testing.assert_allclose(a, b, rtol=0, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# Numbers the paper prints.
# ---------------------------------------------------------------------------------------------
def test_table3_sizes_as_printed():
    """Pin (printed values, Table III): 16 Nb^2 Nm Ne Np bytes, printed in GiB."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table3_sizes.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 11
    for width, nb, nm, ne, np_, printed in rows:
        gib = oracle.g_bytes(float(nb), float(nm), float(ne), float(np_)) / 2**30
        digits = len(printed.split(".")[1]) if "." in printed else 0
        assert abs(gib - float(printed)) <= 0.5 * 10 ** (-digits) + 1e-9, (width, gib, printed)


def test_silicon_size_and_eq12_ratio_as_printed():
    """Pins (printed values): silicon g is "0.4 GB"; N^NL/N^SL ~ 1/93 for Nk >> Np
    (Eq. 12), evaluated from the multiplication counts of Eqs. 8 and 11."""
    nb, nm, ne, np_, denom, gb = [float(x) for x in
                                  [l for l in open(os.path.join(GOLDEN, "si_eq12.txt")) if not l.startswith("#")][0].split()]
    assert round(oracle.g_bytes(nb, nm, ne, np_) / 1e9, 1) == gb or round(oracle.g_bytes(nb, nm, ne, np_) / 2**30, 1) == gb - 0.1
    nk = nq = 96.0**3
    ratio = oracle.nmul_nested_loop(nb, nm, ne, np_, nk, nq) / oracle.nmul_single_loop(nb, nm, ne, np_, nk, nq)
    eq12 = 1 / nk + (1 / np_) * (1 + 2 / ne + nm / ne)
    assert abs(ratio - eq12) / eq12 < 0.02  # Eq. 12 drops the small terms of Eq. 8 ("approximately")
    assert abs(ratio * denom - 1) < 0.02


# ---------------------------------------------------------------------------------------------
# Gauge part of Eq. 6 (Bloch -> Wannier), the step before the hot path.
# ---------------------------------------------------------------------------------------------
def test_eq6_unrotate_matches_matrix_algebra_and_inverts_the_forward_rotations():
    """Pin (textbook matrix algebra + invariant): PAPER.md:L78-80 with reading G4 gives, per mode,
    g~_nu = V_{k+q} g_nu V_k^dagger, then g~_ka = sum_nu g~_nu sqrt(2 omega_nu) conj(e[ka,nu]) -- written here with
    numpy matmul on mathematical matrices; and it must undo oracle_mode_rotate + oracle_band_rotate (both pinned
    above), including which index carries k+q and where the conjugates sit."""
    nb, nm = 4, 3
    Ukq, Uk, e = random_unitary_cm(nb), random_unitary_cm(nb), random_unitary_cm(nm)
    omega = np.array([0.7, 1.3, 2.1])
    g = crandn(nm, nb, nb)  # [nu][n][m]
    got = oracle.eq6_unrotate(g, Ukq, Uk, e, omega)
    Vkq, Vk, E = cm(Ukq), cm(Uk), cm(e)  # mathematical matrices [row, col]
    gw = np.stack([Vkq @ g[nu].T @ Vk.conj().T for nu in range(nm)])  # [nu][m'][n']
    ref = np.einsum("vab,kv->kab", gw * np.sqrt(2 * omega)[:, None, None], E.conj())  # [ka][m'][n']
    np.testing.assert_allclose(got, np.swapaxes(ref, 1, 2), rtol=0, atol=1e-14)
    # inverse of the forward rotations
    gt = crandn(nm, nb, nb)  # [ka][n'][m']
    fwd = oracle.band_rotate(oracle.mode_rotate(gt, e, omega), Ukq, Uk)
    np.testing.assert_allclose(oracle.eq6_unrotate(fwd, Ukq, Uk, e, omega), gt, rtol=0, atol=1e-13)
    # transposing a U or swapping k <-> k+q is detected
    assert np.abs(oracle.eq6_unrotate(fwd, Uk, Ukq, e, omega) - gt).max() > 1e-2


# ---------------------------------------------------------------------------------------------
# Energy-window pre-screening.
# ---------------------------------------------------------------------------------------------
def test_window_mask_hand_example_and_bruteforce():
    """Pin (worked example + brute force): a pair is kept iff some band of eps_k AND some band of eps_{k+q} lies in
    the closed window.  Hand example first, then random spectra against the one-line numpy statement."""
    eps_k = np.array([[-1.0, 0.1, 2.0], [0.5, 0.6, 0.7], [-3.0, -2.0, 5.0]])            # k0 in, k1 out, k2 out for [0, 0.3]
    eps_kq = np.array([[[0.3, 9.0, 9.0], [0.0, 0.0, 0.0], [0.2, 0.2, 0.2]],              # q0: kq in / in / in
                       [[0.31, 9.0, 9.0], [0.1, 9.0, 9.0], [-0.01, 0.4, 1.0]]])          # q1: out / in / out
    got = oracle.window_mask(eps_k, eps_kq, 0.0, 0.3)
    np.testing.assert_array_equal(got, [[1, 0, 0], [0, 0, 0]])
    got = oracle.window_mask(eps_k, eps_kq, 0.0, 0.5)                                     # edge value 0.5 is inside
    np.testing.assert_array_equal(got, [[1, 1, 0], [1, 1, 0]])
    ek, ekq = rng.uniform(-1, 1, (7, 4)), rng.uniform(-1, 1, (5, 7, 4))
    ref = (((ek >= -0.2) & (ek <= 0.1)).any(-1)[None, :] & ((ekq >= -0.2) & (ekq <= 0.1)).any(-1)).astype(np.uint8)
    np.testing.assert_array_equal(oracle.window_mask(ek, ekq, -0.2, 0.1), ref)
    assert 0 < ref.sum() < ref.size


# ---------------------------------------------------------------------------------------------
# NEXT-4 consumer: Im Sigma_nk accumulator (reading G18; the paper names the consumer, not its formula)
# ---------------------------------------------------------------------------------------------
def test_selfenergy_energy_integral_linearity_and_zero_temperature_selection():
    """Pins that do not retype the formula:
    (1) each broadened delta integrates to one, so the integral of Im Sigma over the initial-state energy is
        pi w |g|^2 (2 n_B + 1) -- the Fermi factors cancel between absorption and emission;
    (2) linear in |g|^2 and in w_q, additive over q, accumulating into `out`;
    (3) T -> 0: an electron above a filled sea can only EMIT (final energy e - w, which must be empty), never absorb;
        an initial state inside the sea only scatters into the empty state reached by ABSORPTION if that is what
        energy conservation selects -- fixes which delta carries which occupation factor and the sign of w."""
    nb, nm = 1, 1
    w, e2, mu, kT, sigma, g2v, wq = 0.05, 0.3, 0.1, 0.02, 0.004, 0.7, 0.25
    es = np.linspace(e2 - 0.2, e2 + 0.2, 4001)            # the "k-points": a fine grid of initial-state energies
    g2 = np.full((1, len(es), nm, nb, nb), g2v)
    out = oracle.selfenergy_accumulate(g2, es[:, None], np.full((1, len(es), 1), e2), [[w]], [wq], mu, kT, sigma)
    nB = 1.0 / np.expm1(w / kT)
    integral = np.sum(out[:, 0]) * (es[1] - es[0])    # peaks are far inside the grid; rectangle rule on smooth Gaussians
    assert abs(integral - np.pi * wq * g2v * (2 * nB + 1)) < 1e-9 * integral
    # the two peaks sit at e2 - w (absorption: e + w = e2) and e2 + w (emission: e - w = e2)
    below, above = es < e2, es > e2
    peaks = [es[below][np.argmax(out[below, 0])], es[above][np.argmax(out[above, 0])]]
    np.testing.assert_allclose(peaks, [e2 - w, e2 + w], atol=2e-4)
    # (2) linearity / additivity / accumulation
    out2 = oracle.selfenergy_accumulate(np.concatenate([g2, 3 * g2]), es[:, None], np.full((2, len(es), 1), e2),
                                        [[w], [w]], [wq, 2 * wq], mu, kT, sigma, out=out.copy())
    np.testing.assert_allclose(out2, out * (1 + 1 + 6), rtol=1e-12, atol=1e-300)   # atol: denormal tails of the Gaussians
    # (3) zero temperature: final state e2 EMPTY (above mu): only the emission peak (e = e2 + w) survives, weight 1
    cold = oracle.selfenergy_accumulate(g2, es[:, None], np.full((1, len(es), 1), e2), [[w]], [1.0], mu, 1e-5, sigma)
    lo, hi = es < e2, es > e2
    assert cold[lo, 0].max() < 1e-12 * cold[hi, 0].max()
    assert abs(np.sum(cold[hi, 0]) * (es[1] - es[0]) - np.pi * g2v) < 1e-9
    # final state FILLED (below mu): only the absorption peak (e = e2 - w) survives
    cold2 = oracle.selfenergy_accumulate(g2, es[:, None], np.full((1, len(es), 1), e2), [[w]], [1.0], e2 + 1.0, 1e-5, sigma)
    assert cold2[hi, 0].max() < 1e-12 * cold2[lo, 0].max()
    assert abs(np.sum(cold2[lo, 0]) * (es[1] - es[0]) - np.pi * g2v) < 1e-9
    # modes with omega <= 0 do not contribute
    assert not oracle.selfenergy_accumulate(g2, es[:, None], np.full((1, len(es), 1), e2), [[-0.01]], None, mu, kT, sigma).any()
