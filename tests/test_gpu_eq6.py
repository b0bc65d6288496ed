"""GPU parity tests of Eq. 6, the Bloch -> Wannier step before the hot path:
epw_eq6_unrotate and epw_wannier_from_bloch against oracle/, and a device-only round trip Eq. 6 -> Eq. 7."""
import numpy as np
import pytest

import oracle
import synth
from test_gpu_parity import crandn, dev, epw, zdev, znp  # noqa: F401  (epw is the module fixture)

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def unitary_cm(n, rng):
    q, _ = np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))
    return np.ascontiguousarray(q.T)  # column-major storage [col][row]


def grid(N):
    ax = [np.arange(n) / n for n in N]
    return np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)


def residue_vectors(N, shift):
    ax = [np.arange(n) - s for n, s in zip(N, shift)]
    return np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.int32)


@pytest.mark.parametrize("nb,nm,nkc,nqc", [(2, 3, 5, 3), (8, 6, 9, 4), (11, 9, 3, 2), (1, 1, 1, 1), (20, 7, 2, 2)])
def test_eq6_unrotate(epw, nb, nm, nkc, nqc):
    rng = np.random.default_rng(100 + nb)
    g = crandn(nqc, nkc, nm, nb, nb)
    Uk = np.stack([unitary_cm(nb, rng) for _ in range(nkc)])
    Ukq = np.stack([[unitary_cm(nb, rng) for _ in range(nkc)] for _ in range(nqc)])
    e = np.stack([unitary_cm(nm, rng) for _ in range(nqc)])
    om = rng.uniform(0.3, 2.0, size=(nqc, nm))
    out = torch.empty((nqc, nkc, nm, nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_eq6_unrotate(zdev(g), zdev(Uk), zdev(Ukq), zdev(e), dev(om), nb, nm, nkc, nqc, out)
    got = znp(out)
    for iq in range(nqc):
        for ik in range(nkc):
            ref = oracle.eq6_unrotate(g[iq, ik], Ukq[iq, ik], Uk[ik], e[iq], om[iq])
            assert np.abs(got[iq, ik] - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("Nk,Nq,nb,nm", [((3, 2, 4), (2, 3, 1), 2, 3), ((4, 4, 1), (2, 2, 1), 5, 3), ((5, 1, 1), (3, 1, 1), 8, 6)])
def test_wannier_from_bloch_matches_oracle(epw, Nk, Nq, nb, nm):
    """Both inverse Fourier sums against the oracle's Eq. 6 (itself pinned by numpy.fft), ragged tiles everywhere."""
    Re = residue_vectors(Nk, tuple(n // 2 for n in Nk))
    Rp = residue_vectors(Nq, tuple(n // 2 for n in Nq))
    kc, qc = grid(Nk), grid(Nq)
    G = crandn(len(qc), len(kc), nm, nb, nb)
    ref = oracle.eq6_wannier_from_bloch(G, kc, qc, Re, Rp)
    out = torch.empty((len(Rp), nm, len(Re), nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_wannier_from_bloch(zdev(G), dev(kc), len(kc), dev(qc), len(qc), dev(Re), len(Re), dev(Rp), len(Rp), nb, nm, out)
    got = znp(out)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


def test_wannier_from_bloch_non_grid_points_and_truncated_lists(epw):
    """k', q' need not be grids and the R lists need not be complete: the sums are plain (parity with the oracle)."""
    nb, nm = 3, 2
    kc, qc = rng_points(7), rng_points(5)
    Re = np.array([[0, 0, 0], [1, 0, -1], [-2, 1, 0], [0, 3, 1]], dtype=np.int32)
    Rp = np.array([[0, 0, 0], [0, -1, 2], [1, 1, 1]], dtype=np.int32)
    G = crandn(len(qc), len(kc), nm, nb, nb)
    ref = oracle.eq6_wannier_from_bloch(G, kc, qc, Re, Rp)
    out = torch.empty((len(Rp), nm, len(Re), nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_wannier_from_bloch(zdev(G), dev(kc), len(kc), dev(qc), len(qc), dev(Re), len(Re), dev(Rp), len(Rp), nb, nm, out)
    assert np.abs(znp(out) - ref).max() <= 1e-13 * np.abs(ref).max()


def rng_points(n):
    return np.random.default_rng(n).uniform(0, 1, size=(n, 3))


def test_device_round_trip_eq6_then_eq7(epw):
    """Eq. 6 and Eq. 7 are inverse generalized Fourier transforms: coarse-grid data pushed through
    epw_wannier_from_bloch and interpolated back AT THE COARSE POINTS by the hot path must reproduce itself.  H(R), D(R)
    are R = 0 only and diagonal with distinct entries, so U = e = 1 and |g|^2 = |G|^2 / (2 omega) element by element
    (the diagonal-operator pin of the oracle, here device to device); everything stays on the GPU."""
    Nk, Nq, nb, nm = (4, 3, 2), (2, 3, 2), 4, 3
    Re = residue_vectors(Nk, (2, 1, 1))
    Rp = residue_vectors(Nq, (1, 1, 1))
    kc, qc = grid(Nk), grid(Nq)
    G = crandn(len(qc), len(kc), nm, nb, nb)
    g_rr = torch.empty((len(Rp), nm, len(Re), nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_wannier_from_bloch(zdev(G), dev(kc), len(kc), dev(qc), len(qc), dev(Re), len(Re), dev(Rp), len(Rp), nb, nm, g_rr)
    dH, dD = np.array([-1.0, 0.2, 0.9, 2.5]), np.array([1.0, 2.0, 4.0])
    H_R = np.zeros((len(Re), nb, nb), dtype=np.complex128)
    D_R = np.zeros((len(Rp), nm, nm), dtype=np.complex128)
    H_R[[i for i, r in enumerate(Re) if not r.any()][0]] = np.diag(dH)
    D_R[[i for i, r in enumerate(Rp) if not r.any()][0]] = np.diag(dD)
    h = epw.EpwInterp(nb, nm, len(Re), len(Rp))
    try:
        epw.epw_interp_set_wannier_operators(h.h, zdev(H_R), zdev(D_R), g_rr, dev(Re), dev(np.ones(len(Re))), dev(Rp),
                                             dev(np.ones(len(Rp))), 1)
        for use_grid in (True, False):
            if use_grid:
                eps_k, eps_kq, om, g2 = h.interpolate_grid(Nk, dev(qc))
            else:
                eps_k, eps_kq, om, g2 = h.interpolate(dev(kc), dev(qc))
            epw.epw_interp_sync(h.h)
            np.testing.assert_allclose(om.cpu().numpy(), np.tile(np.sqrt(dD), (len(qc), 1)), rtol=1e-13)
            np.testing.assert_allclose(eps_k.cpu().numpy(), np.tile(dH, (len(kc), 1)), atol=1e-13)
            ref = np.abs(G) ** 2 / (2 * np.sqrt(dD))[None, None, :, None, None]
            np.testing.assert_allclose(g2.cpu().numpy(), ref, rtol=1e-11, atol=1e-13 * ref.max())
    finally:
        h.close()


def test_eq6_full_gauge_round_trip_against_the_path(epw):
    """Bloch-gauge coarse data: run the path on a random workload at coarse points, take its complex g (oracle) in the
    Bloch gauge, and check that unrotate (device) + inverse sums (device) give back the workload's g(Re,Rp)."""
    Nk, Nq = (3, 3, 1), (3, 3, 1)
    w = synth.make_custom("rt", 3, 3, (1, 1, 0), 1.0, 0.1, 1.0, Nk, ("grid", Nq), seed=41)
    g_rr = w.g_full()
    kc, qc = w.k_list, w.q_list
    nb, nm = w.nbnd, w.nmodes
    gB = np.empty((len(qc), len(kc), nm, nb, nb), dtype=np.complex128)
    Uk = np.empty((len(kc), nb, nb), dtype=np.complex128)
    Ukq = np.empty((len(qc), len(kc), nb, nb), dtype=np.complex128)
    e = np.empty((len(qc), nm, nm), dtype=np.complex128)
    om = np.empty((len(qc), nm))
    for iq, q in enumerate(qc):
        e[iq], om[iq] = oracle.phonon(w.D_R, w.Rp, w.w_p, q)
        g1 = oracle.rp_to_q(g_rr, w.Rp, w.w_p, q)
        for ik, k in enumerate(kc):
            _, Uk[ik], _ = oracle.eigh_jacobi(oracle.interp_operator(w.H_R, w.Re, w.w_e, k))
            _, Ukq[iq, ik], _ = oracle.eigh_jacobi(oracle.interp_operator(w.H_R, w.Re, w.w_e, k + q))
            gt = oracle.re_to_k(g1, w.Re, w.w_e, k)
            gB[iq, ik] = oracle.band_rotate(oracle.mode_rotate(gt, e[iq], om[iq]), Ukq[iq, ik], Uk[ik])
    gt_d = torch.empty((len(qc), len(kc), nm, nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_eq6_unrotate(zdev(gB), zdev(Uk), zdev(Ukq), zdev(e), dev(om), nb, nm, len(kc), len(qc), gt_d)
    out = torch.empty((w.np_, nm, w.ne, nb, nb, 2), dtype=torch.float64, device="cuda")
    epw.epw_wannier_from_bloch(gt_d, dev(kc), len(kc), dev(qc), len(qc), dev(w.Re), w.ne, dev(w.Rp), w.np_, nb, nm, out)
    # Re = Rp = all |n_i| <= 1 = one vector per residue class of the 3x3x1 grids: Eq. 6 inverts Eq. 7 exactly
    assert np.abs(znp(out) - g_rr).max() <= 1e-12 * np.abs(g_rr).max()
