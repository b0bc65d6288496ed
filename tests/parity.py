"""Tolerances and comparison helpers shared by the GPU parity tests, smoke() and bench.py.

Tolerances are BASELINE.json north_star's ("eigenvalues and omega to 1e-10 relative, |g|^2 to 1e-9 relative,
summed over degenerate subspaces (gap < 1e-6 eV)") made well defined as in DESIGN.md reading G11:
  eigenvalues / omega : |a-b| <= 1e-10 * max(|b|, 1e-3 * max|spectrum|)
  |g|^2 block sums    : |a-b| <= 1e-9 * |b| + 1e-11 * max over the (k,q) block of |b|
"""
import numpy as np

import oracle

EIG_RTOL = 1e-10
G2_RTOL = 1e-9
G2_FLOOR = 1e-11
DEGEN_GAP = 1e-6


def eig_close(a, b):
    a, b = np.asarray(a), np.asarray(b)
    scale = np.maximum(np.abs(b), 1e-3 * np.abs(b).max(axis=-1, keepdims=True))
    err = np.abs(a - b) / scale
    return err.max(), bool((err <= EIG_RTOL).all())


def g2_pair_close(g2_a, g2_b, eps_kq, eps_k, omega):
    """Compare one (k,q) block [nu][n][m] after summing over degenerate subspaces taken from the reference spectra."""
    sa = oracle.block_sum_g2(np.asarray(g2_a), eps_kq, eps_k, omega, DEGEN_GAP)
    sb = oracle.block_sum_g2(np.asarray(g2_b), eps_kq, eps_k, omega, DEGEN_GAP)
    tol = G2_RTOL * np.abs(sb) + G2_FLOOR * np.abs(sb).max()
    err = np.abs(sa - sb)
    return float((err / np.maximum(tol, 1e-300)).max()), bool((err <= tol).all())


def assert_path_close(gpu, ref, pairs=None):
    """gpu/ref = (eps_k [nk,Nb], eps_kq [nq,nk,Nb], omega [nq,Nm], g2 [nq,nk,Nm,Nb,Nb]); pairs = iterable of (iq, ik)."""
    eps_k, eps_kq, om, g2 = [np.asarray(x) for x in gpu]
    r_eps_k, r_eps_kq, r_om, r_g2 = ref
    e, ok = eig_close(eps_k, r_eps_k)
    assert ok, f"eps_k mismatch: max scaled err {e:.3e}"
    e, ok = eig_close(om, r_om)
    assert ok, f"omega mismatch: max scaled err {e:.3e}"
    if eps_kq is not None and r_eps_kq is not None:
        e, ok = eig_close(eps_kq, r_eps_kq)
        assert ok, f"eps_kq mismatch: max scaled err {e:.3e}"
    nq, nk = g2.shape[:2]
    if pairs is None:
        pairs = [(iq, ik) for iq in range(nq) for ik in range(nk)]
    worst = 0.0
    for iq, ik in pairs:
        w, ok = g2_pair_close(g2[iq, ik], r_g2[iq, ik], r_eps_kq[iq, ik], r_eps_k[ik], r_om[iq])
        worst = max(worst, w)
        assert ok, f"|g|^2 mismatch at (iq={iq}, ik={ik}): {w:.3f} x tolerance"
    return worst
