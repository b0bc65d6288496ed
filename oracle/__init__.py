"""ctypes binding of the CPU oracle (oracle/epw_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
imports nothing from paper_2603_10295_b200 and the CUDA library imports nothing
from here.

Every function takes/returns numpy arrays in the conventions of the C file
(matrices column-major, eigenvectors as columns; see the header of
epw_oracle.c).  Numpy views used here: a column-major n x n matrix A[i + n*j]
is the C-ordered array M[j, i]; helper `cm(M)` returns the mathematical matrix
(M.T) for use in test formulas.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "epw_oracle.c")
_LIB = os.path.join(_HERE, "libepw_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99, OpenMP only over independent k)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-std=gnu99", "-O2", "-fcx-limited-range", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i, i64, f64, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        L.oracle_phase.argtypes = [vp, vp]
        L.oracle_phase.restype = f64
        L.oracle_rp_to_q.argtypes = [i, i, i, i, vp, vp, vp, vp, vp]
        L.oracle_re_to_k.argtypes = [i, i, i, vp, vp, vp, vp, vp]
        L.oracle_interp_operator.argtypes = [i, i, vp, vp, vp, vp, vp]
        L.oracle_eigh_jacobi.argtypes = [i, vp, vp, vp]
        L.oracle_eigh_jacobi.restype = i
        L.oracle_omega_from_lambda.argtypes = [i, vp, vp]
        L.oracle_mode_rotate.argtypes = [i, i, vp, vp, vp, f64, vp]
        L.oracle_band_rotate.argtypes = [i, i, vp, vp, vp, vp]
        L.oracle_pair.argtypes = [i, i, i, vp, vp, vp, vp, vp, vp, f64, vp, vp, vp, vp, vp, vp]
        L.oracle_pair.restype = i
        L.oracle_phonon.argtypes = [i, i, vp, vp, vp, vp, vp, vp]
        L.oracle_phonon.restype = i
        L.oracle_interpolate.argtypes = [i, i, i, i, vp, vp, vp, vp, vp, vp, vp, f64, vp, i64, vp, i64, vp, vp, vp, vp]
        L.oracle_interpolate.restype = i
        L.oracle_eq7_direct.argtypes = [i, i, i, i, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.oracle_eq6_wannier_from_bloch.argtypes = [i, i, i, i, vp, vp, i, vp, i, vp, vp, vp]
        L.oracle_eq6_unrotate.argtypes = [i, i, vp, vp, vp, vp, vp, vp]
        L.oracle_window_mask.argtypes = [i, i64, i64, vp, vp, f64, f64, vp]
        L.oracle_selfenergy_accumulate.argtypes = [i, i, i64, i64, vp, vp, vp, vp, vp, f64, f64, f64, vp]
        for name in ("oracle_g_bytes",):
            getattr(L, name).argtypes = [f64] * 4
            getattr(L, name).restype = f64
        for name in ("oracle_nmul_single_loop", "oracle_nmul_nested_loop"):
            getattr(L, name).argtypes = [f64] * 6
            getattr(L, name).restype = f64
        _lib = L
    return _lib


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def _p(a):
    return a.ctypes.data if a is not None else None


def cm(M: np.ndarray) -> np.ndarray:
    """Column-major storage M[j, i] -> mathematical matrix A[i, j] (also for stacks [..., j, i])."""
    return np.swapaxes(M, -1, -2)


def phase(x, R) -> float:
    x = _c(x, np.float64)
    R = _c(R, np.int32)
    return lib().oracle_phase(_p(x), _p(R))


def rp_to_q(g_RR, Rp, w_p, q) -> np.ndarray:
    """Eq. 9.  g_RR [Np][Nm][Ne][Nb][Nb] -> g(Re,q) [Nm][Ne][Nb][Nb]."""
    g_RR = _c(g_RR, np.complex128)
    np_, nm, ne, nb, _ = g_RR.shape
    Rp, w_p, q = _c(Rp, np.int32), _c(w_p, np.float64), _c(q, np.float64)
    out = np.empty((nm, ne, nb, nb), dtype=np.complex128)
    lib().oracle_rp_to_q(nb, nm, ne, np_, _p(g_RR), _p(Rp), _p(w_p), _p(q), _p(out))
    return out


def re_to_k(g1, Re, w_e, k) -> np.ndarray:
    """FT part of Eq. 10.  g(Re,q) [Nm][Ne][Nb][Nb] -> g~(k,q) [Nm][n'][m']."""
    g1 = _c(g1, np.complex128)
    nm, ne, nb, _ = g1.shape
    Re, w_e, k = _c(Re, np.int32), _c(w_e, np.float64), _c(k, np.float64)
    out = np.empty((nm, nb, nb), dtype=np.complex128)
    lib().oracle_re_to_k(nb, nm, ne, _p(g1), _p(Re), _p(w_e), _p(k), _p(out))
    return out


def interp_operator(Op_R, R, w, x) -> np.ndarray:
    """Op_R [NR][j][i] -> Op(x) [j][i] (column-major n x n)."""
    Op_R = _c(Op_R, np.complex128)
    nr, n, _ = Op_R.shape
    R, w, x = _c(R, np.int32), _c(w, np.float64), _c(x, np.float64)
    out = np.empty((n, n), dtype=np.complex128)
    lib().oracle_interp_operator(n, nr, _p(Op_R), _p(R), _p(w), _p(x), _p(out))
    return out


def eigh_jacobi(A_cm):
    """A_cm [j][i] column-major Hermitian -> (evals ascending [n], V_cm [col][row], sweeps)."""
    A_cm = _c(A_cm, np.complex128)
    n = A_cm.shape[0]
    ev = np.empty(n, dtype=np.float64)
    V = np.empty((n, n), dtype=np.complex128)
    sweeps = lib().oracle_eigh_jacobi(n, _p(A_cm), _p(ev), _p(V))
    return ev, V, sweeps


def omega_from_lambda(lam) -> np.ndarray:
    lam = _c(lam, np.float64)
    out = np.empty_like(lam)
    lib().oracle_omega_from_lambda(lam.shape[0], _p(lam), _p(out))
    return out


def mode_rotate(gt, e_cm, omega, omega_min=0.0) -> np.ndarray:
    gt = _c(gt, np.complex128)
    nm, nb, _ = gt.shape
    e_cm, omega = _c(e_cm, np.complex128), _c(omega, np.float64)
    out = np.empty_like(gt)
    lib().oracle_mode_rotate(nb, nm, _p(gt), _p(e_cm), _p(omega), omega_min, _p(out))
    return out


def band_rotate(gh, Ukq_cm, Uk_cm) -> np.ndarray:
    gh = _c(gh, np.complex128)
    nm, nb, _ = gh.shape
    Ukq_cm, Uk_cm = _c(Ukq_cm, np.complex128), _c(Uk_cm, np.complex128)
    out = np.empty_like(gh)
    lib().oracle_band_rotate(nb, nm, _p(gh), _p(Ukq_cm), _p(Uk_cm), _p(out))
    return out


def phonon(D_R, Rp, w_p, q):
    """D(q) eigen-system: (e_cm [nu][ka], omega [Nm])."""
    D_R = _c(D_R, np.complex128)
    np_, nm, _ = D_R.shape
    Rp, w_p, q = _c(Rp, np.int32), _c(w_p, np.float64), _c(q, np.float64)
    e = np.empty((nm, nm), dtype=np.complex128)
    om = np.empty(nm, dtype=np.float64)
    rc = lib().oracle_phonon(nm, np_, _p(D_R), _p(Rp), _p(w_p), _p(q), _p(e), _p(om))
    if rc:
        raise RuntimeError("oracle Jacobi did not converge (D(q))")
    return e, om


def pair(g1, H_R, Re, w_e, e_cm, omega, k, q, omega_min=0.0, want_g=False):
    """One (k,q) pair from g(Re,q): returns (g2 [nu][n][m], eps_k, eps_kq[, g complex])."""
    g1 = _c(g1, np.complex128)
    nm, ne, nb, _ = g1.shape
    H_R, Re, w_e = _c(H_R, np.complex128), _c(Re, np.int32), _c(w_e, np.float64)
    e_cm, omega, k, q = _c(e_cm, np.complex128), _c(omega, np.float64), _c(k, np.float64), _c(q, np.float64)
    g2 = np.empty((nm, nb, nb), dtype=np.float64)
    ek = np.empty(nb, dtype=np.float64)
    ekq = np.empty(nb, dtype=np.float64)
    g = np.empty((nm, nb, nb), dtype=np.complex128) if want_g else None
    rc = lib().oracle_pair(nb, nm, ne, _p(g1), _p(H_R), _p(Re), _p(w_e), _p(e_cm), _p(omega), omega_min, _p(k), _p(q),
                           _p(g2), _p(ek), _p(ekq), _p(g))
    if rc:
        raise RuntimeError("oracle Jacobi did not converge (H)")
    return (g2, ek, ekq, g) if want_g else (g2, ek, ekq)


def interpolate(H_R, D_R, g_RR, Re, w_e, Rp, w_p, k_list, q_list, omega_min=0.0, want_eps_kq=True):
    """Whole path on host arrays, mirroring the C ABI: (eps_k, eps_kq, omega_q, g2)."""
    H_R, D_R, g_RR = _c(H_R, np.complex128), _c(D_R, np.complex128), _c(g_RR, np.complex128)
    np_, nm, ne, nb, _ = g_RR.shape
    Re, w_e, Rp, w_p = _c(Re, np.int32), _c(w_e, np.float64), _c(Rp, np.int32), _c(w_p, np.float64)
    k_list, q_list = _c(k_list, np.float64).reshape(-1, 3), _c(q_list, np.float64).reshape(-1, 3)
    nk, nq = k_list.shape[0], q_list.shape[0]
    eps_k = np.empty((nk, nb), dtype=np.float64)
    eps_kq = np.empty((nq, nk, nb), dtype=np.float64) if want_eps_kq else None
    omega_q = np.empty((nq, nm), dtype=np.float64)
    g2 = np.empty((nq, nk, nm, nb, nb), dtype=np.float64)
    rc = lib().oracle_interpolate(nb, nm, ne, np_, _p(H_R), _p(D_R), _p(g_RR), _p(Re), _p(w_e), _p(Rp), _p(w_p),
                                  omega_min, _p(k_list), nk, _p(q_list), nq, _p(eps_k), _p(eps_kq), _p(omega_q), _p(g2))
    if rc:
        raise RuntimeError("oracle Jacobi did not converge")
    return eps_k, eps_kq, omega_q, g2


def eq7_direct(g_RR, Re, w_e, Rp, w_p, Ukq_cm, Uk_cm, e_cm, omega, k, q) -> np.ndarray:
    """Single-loop Eq. 7 for one pair (complex g [nu][n][m]); tiny inputs only."""
    g_RR = _c(g_RR, np.complex128)
    np_, nm, ne, nb, _ = g_RR.shape
    Re, w_e, Rp, w_p = _c(Re, np.int32), _c(w_e, np.float64), _c(Rp, np.int32), _c(w_p, np.float64)
    Ukq_cm, Uk_cm, e_cm = _c(Ukq_cm, np.complex128), _c(Uk_cm, np.complex128), _c(e_cm, np.complex128)
    omega, k, q = _c(omega, np.float64), _c(k, np.float64), _c(q, np.float64)
    out = np.empty((nm, nb, nb), dtype=np.complex128)
    lib().oracle_eq7_direct(nb, nm, ne, np_, _p(g_RR), _p(Re), _p(w_e), _p(Rp), _p(w_p), _p(Ukq_cm), _p(Uk_cm),
                            _p(e_cm), _p(omega), _p(k), _p(q), _p(out))
    return out


def eq6_wannier_from_bloch(G, kc, qc, Re, Rp) -> np.ndarray:
    """Eq. 6 in the Wannier gauge.  G [nqc][nkc][Nm][n'][m'] -> g_RR [Np][Nm][Ne][Nb][Nb]."""
    G = _c(G, np.complex128)
    nqc, nkc, nm, nb, _ = G.shape
    kc, qc = _c(kc, np.float64), _c(qc, np.float64)
    Re, Rp = _c(Re, np.int32), _c(Rp, np.int32)
    ne, np_ = Re.shape[0], Rp.shape[0]
    out = np.empty((np_, nm, ne, nb, nb), dtype=np.complex128)
    lib().oracle_eq6_wannier_from_bloch(nb, nm, ne, np_, _p(G), _p(kc), nkc, _p(qc), nqc, _p(Re), _p(Rp), _p(out))
    return out


def eq6_unrotate(g, Ukq_cm, Uk_cm, e_cm, omega) -> np.ndarray:
    """Gauge part of Eq. 6 for one (k',q') block: Bloch g [nu][n][m] -> Wannier-gauge g~ [ka][n'][m']."""
    g = _c(g, np.complex128)
    nm, nb, _ = g.shape
    Ukq_cm, Uk_cm, e_cm = _c(Ukq_cm, np.complex128), _c(Uk_cm, np.complex128), _c(e_cm, np.complex128)
    omega = _c(omega, np.float64)
    out = np.empty_like(g)
    lib().oracle_eq6_unrotate(nb, nm, _p(g), _p(Ukq_cm), _p(Uk_cm), _p(e_cm), _p(omega), _p(out))
    return out


def window_mask(eps_k, eps_kq, emin, emax) -> np.ndarray:
    """Energy-window pre-screening: uint8 [nq][nk], 1 = pair kept."""
    eps_k, eps_kq = _c(eps_k, np.float64), _c(eps_kq, np.float64)
    nq, nk, nb = eps_kq.shape
    out = np.empty((nq, nk), dtype=np.uint8)
    lib().oracle_window_mask(nb, nk, nq, _p(eps_k), _p(eps_kq), float(emin), float(emax), _p(out))
    return out


def selfenergy_accumulate(g2, eps_k, eps_kq, omega, w_q, mu, kT, sigma, out=None) -> np.ndarray:
    """Im Sigma_nk accumulator (NEXT-4 consumer, reading G18): g2 [nq][nk][Nm][Nb][Nb] -> out [nk][Nb] (+=)."""
    g2, eps_k, eps_kq, omega = _c(g2, np.float64), _c(eps_k, np.float64), _c(eps_kq, np.float64), _c(omega, np.float64)
    nq, nk, nm, nb, _ = g2.shape
    w_q = None if w_q is None else _c(w_q, np.float64)
    if out is None:
        out = np.zeros((nk, nb), dtype=np.float64)
    lib().oracle_selfenergy_accumulate(nb, nm, nk, nq, _p(g2), _p(eps_k), _p(eps_kq), _p(omega), _p(w_q), float(mu),
                                       float(kT), float(sigma), _p(out))
    return out


def g_bytes(nb, nm, ne, np_) -> float:
    return lib().oracle_g_bytes(nb, nm, ne, np_)


def nmul_single_loop(nb, nm, ne, np_, nk, nq) -> float:
    return lib().oracle_nmul_single_loop(nb, nm, ne, np_, nk, nq)


def nmul_nested_loop(nb, nm, ne, np_, nk, nq) -> float:
    return lib().oracle_nmul_nested_loop(nb, nm, ne, np_, nk, nq)


# ----------------------------------------------------------------------------------------------
# Gauge-free comparison helper [reading G10/G11]: sum |g|^2 over degenerate blocks.
# Written for the tests (both sides of a parity comparison go through the same function).
# ----------------------------------------------------------------------------------------------
def degenerate_blocks(ev: np.ndarray, gap: float = 1e-6) -> list[tuple[int, int]]:
    """Chains of consecutive (ascending) eigenvalues with gap < `gap` -> [(start, stop), ...]."""
    blocks, start = [], 0
    for i in range(1, len(ev) + 1):
        if i == len(ev) or ev[i] - ev[i - 1] >= gap:
            blocks.append((start, i))
            start = i
    return blocks


def block_sum_g2(g2: np.ndarray, eps_kq: np.ndarray, eps_k: np.ndarray, omega: np.ndarray, gap: float = 1e-6) -> np.ndarray:
    """g2 [nu][n][m] -> sums over degenerate blocks in nu (omega), n (eps_k), m (eps_kq)."""
    bm, bn, bv = degenerate_blocks(eps_kq, gap), degenerate_blocks(eps_k, gap), degenerate_blocks(omega, gap)
    out = np.empty((len(bv), len(bn), len(bm)))
    for a, (v0, v1) in enumerate(bv):
        for b, (n0, n1) in enumerate(bn):
            for c, (m0, m1) in enumerate(bm):
                out[a, b, c] = g2[v0:v1, n0:n1, m0:m1].sum()
    return out
