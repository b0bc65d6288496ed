"""Seeded synthetic workloads shaped like the paper's Si / MoS2 / stanene cases.

This package is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
library (`paper_2603_10295_b200/`).  It holds no arithmetic of the method: it
only draws random operators H(R), D(R), g(Re,Rp), the lattice-vector lists, the
k grids and the q lists that `BASELINE.json` `configs[0..4]` describe (recipe in
DESIGN.md, "Input recipe").

The paper's own inputs (PAPER.md:L241 silicon, L251 MoS2, L265/Table III
stanene nanoribbons) are not available offline; these seeded
tensors stand in for them with the same shapes and the same exponential decay
in |Re|, |Rp|.

Array conventions (all complex128, "Fortran" = first index fastest):
  H_R   flat[i + Nb*(j + Nb*ie)]                        shape (Ne, Nb, Nb) in numpy C order = [ie][j][i]
  D_R   flat[a + Nm*(b + Nm*ip)]                        shape (Np, Nm, Nm)              = [ip][b][a]
  g_RR  flat[m' + Nb*(n' + Nb*(ie + Ne*(ka + Nm*ip)))]  shape (Np, Nm, Ne, Nb, Nb)      = [ip][ka][ie][n'][m']
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "synth.c")
_LIB = os.path.join(_HERE, "libsynth.so")

STREAM_H, STREAM_D, STREAM_G, STREAM_Q = 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile synth.c -> libsynth.so with gcc (host only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", tmp, _SRC, "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u64, i32, f64, vp = ctypes.c_uint64, ctypes.c_int32, ctypes.c_double, ctypes.c_void_p
        lib.synth_gauss_complex.argtypes = [u64, u64, u64, u64, f64, vp]
        lib.synth_gauss_complex.restype = None
        lib.synth_uniform.argtypes = [u64, u64, u64, u64, vp]
        lib.synth_uniform.restype = None
        lib.synth_fill_g.argtypes = [u64, u64, i32, i32, i32, i32, i32, i32, f64, vp, vp, f64, f64, vp]
        lib.synth_fill_g.restype = None
        _lib = lib
    return _lib


def gauss_complex(seed: int, stream: int, start: int, count: int, scale: float = 1.0) -> np.ndarray:
    out = np.empty(count, dtype=np.complex128)
    _load().synth_gauss_complex(seed, stream, start, count, scale, out.ctypes.data)
    return out


def uniform(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    out = np.empty(count, dtype=np.float64)
    _load().synth_uniform(seed, stream, start, count, out.ctypes.data)
    return out


def lattice_vectors(nmax: tuple[int, int, int]) -> np.ndarray:
    """All integer (n1,n2,n3) with |n_i| <= nmax[i]; lexicographic, n3 fastest. int32 [N,3]."""
    ax = [np.arange(-m, m + 1, dtype=np.int32) for m in nmax]
    g = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    return np.ascontiguousarray(g)


def uniform_grid(n: tuple[int, int, int]) -> np.ndarray:
    """Gamma-centred uniform grid (i1/N1, i2/N2, i3/N3), i3 fastest. float64 [N,3]."""
    ax = [np.arange(m, dtype=np.float64) / m for m in n]
    g = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    return np.ascontiguousarray(g)


def grid_kq_map(n: tuple[int, int, int], kq_n: tuple[int, int, int]) -> np.ndarray:
    """kq_map[iq, ik] = index in the k grid `n` of k+q folded into [0,1), q from the grid `kq_n`.

    Requires every q-grid dimension to divide the k-grid dimension (q points lie on the k grid).
    """
    n = np.asarray(n)
    kq_n = np.asarray(kq_n)
    assert np.all(n % kq_n == 0)
    step = n // kq_n
    ki = np.stack(np.meshgrid(*[np.arange(m) for m in n], indexing="ij"), axis=-1).reshape(-1, 3)
    qi = np.stack(np.meshgrid(*[np.arange(m) for m in kq_n], indexing="ij"), axis=-1).reshape(-1, 3) * step
    s = (ki[None, :, :] + qi[:, None, :]) % n
    return np.ascontiguousarray((s[..., 0] * n[1] + s[..., 1]) * n[2] + s[..., 2]).astype(np.int32)


def _hermitian_family(seed: int, stream: int, n: int, R: np.ndarray, lam: float) -> np.ndarray:
    """Op(R) = 0.5*exp(-|R|/lam)*Z_R for one of each +-R pair, Op(-R) = Op(R)^dagger, Op(0) hermitised.

    Returns [NR][j][i] (Fortran per matrix: element (i,j) at [ir, j, i]).
    """
    nr = R.shape[0]
    # the R sets are symmetric and lexicographically ordered, so -R_i = R_{nr-1-i}
    assert np.array_equal(R, -R[::-1])
    norm = np.sqrt((R.astype(np.float64) ** 2).sum(axis=1))
    out = np.zeros((nr, n, n), dtype=np.complex128)
    for ir in range(nr):
        jr = nr - 1 - ir
        if ir > jr:
            continue
        z = gauss_complex(seed, stream, ir * n * n, n * n).reshape(n, n)  # z[j][i] <-> element (i,j)
        m = 0.5 * np.exp(-norm[ir] / lam) * z
        if ir == jr:
            out[ir] = 0.5 * (m + m.conj().T)
        else:
            out[ir] = m
            out[jr] = m.conj().T
    return out


@dataclass
class Workload:
    """One synthetic configuration.  `g_slab(ip)` regenerates any Rp slab on demand."""

    name: str
    index: int
    seed: int
    nbnd: int
    nmodes: int
    Re: np.ndarray  # int32 [Ne,3]
    Rp: np.ndarray  # int32 [Np,3]
    w_e: np.ndarray  # float64 [Ne]
    w_p: np.ndarray  # float64 [Np]
    H_R: np.ndarray  # complex128 [Ne][j][i]
    D_R: np.ndarray  # complex128 [Np][b][a]
    k_grid: tuple[int, int, int]
    q_desc: str
    g_amp: float
    lam_g_e: float
    lam_g_p: float
    q_list: np.ndarray  # float64 [Nq,3]
    q_grid: tuple[int, int, int] | None = None
    _k_list: np.ndarray | None = field(default=None, repr=False)

    @property
    def ne(self) -> int:
        return int(self.Re.shape[0])

    @property
    def np_(self) -> int:
        return int(self.Rp.shape[0])

    @property
    def nk(self) -> int:
        return int(np.prod(self.k_grid))

    @property
    def nq(self) -> int:
        return int(self.q_list.shape[0])

    @property
    def elements_per_pair(self) -> int:
        return self.nbnd * self.nbnd * self.nmodes

    @property
    def k_list(self) -> np.ndarray:
        if self._k_list is None:
            self._k_list = uniform_grid(self.k_grid)
        return self._k_list

    def k_slice(self, start: int, stop: int) -> np.ndarray:
        """Rows start..stop-1 of the uniform k grid without building the whole list."""
        idx = np.arange(start, stop, dtype=np.int64)
        n1, n2, n3 = self.k_grid
        i3 = idx % n3
        i2 = (idx // n3) % n2
        i1 = idx // (n3 * n2)
        return np.ascontiguousarray(np.stack([i1 / n1, i2 / n2, i3 / n3], axis=1).astype(np.float64))

    @property
    def kq_map(self) -> np.ndarray | None:
        """[Nq,Nk] int32 index of k+q in the k grid when q lies on the k grid, else None."""
        if self.q_grid is None:
            return None
        return grid_kq_map(self.k_grid, self.q_grid)

    @property
    def slab_elems(self) -> int:
        return self.nbnd * self.nbnd * self.ne * self.nmodes

    @property
    def g_bytes(self) -> int:
        """Table III caption: 16*Nb^2*Nm*Ne*Np bytes."""
        return 16 * self.slab_elems * self.np_

    def g_slabs(self, ip_start: int, ip_count: int) -> np.ndarray:
        """complex128 [ip_count][ka][ie][n'][m'] for Rp indices ip_start..ip_start+ip_count-1."""
        out = np.empty((ip_count, self.nmodes, self.ne, self.nbnd, self.nbnd), dtype=np.complex128)
        re_norm = np.sqrt((self.Re.astype(np.float64) ** 2).sum(axis=1))
        rp_norm = np.sqrt((self.Rp.astype(np.float64) ** 2).sum(axis=1))
        _load().synth_fill_g(
            self.seed, STREAM_G, self.nbnd, self.nmodes, self.ne, self.np_, ip_start, ip_count, self.g_amp,
            re_norm.ctypes.data, rp_norm.ctypes.data, self.lam_g_e, self.lam_g_p, out.ctypes.data,
        )
        return out

    def g_slab(self, ip: int) -> np.ndarray:
        return self.g_slabs(ip, 1)[0]

    def g_full(self) -> np.ndarray:
        """complex128 [Np][Nm][Ne][Nb][Nb]; refuse silly sizes (config 4 is 49 GB: use slabs)."""
        if self.g_bytes > 8 << 30:
            raise MemoryError(f"g is {self.g_bytes / 2**30:.1f} GiB; stream it with g_slabs()")
        return self.g_slabs(0, self.np_)


# name, nbnd, nmodes, R nmax, lambda(H,D), g amp, lambda g (e,p), k grid, q spec
_CONFIGS = [
    dict(name="tiny-si", nbnd=8, nmodes=6, rmax=(1, 1, 1), lam=1.0, amp=0.1, lam_g=1.0,
         k_grid=(4, 4, 4), q=("grid", (4, 4, 4))),
    dict(name="si-production", nbnd=8, nmodes=6, rmax=(3, 3, 3), lam=1.5, amp=0.1, lam_g=1.5,
         k_grid=(40, 40, 40), q=("random", 1000, 3)),
    dict(name="mos2-2d", nbnd=11, nmodes=9, rmax=(6, 6, 0), lam=2.0, amp=0.1, lam_g=2.0,
         k_grid=(120, 120, 1), q=("random", 2000, 2)),
    dict(name="si-large-grid", nbnd=8, nmodes=6, rmax=(4, 4, 4), lam=1.5, amp=0.1, lam_g=1.5,
         k_grid=(100, 100, 100), q=("random", 256, 3)),
    dict(name="zsnr-1d", nbnd=192, nmodes=288, rmax=(8, 0, 0), lam=1.0, amp=0.05, lam_g=2.0,
         k_grid=(200, 1, 1), q=("grid", (200, 1, 1))),
]

NUM_CONFIGS = len(_CONFIGS)


def make_custom(name: str, nbnd: int, nmodes: int, rmax, lam: float, amp: float, lam_g: float, k_grid, q,
                seed: int, index: int = -1) -> Workload:
    """Build a workload from an explicit recipe (used for reduced-size test cases)."""
    R = lattice_vectors(tuple(rmax))
    nr = R.shape[0]
    H = _hermitian_family(seed, STREAM_H, nbnd, R, lam)
    D = _hermitian_family(seed, STREAM_D, nmodes, R, lam)
    # D(0) += (1 + sum_R ||D(R)||_F) * I  => D(q) positive definite for every q
    shift = 1.0 + sum(np.linalg.norm(D[i]) for i in range(nr))
    D[nr // 2] += shift * np.eye(nmodes)
    if q[0] == "grid":
        q_list = uniform_grid(tuple(q[1]))
        q_grid = tuple(q[1])
        q_desc = "grid %dx%dx%d" % tuple(q[1])
    else:
        nq, dims = int(q[1]), int(q[2])
        u = uniform(seed, STREAM_Q, 0, 3 * nq).reshape(nq, 3)
        u[:, dims:] = 0.0
        q_list = np.ascontiguousarray(u)
        q_grid = None
        q_desc = f"{nq} seeded uniform-random points ({dims}D)"
    return Workload(
        name=name, index=index, seed=seed, nbnd=nbnd, nmodes=nmodes, Re=R, Rp=R.copy(),
        w_e=np.ones(nr), w_p=np.ones(nr), H_R=H, D_R=D, k_grid=tuple(k_grid), q_desc=q_desc,
        g_amp=amp, lam_g_e=lam_g, lam_g_p=lam_g, q_list=q_list, q_grid=q_grid,
    )


def make_config(index: int) -> Workload:
    """BASELINE.json configs[index]; seed = index (config 0: seed 0 as stated there)."""
    c = _CONFIGS[index]
    return make_custom(c["name"], c["nbnd"], c["nmodes"], c["rmax"], c["lam"], c["amp"], c["lam_g"],
                       c["k_grid"], c["q"], seed=index, index=index)
