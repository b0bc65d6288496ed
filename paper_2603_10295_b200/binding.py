"""Thin ctypes binding of include/epw_interp.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of
libepw_interp.so.  PyTorch appears here solely as the owner of device memory and
streams (`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`).
The functions carry the names of the C entry points; `EpwInterp` is a small
convenience wrapper that owns a handle.

There is no CPU fallback: importing works without a GPU (so that the symbol
table can be checked on a CPU box), but every compute call raises `EpwError`
when the library reports EPW_ECUDA.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int, c_int32, c_int64, c_size_t, c_void_p

PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(PKG, "libepw_interp.so")

EPW_OK, EPW_EINVAL, EPW_ENOMEM, EPW_ECUDA, EPW_ENOTCONVERGED, EPW_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
EPW_PATH_AUTO, EPW_PATH_SMALL, EPW_PATH_LARGE = 0, 1, 2
EPW_FLAG_GRID_UNFUSED, EPW_FLAG_GRID_FUSED = 1, 2
EPW_NUM_STAGES = 9
STAGE_NAMES = ["S0_phase_tables", "S1_rp_to_q", "phonon_Dq_eig_S4a_pack", "Hk_eig", "S2_re_to_k_dmma", "Hkq_eig",
               "S4b_rotate_g2", "total", "S4a_mode_rotation"]
EPW_DBG_G_REQ, EPW_DBG_G_TILDE, EPW_DBG_H_K, EPW_DBG_U_K, EPW_DBG_U_KQ, EPW_DBG_E_Q = 1, 2, 3, 4, 5, 6

# every symbol include/epw_interp.h declares (tests check that the library exports each of them)
EXPORTED_SYMBOLS = [
    "epw_interp_create", "epw_interp_destroy", "epw_interp_set_wannier_operators", "epw_interp_set_g_slabs",
    "epw_interp_interpolate", "epw_interp_interpolate_host", "epw_interp_interpolate_grid",
    "epw_interp_interpolate_grid_host", "epw_interp_sync", "epw_interp_get_stage_times",
    "epw_interp_enable_stage_timing", "epw_interp_get_stage_launches", "epw_interp_last_launch_count", "epw_interp_get_eigh_rotations", "epw_interp_last_plan", "epw_interp_debug_get", "epw_interp_last_error",
    "epw_phase_table", "epw_rp_to_q", "epw_interp_operator", "epw_eigh_batched", "epw_eigh_batched_algo", "epw_zgemm", "epw_zgemm_noalloc", "epw_zgemm_strided",
    "epw_rotate_g2", "epw_axis_pass_dmma",
    "epw_eq6_unrotate", "epw_wannier_from_bloch",
    "epw_interp_set_energy_window", "epw_interp_set_selfenergy_consumer", "epw_interp_set_rp_shard", "epw_interp_rp_to_q_partial", "epw_interp_rp_to_q_scatter_add", "epw_interp_set_gq",
    "epw_probe_peaks", "epw_version",
]


class EpwError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"epw_interp error {code}: {msg}")
        self.code = code


class epw_interp_config(ctypes.Structure):
    _fields_ = [("nbnd", c_int32), ("nmodes", c_int32), ("ne", c_int32), ("np", c_int32), ("device", c_int32),
                ("q_batch", c_int32), ("path", c_int32), ("flags", c_int32), ("workspace_bytes", c_size_t), ("degen_tol", c_double), ("omega_min", c_double)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree CUDA library; fail loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2603_10295_b200.build` "
                "(there is no CPU fallback for the interpolation path)")
        L = ctypes.CDLL(LIB_PATH)
        vp = c_void_p
        L.epw_interp_create.argtypes = [POINTER(vp), POINTER(epw_interp_config)]
        L.epw_interp_destroy.argtypes = [vp]
        L.epw_interp_destroy.restype = None
        L.epw_interp_set_wannier_operators.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, c_int]
        L.epw_interp_set_g_slabs.argtypes = [vp, c_int32, c_int32, vp, c_int]
        L.epw_interp_interpolate.argtypes = [vp, vp, c_int64, vp, c_int64, vp, vp, vp, vp, vp, vp]
        L.epw_interp_interpolate_host.argtypes = [vp, vp, c_int64, vp, c_int64, vp, vp, vp, vp, vp, vp]
        L.epw_interp_interpolate_grid.argtypes = [vp, vp, vp, vp, c_int64, vp, vp, vp, vp, vp, vp]
        L.epw_interp_interpolate_grid_host.argtypes = [vp, vp, vp, vp, c_int64, vp, vp, vp, vp, vp, vp]
        L.epw_interp_set_energy_window.argtypes = [vp, c_int, c_double, c_double, vp]
        L.epw_interp_set_selfenergy_consumer.argtypes = [vp, c_int, c_double, c_double, c_double, vp, vp]
        L.epw_interp_set_rp_shard.argtypes = [vp, c_int32, c_int32]
        L.epw_interp_rp_to_q_partial.argtypes = [vp, vp, c_int64, vp, vp]
        L.epw_interp_rp_to_q_scatter_add.argtypes = [vp, vp, c_int64, vp, vp]
        L.epw_interp_set_gq.argtypes = [vp, vp]
        L.epw_interp_sync.argtypes = [vp]
        L.epw_interp_get_stage_times.argtypes = [vp, POINTER(c_double), c_int]
        L.epw_interp_enable_stage_timing.argtypes = [vp, c_int]
        L.epw_interp_get_stage_launches.argtypes = [vp, POINTER(c_int64), c_int]
        L.epw_interp_last_launch_count.argtypes = [vp]
        L.epw_interp_last_launch_count.restype = c_int64
        L.epw_interp_get_eigh_rotations.argtypes = [vp, POINTER(ctypes.c_uint64), c_int]
        L.epw_interp_last_plan.argtypes = [vp, POINTER(c_int64), c_int]
        L.epw_interp_debug_get.argtypes = [vp, c_int, vp, c_size_t]
        L.epw_interp_debug_get.restype = c_int64
        L.epw_interp_last_error.argtypes = [vp]
        L.epw_interp_last_error.restype = c_char_p
        L.epw_phase_table.argtypes = [vp, c_int64, vp, vp, c_int32, vp, vp]
        L.epw_rp_to_q.argtypes = [vp, c_int64, c_int32, vp, c_int32, vp, vp]
        L.epw_interp_operator.argtypes = [vp, c_int32, c_int32, vp, c_int64, vp, vp]
        L.epw_eigh_batched.argtypes = [vp, c_int64, c_int32, c_int64, vp, vp, c_int, vp, vp]
        L.epw_eigh_batched_algo.argtypes = [vp, c_int64, c_int32, c_int64, vp, vp, c_int, vp, c_int, vp]
        L.epw_zgemm.argtypes = [vp, vp, vp, c_int64, c_int32, c_int32, c_int64, vp]
        L.epw_zgemm_noalloc.argtypes = [vp, vp, vp, c_int64, c_int32, c_int32, c_int64, vp, c_char_p, c_size_t]
        L.epw_zgemm_strided.argtypes = [vp, c_int64, c_int64, c_int64, c_int64, vp, c_int64, c_int64, c_int64, c_int, vp,
                                        c_int64, vp, c_int64, c_int64, c_int64, c_int64, c_int64, c_int, c_int64,
                                        c_int32, c_int32, c_int64, vp]
        L.epw_rotate_g2.argtypes = [vp, c_int64, vp, vp, vp, c_int32, c_int32, c_int64, vp, vp]
        L.epw_axis_pass_dmma.argtypes = [vp, c_int64, c_int32, c_int32, vp, c_int32, c_int32, vp, c_int64, c_int32, c_int64,
                                         c_int64, vp]
        L.epw_eq6_unrotate.argtypes = [vp, vp, vp, vp, vp, c_int32, c_int32, c_int64, c_int64, vp, vp]
        L.epw_wannier_from_bloch.argtypes = [vp, vp, c_int64, vp, c_int64, vp, c_int32, vp, c_int32, c_int32, c_int32, vp, vp]
        L.epw_probe_peaks.argtypes = [c_int32, POINTER(c_double)]
        L.epw_version.restype = c_char_p
        _lib = L
    return _lib


def _ptr(t):
    """Device/host pointer of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream():
    import torch

    return torch.cuda.current_stream().cuda_stream


def _check(rc: int, h=None):
    if rc < 0:
        msg = load_library().epw_interp_last_error(h)
        raise EpwError(rc, msg.decode() if msg else "")
    return rc


# ---- the calls of include/epw_interp.h, same names --------------------------------------------------------
def epw_version() -> str:
    return load_library().epw_version().decode()


def epw_interp_create(nbnd, nmodes, ne, np_, device=0, q_batch=0, workspace_bytes=0, degen_tol=1e-6, omega_min=0.0,
                      path=EPW_PATH_AUTO, flags=0):
    cfg = epw_interp_config(nbnd, nmodes, ne, np_, device, q_batch, path, flags, workspace_bytes, degen_tol, omega_min)
    h = c_void_p()
    _check(load_library().epw_interp_create(byref(h), byref(cfg)))
    return h


def epw_interp_last_error(h=None) -> str:
    msg = load_library().epw_interp_last_error(h)
    return msg.decode() if msg else ""


def epw_interp_destroy(h):
    load_library().epw_interp_destroy(h)


def epw_interp_set_wannier_operators(h, H_R, D_R, g_RR, Re, w_e, Rp, w_p, on_device):
    _check(load_library().epw_interp_set_wannier_operators(h, _ptr(H_R), _ptr(D_R), _ptr(g_RR), _ptr(Re), _ptr(w_e),
                                                           _ptr(Rp), _ptr(w_p), int(on_device)), h)


def epw_interp_set_g_slabs(h, ip_start, ip_count, g_slabs, on_device):
    _check(load_library().epw_interp_set_g_slabs(h, ip_start, ip_count, _ptr(g_slabs), int(on_device)), h)


def epw_interp_interpolate(h, k_list, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, stream=None):
    _check(load_library().epw_interp_interpolate(h, _ptr(k_list), nk, _ptr(q_list), nq, _ptr(kq_map), _ptr(eps_k),
                                                 _ptr(eps_kq), _ptr(omega_q), _ptr(g2),
                                                 _stream() if stream is None else stream), h)


def epw_interp_interpolate_host(h, k_list, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, stream=None):
    _check(load_library().epw_interp_interpolate_host(h, _ptr(k_list), nk, _ptr(q_list), nq, _ptr(kq_map), _ptr(eps_k),
                                                      _ptr(eps_kq), _ptr(omega_q), _ptr(g2),
                                                      _stream() if stream is None else stream), h)


def _grid_args(k_grid, k_shift):
    """k_grid / k_shift are HOST triples (the only host arguments of the grid entry points)."""
    g = (c_int32 * 3)(*[int(x) for x in k_grid])
    s = None if k_shift is None else (c_double * 3)(*[float(x) for x in k_shift])
    return g, s


def epw_interp_interpolate_grid(h, k_grid, k_shift, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, stream=None):
    g, s = _grid_args(k_grid, k_shift)
    _check(load_library().epw_interp_interpolate_grid(h, g, s, _ptr(q_list), nq, _ptr(kq_map), _ptr(eps_k), _ptr(eps_kq),
                                                      _ptr(omega_q), _ptr(g2),
                                                      _stream() if stream is None else stream), h)


def epw_interp_interpolate_grid_host(h, k_grid, k_shift, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2, stream=None):
    g, s = _grid_args(k_grid, k_shift)
    _check(load_library().epw_interp_interpolate_grid_host(h, g, s, _ptr(q_list), nq, _ptr(kq_map), _ptr(eps_k),
                                                           _ptr(eps_kq), _ptr(omega_q), _ptr(g2),
                                                           _stream() if stream is None else stream), h)


def epw_interp_set_energy_window(h, enabled, emin=0.0, emax=0.0, mask_out=None):
    _check(load_library().epw_interp_set_energy_window(h, int(bool(enabled)), float(emin), float(emax), _ptr(mask_out)), h)


def epw_interp_set_selfenergy_consumer(h, enabled, mu=0.0, kT=1.0, sigma=1.0, w_q=None, im_sigma=None):
    _check(load_library().epw_interp_set_selfenergy_consumer(h, int(bool(enabled)), float(mu), float(kT), float(sigma),
                                                             _ptr(w_q), _ptr(im_sigma)), h)


def epw_interp_set_rp_shard(h, ip_start, ip_count):
    _check(load_library().epw_interp_set_rp_shard(h, ip_start, ip_count), h)


def epw_interp_rp_to_q_partial(h, q_list, nq, g1_partial, stream=None):
    _check(load_library().epw_interp_rp_to_q_partial(h, _ptr(q_list), nq, _ptr(g1_partial),
                                                     _stream() if stream is None else stream), h)


def epw_interp_rp_to_q_scatter_add(h, q_list, nq, dst_ptrs, stream=None):
    """dst_ptrs: sequence of nq device pointers (ints) or tensors; see include/epw_interp.h."""
    arr = (c_void_p * nq)(*[(_ptr(d) if not isinstance(d, int) else d) for d in dst_ptrs])
    _check(load_library().epw_interp_rp_to_q_scatter_add(h, _ptr(q_list), nq, arr, _stream() if stream is None else stream), h)


def epw_interp_set_gq(h, g1_reduced):
    _check(load_library().epw_interp_set_gq(h, _ptr(g1_reduced)), h)


def epw_interp_sync(h):
    _check(load_library().epw_interp_sync(h), h)


def epw_interp_enable_stage_timing(h, on=True):
    _check(load_library().epw_interp_enable_stage_timing(h, int(on)), h)


def epw_interp_get_stage_times(h) -> dict:
    buf = (c_double * EPW_NUM_STAGES)()
    n = _check(load_library().epw_interp_get_stage_times(h, buf, EPW_NUM_STAGES), h)
    return {STAGE_NAMES[i]: buf[i] for i in range(n)}


def epw_interp_get_stage_launches(h) -> dict:
    buf = (c_int64 * EPW_NUM_STAGES)()
    n = _check(load_library().epw_interp_get_stage_launches(h, buf, EPW_NUM_STAGES), h)
    return {STAGE_NAMES[i]: int(buf[i]) for i in range(n)}


def epw_interp_last_launch_count(h) -> int:
    return int(load_library().epw_interp_last_launch_count(h))


def epw_interp_get_eigh_rotations(h) -> dict:
    buf = (ctypes.c_uint64 * 3)()
    _check(load_library().epw_interp_get_eigh_rotations(h, buf, 3), h)
    return {"Hk": int(buf[0]), "Hkq": int(buf[1]), "Dq": int(buf[2])}


def epw_interp_last_plan(h) -> dict:
    buf = (c_int64 * 4)()
    _check(load_library().epw_interp_last_plan(h, buf, 4), h)
    return {"path": "large" if buf[0] == EPW_PATH_LARGE else "small", "q_batch": int(buf[1]), "k_chunk": int(buf[2]),
            "k_mode": ("list", "grid", "grid-fused")[int(buf[3])]}


def epw_interp_debug_get(h, what, dst_host):
    return _check(load_library().epw_interp_debug_get(h, what, _ptr(dst_host), dst_host.nbytes), h)


def epw_phase_table(x_list, nx, R, w, nr, P_out, stream=None):
    _check(load_library().epw_phase_table(_ptr(x_list), nx, _ptr(R), _ptr(w), nr, _ptr(P_out),
                                          _stream() if stream is None else stream))


def epw_rp_to_q(g_RR, rows, np_, Pq, nq, g1_out, stream=None):
    _check(load_library().epw_rp_to_q(_ptr(g_RR), rows, np_, _ptr(Pq), nq, _ptr(g1_out),
                                      _stream() if stream is None else stream))


def epw_interp_operator(Op_R, n, nr, P, nx, out, stream=None):
    _check(load_library().epw_interp_operator(_ptr(Op_R), n, nr, _ptr(P), nx, _ptr(out),
                                              _stream() if stream is None else stream))


def epw_eigh_batched(A, stride_a, n, batch, evals, V, sqrt_mode=0, status=None, stream=None):
    _check(load_library().epw_eigh_batched(_ptr(A), stride_a, n, batch, _ptr(evals), _ptr(V), int(sqrt_mode),
                                           _ptr(status), _stream() if stream is None else stream))


EPW_EIGH_AUTO, EPW_EIGH_WARP, EPW_EIGH_THREAD, EPW_EIGH_COLS = 0, 1, 2, 3


def epw_eigh_batched_algo(A, stride_a, n, batch, evals, V, sqrt_mode=0, status=None, algo=EPW_EIGH_AUTO, stream=None):
    _check(load_library().epw_eigh_batched_algo(_ptr(A), stride_a, n, batch, _ptr(evals), _ptr(V), int(sqrt_mode),
                                                _ptr(status), int(algo), _stream() if stream is None else stream))


def epw_zgemm(A, B, C, M, N, K, ldc, stream=None):
    _check(load_library().epw_zgemm(_ptr(A), _ptr(B), _ptr(C), M, N, K, ldc, _stream() if stream is None else stream))


EPW_ZGEMM_NOALLOC_SCRATCH_BYTES = 16 * 1024 * 1024


def epw_zgemm_noalloc(A, B, C, M, N, K, ldc, stream=None):
    """epw_zgemm without any device allocation inside the library (packed operands in the library's fixed 16 MiB array).
    For callers whose device memory belongs to their own pool, or whose loop may not hit the device-wide stall of
    cudaMalloc / cudaFree.  Asynchronous; raises EpwError(EPW_EUNSUPPORTED) with the library's message when
    ceil(M/128) ceil(K/8) + ceil(N/64) ceil(K/8) exceeds 1,024.  Calls that can overlap on the GPU share the array and
    race; the first call on a device does the one-time address look-up and should come before any stream capture."""
    err = ctypes.create_string_buffer(512)
    rc = load_library().epw_zgemm_noalloc(_ptr(A), _ptr(B), _ptr(C), M, N, K, ldc, _stream() if stream is None else stream,
                                          err, len(err))
    if rc < 0:
        raise EpwError(rc, err.value.decode())


def epw_zgemm_strided(A, a_rb, a_bs, a_ks, a_batch, B, b_sr, b_sn, b_batch, b_conj, b_gather, nb_mats, C, c_rb, c_bs,
                      c_rs, c_cs, c_batch, abs2, M, N, K, batch, stream=None):
    _check(load_library().epw_zgemm_strided(_ptr(A), a_rb, a_bs, a_ks, a_batch, _ptr(B), b_sr, b_sn, b_batch,
                                            int(b_conj), _ptr(b_gather), nb_mats, _ptr(C), c_rb, c_bs, c_rs, c_cs,
                                            c_batch, int(abs2), M, N, K, batch,
                                            _stream() if stream is None else stream))


def epw_axis_pass_dmma(T, slab, ncols, L, P, cnt, nb, out, out_stride, nbatch=1, in_bstride=0, out_bstride=0, stream=None):
    _check(load_library().epw_axis_pass_dmma(_ptr(T), slab, ncols, L, _ptr(P), cnt, nb, _ptr(out), out_stride, nbatch,
                                             in_bstride, out_bstride, _stream() if stream is None else stream))


def epw_rotate_g2(gt, stride_gt, Uk, Ukq, kq_idx, nb, nm, nk, g2, stream=None):
    _check(load_library().epw_rotate_g2(_ptr(gt), stride_gt, _ptr(Uk), _ptr(Ukq), _ptr(kq_idx), nb, nm, nk, _ptr(g2),
                                        _stream() if stream is None else stream))


def epw_eq6_unrotate(g_bloch, Uk, Ukq, e_q, omega_q, nb, nm, nkc, nqc, gt_out, stream=None):
    _check(load_library().epw_eq6_unrotate(_ptr(g_bloch), _ptr(Uk), _ptr(Ukq), _ptr(e_q), _ptr(omega_q), nb, nm, nkc, nqc,
                                           _ptr(gt_out), _stream() if stream is None else stream))


def epw_wannier_from_bloch(gt, kc, nkc, qc, nqc, Re, ne, Rp, np_, nb, nm, g_RR_out, stream=None):
    _check(load_library().epw_wannier_from_bloch(_ptr(gt), _ptr(kc), nkc, _ptr(qc), nqc, _ptr(Re), ne, _ptr(Rp), np_, nb,
                                                 nm, _ptr(g_RR_out), _stream() if stream is None else stream))


def epw_probe_peaks(device=0) -> dict:
    out = (c_double * 4)()
    _check(load_library().epw_probe_peaks(device, out))
    return {"fp64_dmma_tflops": out[0], "fp64_dfma_tflops": out[1], "hbm_read_gbs": out[2], "hbm_copy_gbs": out[3]}


class EpwInterp:
    """Owns one library handle.  `workload` is a synth.Workload-like object (numpy operators on the host)."""

    def __init__(self, nbnd, nmodes, ne, np_, device=0, q_batch=0, workspace_bytes=0, omega_min=0.0,
                 path=EPW_PATH_AUTO, flags=0):
        self.nbnd, self.nmodes, self.ne, self.np = nbnd, nmodes, ne, np_
        self.device = device
        self.h = epw_interp_create(nbnd, nmodes, ne, np_, device, q_batch, workspace_bytes, 1e-6, omega_min, path, flags)

    def close(self):
        if self.h is not None:
            epw_interp_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_operators_from_host(self, w, slab_chunk_bytes=2 << 30, rp_range=None):
        """Upload H, D, R lists from a workload and stream g(Re,Rp) in Rp slabs (never holds all of g on the host).
        rp_range = (start, stop): keep only that Rp shard of g on this GPU (epw_interp_set_rp_shard)."""
        lo, hi = (0, w.np_) if rp_range is None else rp_range
        if rp_range is not None:
            epw_interp_set_rp_shard(self.h, lo, hi - lo)
        epw_interp_set_wannier_operators(self.h, w.H_R, w.D_R, None, w.Re, w.w_e, w.Rp, w.w_p, 0)
        per_slab = 16 * w.slab_elems
        step = max(1, int(slab_chunk_bytes // per_slab))
        for ip in range(lo, hi, step):
            cnt = min(step, hi - ip)
            epw_interp_set_g_slabs(self.h, ip, cnt, w.g_slabs(ip, cnt), 0)

    def interpolate(self, k_list, q_list, kq_map=None, want_eps_kq=True):
        """Device tensors in, device tensors out: (eps_k, eps_kq, omega_q, g2)."""
        import torch

        nk, nq = k_list.shape[0], q_list.shape[0]
        dev = k_list.device
        eps_k = torch.empty((nk, self.nbnd), dtype=torch.float64, device=dev)
        eps_kq = torch.empty((nq, nk, self.nbnd), dtype=torch.float64, device=dev) if want_eps_kq else None
        omega_q = torch.empty((nq, self.nmodes), dtype=torch.float64, device=dev)
        g2 = torch.empty((nq, nk, self.nmodes, self.nbnd, self.nbnd), dtype=torch.float64, device=dev)
        epw_interp_interpolate(self.h, k_list, nk, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2)
        return eps_k, eps_kq, omega_q, g2

    def interpolate_grid(self, k_grid, q_list, k_shift=None, kq_map=None, want_eps_kq=True):
        """Uniform k-grid (host triple of sizes, i3 fastest) and a device q-list in, device tensors out."""
        import torch

        nk, nq = int(k_grid[0]) * int(k_grid[1]) * int(k_grid[2]), q_list.shape[0]
        dev = q_list.device
        eps_k = torch.empty((nk, self.nbnd), dtype=torch.float64, device=dev)
        eps_kq = torch.empty((nq, nk, self.nbnd), dtype=torch.float64, device=dev) if want_eps_kq else None
        omega_q = torch.empty((nq, self.nmodes), dtype=torch.float64, device=dev)
        g2 = torch.empty((nq, nk, self.nmodes, self.nbnd, self.nbnd), dtype=torch.float64, device=dev)
        epw_interp_interpolate_grid(self.h, k_grid, k_shift, q_list, nq, kq_map, eps_k, eps_kq, omega_q, g2)
        return eps_k, eps_kq, omega_q, g2
