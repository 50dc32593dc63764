"""Thin ctypes binding of librift_ile.so (include/rift_ile.h).  Argument marshalling only: every step of
the hot path runs in the CUDA kernels behind the C ABI.  PyTorch (if the caller uses it) only owns device
memory and streams; this module accepts anything with ``data_ptr()`` or a raw integer address.

There is no CPU fallback: if the shared library is missing or cannot be loaded, importing the functions
raises.  Build it with ``python -m paper_2210_07912_b200.build``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "librift_ile.so")

RIFT_OK, RIFT_EINVAL, RIFT_ENOMEM, RIFT_ECUDA, RIFT_EWINDOW, RIFT_ERANGE, RIFT_ESTATE = 0, -1, -2, -3, -4, -5, -6
RIFT_PREC_FP64, RIFT_PREC_MIXED = 0, 1
RIFT_Q_C128, RIFT_Q_C64 = 0, 1
RIFT_MEM_HOST, RIFT_MEM_DEVICE = 0, 1
RIFT_KERNEL_AUTO, RIFT_KERNEL_DIRECT, RIFT_KERNEL_TC, RIFT_KERNEL_TCS, RIFT_KERNEL_MMA, RIFT_KERNEL_SKY = 0, 1, 2, 3, 4, 5
RIFT_OPT_TC_CHUNK_MIB, RIFT_OPT_TC_SORT, RIFT_OPT_QUAD_PROG = 1, 2, 3
RIFT_N_PARAMS = 6

EXPORTS = ("rift_ile_create", "rift_ile_eval_batch", "rift_ile_reduce", "rift_ile_geometry", "rift_ile_set_kernel",
           "rift_ile_launch_count", "rift_ile_kernel_name", "rift_ile_profile", "rift_ile_profile_read",
           "rift_ile_fma_peak", "rift_ile_set_option", "rift_ile_reserve", "rift_ile_eval_batch_host",
           "rift_ile_staged", "rift_ile_eval_batch_dmarg", "rift_ile_precompute", "rift_ile_destroy",
           "rift_ile_strerror", "rift_ile_last_error", "rift_ile_reduce_static", "rift_ile_reduce_static_error",
           "rift_ile_rho_guess")
GMM_EXPORTS = ("rift_gmm_create", "rift_gmm_set_model", "rift_gmm_get_model", "rift_gmm_fit", "rift_gmm_fit_tempered", "rift_gmm_draw",
               "rift_gmm_ln_density", "rift_gmm_box_mass", "rift_gmm_add", "rift_gmm_destroy")
RIFT_GMM_MAX_COMP, RIFT_GMM_MAX_TRIES = 8, 64
SKY_EXPORTS = ("rift_sky_network_frame", "rift_sky_network_to_radec", "rift_sky_radec_to_network")
RIFT_REDUCE_STATIC_MAX_SEG = 1024
AC_EXPORTS = ("rift_ac_create", "rift_ac_draw", "rift_ac_update", "rift_ac_update_dims", "rift_ac_get_masses",
              "rift_ac_ile_ln_weight", "rift_ac_destroy")


class RiftError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"rift_ile error {code}: {msg}")
        self.code = code


class _Config(C.Structure):
    _fields_ = [("n_det", C.c_int32), ("det_location_m", C.c_void_p), ("det_response", C.c_void_p),
                ("gmst_rad", C.c_double), ("n_modes", C.c_int32), ("mode_l", C.c_void_p), ("mode_m", C.c_void_p),
                ("n_points", C.c_int32), ("n_t", C.c_int32), ("delta_t", C.c_double), ("n_tau", C.c_int32),
                ("d_ref_mpc", C.c_double), ("Q", C.c_void_p), ("U", C.c_void_p), ("V", C.c_void_p),
                ("input_mem", C.c_int32), ("precision", C.c_int32), ("q_storage", C.c_int32)]


_lib = None


def lib() -> C.CDLL:
    """Load librift_ile.so; raises if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2210_07912_b200.build` (needs nvcc); "
                              "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.rift_ile_create.argtypes = [C.POINTER(_Config), C.POINTER(vp)]
        L.rift_ile_create.restype = C.c_int
        L.rift_ile_eval_batch.argtypes = [vp, i32, vp, i64, C.POINTER(vp), vp, vp, vp]
        L.rift_ile_eval_batch.restype = C.c_int
        L.rift_ile_reduce.argtypes = [vp, i32, i64, vp, vp, C.POINTER(vp), vp, vp, i32, i32, vp, vp, vp, vp, vp, vp]
        L.rift_ile_reduce.restype = C.c_int
        L.rift_ile_geometry.argtypes = [vp, i32, i64, C.POINTER(vp), vp, vp, vp, vp, vp]
        L.rift_ile_geometry.restype = C.c_int
        L.rift_ile_set_kernel.argtypes = [vp, i32]
        L.rift_ile_set_kernel.restype = C.c_int
        L.rift_ile_eval_batch_host.argtypes = [vp, i32, vp, i64, C.POINTER(vp), vp, vp, i32, vp]
        L.rift_ile_eval_batch_host.restype = C.c_int
        L.rift_ile_eval_batch_dmarg.argtypes = [vp, i32, vp, i64, C.POINTER(vp), dbl, dbl, i32, vp, vp, vp]
        L.rift_ile_eval_batch_dmarg.restype = C.c_int
        L.rift_ile_precompute.argtypes = [i32, i32, i32, i32, vp, vp, vp, vp, vp, i32, dbl, vp, vp, vp, vp]
        L.rift_ile_precompute.restype = C.c_int
        L.rift_ile_staged.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(i64)]
        L.rift_ile_staged.restype = C.c_int
        L.rift_ile_set_option.argtypes = [vp, i32, i64]
        L.rift_ile_set_option.restype = C.c_int
        L.rift_ile_reserve.argtypes = [vp, i32, i64, i32]
        L.rift_ile_reserve.restype = C.c_int
        L.rift_ile_launch_count.argtypes = [vp]
        L.rift_ile_launch_count.restype = i64
        L.rift_ile_kernel_name.argtypes = [vp]
        L.rift_ile_kernel_name.restype = C.c_char_p
        L.rift_ile_profile.argtypes = [vp, i32]
        L.rift_ile_profile.restype = C.c_int
        L.rift_ile_profile_read.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
        L.rift_ile_profile_read.restype = C.c_int
        L.rift_ile_fma_peak.argtypes = [i32, i32, C.POINTER(dbl), vp]
        L.rift_ile_fma_peak.restype = C.c_int
        L.rift_ile_destroy.argtypes = [vp]
        L.rift_ile_destroy.restype = C.c_int
        # include/rift_ac.h
        L.rift_ac_create.argtypes = [i32, i32, vp, vp, C.POINTER(vp)]
        L.rift_ac_create.restype = C.c_int
        L.rift_ac_draw.argtypes = [vp, i64, C.c_uint64, C.c_uint64, C.POINTER(vp), vp, vp]
        L.rift_ac_draw.restype = C.c_int
        L.rift_ac_update.argtypes = [vp, vp, dbl, dbl]
        L.rift_ac_update.restype = C.c_int
        L.rift_ac_update_dims.argtypes = [vp, vp, dbl, dbl, vp]
        L.rift_ac_update_dims.restype = C.c_int
        L.rift_ac_get_masses.argtypes = [vp, vp]
        L.rift_ac_get_masses.restype = C.c_int
        L.rift_ac_ile_ln_weight.argtypes = [i64, C.POINTER(vp), dbl, dbl, vp, vp, vp]
        L.rift_ac_ile_ln_weight.restype = C.c_int
        L.rift_ac_destroy.argtypes = [vp]
        L.rift_ac_destroy.restype = C.c_int
        L.rift_ile_strerror.argtypes = [C.c_int]
        L.rift_ile_strerror.restype = C.c_char_p
        L.rift_ile_last_error.argtypes = [vp]
        L.rift_ile_last_error.restype = C.c_char_p
        L.rift_gmm_create.argtypes = [i32, i32, vp, vp, C.POINTER(vp)]
        L.rift_gmm_set_model.argtypes = [vp, vp, vp, vp, dbl]
        L.rift_gmm_get_model.argtypes = [vp, vp, vp, vp, C.POINTER(dbl)]
        L.rift_gmm_fit.argtypes = [vp, i64, C.POINTER(vp), vp, i32, dbl, dbl, i32, C.POINTER(i32), C.POINTER(dbl), vp]
        L.rift_gmm_fit_tempered.argtypes = [vp, i64, C.POINTER(vp), vp, dbl, i32, dbl, dbl, i32, C.POINTER(dbl), C.POINTER(i32),
                                            C.POINTER(dbl), vp]
        L.rift_gmm_draw.argtypes = [vp, i64, C.c_uint64, C.c_uint64, C.POINTER(vp), vp, C.POINTER(i64), vp]
        L.rift_gmm_ln_density.argtypes = [vp, i64, C.POINTER(vp), vp, vp]
        L.rift_gmm_box_mass.argtypes = [vp, vp]
        L.rift_gmm_destroy.argtypes = [vp]
        L.rift_gmm_add.argtypes = [i64, i32, C.POINTER(vp), vp, vp]
        for name in GMM_EXPORTS:
            getattr(L, name).restype = C.c_int
        L.rift_ile_rho_guess.argtypes = [vp, vp]
        L.rift_ile_rho_guess.restype = C.c_int
        L.rift_sky_network_frame.argtypes = [vp, vp, vp]
        L.rift_sky_network_frame.restype = C.c_int
        L.rift_sky_network_to_radec.argtypes = [i64, vp, dbl, vp, vp, vp, vp, vp]
        L.rift_sky_network_to_radec.restype = C.c_int
        L.rift_sky_radec_to_network.argtypes = [i64, vp, dbl, vp, vp, vp, vp, vp]
        L.rift_sky_radec_to_network.restype = C.c_int
        L.rift_ile_reduce_static.argtypes = [i32, i64, vp, vp, vp, vp]
        L.rift_ile_reduce_static.restype = C.c_int
        L.rift_ile_reduce_static_error.argtypes = []
        L.rift_ile_reduce_static_error.restype = C.c_char_p
        _lib = L
    return _lib


def _ptr(x) -> Optional[int]:
    """Address of a device tensor / numpy array / raw int; None stays NULL."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(type(x))


def _check(rc: int, h=None):
    if rc != RIFT_OK:
        msg = lib().rift_ile_strerror(rc).decode()
        if h:
            detail = lib().rift_ile_last_error(h).decode()
            if detail:
                msg = f"{msg} ({detail})"
        raise RiftError(rc, msg)


def _params6(params) -> "C.Array":
    """params: a [6][N] device tensor or a sequence of six device arrays (fp64, contiguous)."""
    ptrs = []
    if hasattr(params, "data_ptr") and not isinstance(params, (list, tuple)):
        if params.shape[0] != 6:
            raise ValueError("params must be [6][N]")
        for d in range(6):
            row = params[d]
            if hasattr(row, "is_contiguous") and not row.is_contiguous():
                raise ValueError("params rows must be contiguous")
            ptrs.append(_ptr(row))
    else:
        if len(params) != 6:
            raise ValueError("params must have six entries")
        ptrs = [_ptr(p) for p in params]
    return (C.c_void_p * 6)(*ptrs)


def rift_ile_strerror(code: int) -> str:
    return lib().rift_ile_strerror(int(code)).decode()


def rift_ile_last_error(h) -> str:
    return lib().rift_ile_last_error(h).decode()


def rift_ile_create(det_location_m, det_response, gmst_rad: float, mode_l, mode_m, n_points: int, n_t: int,
                    delta_t: float, n_tau: int, d_ref_mpc: float, Q, U, V, input_mem: int = RIFT_MEM_HOST,
                    precision: int = RIFT_PREC_FP64, q_storage: Optional[int] = None):
    """Returns an opaque handle (ctypes.c_void_p).  Q/U/V: numpy complex128 (host) or device tensors."""
    loc = np.ascontiguousarray(det_location_m, dtype=np.float64)
    resp = np.ascontiguousarray(det_response, dtype=np.float64)
    ml = np.ascontiguousarray(mode_l, dtype=np.int32)
    mm = np.ascontiguousarray(mode_m, dtype=np.int32)
    keep = []
    if input_mem == RIFT_MEM_HOST:
        Q, U, V = (np.ascontiguousarray(a, dtype=np.complex128) for a in (Q, U, V))
        keep = [Q, U, V]
    if q_storage is None:
        q_storage = RIFT_Q_C64 if precision == RIFT_PREC_MIXED else RIFT_Q_C128
    cfg = _Config(int(loc.shape[0]), loc.ctypes.data, resp.ctypes.data, float(gmst_rad), int(ml.size), ml.ctypes.data,
                  mm.ctypes.data, int(n_points), int(n_t), float(delta_t), int(n_tau), float(d_ref_mpc), _ptr(Q),
                  _ptr(U), _ptr(V), int(input_mem), int(precision), int(q_storage))
    h = C.c_void_p()
    _check(lib().rift_ile_create(C.byref(cfg), C.byref(h)))
    del keep
    return h


def rift_ile_destroy(h) -> None:
    _check(lib().rift_ile_destroy(h))


def rift_ile_eval_batch(h, intrinsic_ids: Sequence[int], n_per_seg: int, params, lnL_out, shift_out=None,
                        cuda_stream: int = 0) -> None:
    ids = np.ascontiguousarray(intrinsic_ids, dtype=np.int32)
    _check(lib().rift_ile_eval_batch(h, int(ids.size), ids.ctypes.data, int(n_per_seg), _params6(params), _ptr(lnL_out),
                                     _ptr(shift_out), int(cuda_stream) or None), h)


def rift_ile_eval_batch_host(h, intrinsic_ids: Sequence[int], n_per_seg: int, params, ln_weight, lnL_out,
                             n_slices: int = 0, cuda_stream: int = 0) -> None:
    """params: [6][N] HOST array (numpy, or a pinned torch CPU tensor) or six host arrays; lnL_out: HOST array [N]."""
    ids = np.ascontiguousarray(intrinsic_ids, dtype=np.int32)
    _check(lib().rift_ile_eval_batch_host(h, int(ids.size), ids.ctypes.data, int(n_per_seg), _params6(params),
                                          _ptr(ln_weight), _ptr(lnL_out), int(n_slices), int(cuda_stream) or None), h)


def rift_ile_eval_batch_dmarg(h, intrinsic_ids: Sequence[int], n_per_seg: int, params5, d_min_mpc: float, d_max_mpc: float,
                              n_dist: int, lnL_out, shift_out=None, cuda_stream: int = 0) -> None:
    """params5: a [5][N] (or [6][N]: the distance row is ignored) device tensor or five device arrays."""
    ids = np.ascontiguousarray(intrinsic_ids, dtype=np.int32)
    rows = [params5[d] for d in range(5)]
    ptrs = (C.c_void_p * 5)(*[_ptr(r) for r in rows])
    _check(lib().rift_ile_eval_batch_dmarg(h, int(ids.size), ids.ctypes.data, int(n_per_seg), ptrs, float(d_min_mpc),
                                           float(d_max_mpc), int(n_dist), _ptr(lnL_out), _ptr(shift_out),
                                           int(cuda_stream) or None), h)


def rift_ile_precompute(n_points: int, n_det: int, n_modes: int, h_modes, data, weight, freq_hz_host, freq_hz, n_t: int,
                        delta_t: float, Q, U, V, cuda_stream: int = 0) -> None:
    """Q, U, V (device, complex128) from the frequency series h_modes [P][K][M][NF], data [P][K][NF] (device, complex128),
    weight [K][NF], freq_hz [NF] (device, fp64); freq_hz_host: the frequencies as a host array."""
    fh = np.ascontiguousarray(freq_hz_host, dtype=np.float64)
    _check(lib().rift_ile_precompute(int(n_points), int(n_det), int(n_modes), int(fh.size), _ptr(h_modes), _ptr(data),
                                     _ptr(weight), fh.ctypes.data, _ptr(freq_hz), int(n_t), float(delta_t), _ptr(Q), _ptr(U),
                                     _ptr(V), int(cuda_stream) or None))


def rift_ile_staged(h) -> dict:
    """Device copies left by the last eval_batch_host: dict(params=[6 addresses], ln_weight=address or None, lnL=address, n)."""
    p = (C.c_void_p * 6)()
    w, l, n = C.c_void_p(), C.c_void_p(), C.c_int64()
    _check(lib().rift_ile_staged(h, p, C.byref(w), C.byref(l), C.byref(n)), h)
    return dict(params=[int(x) for x in p], ln_weight=(int(w.value) if w.value else None), lnL=int(l.value), n=int(n.value))


def rift_ile_geometry(h, intrinsic_id: int, n: int, params, F=None, Y=None, shift=None, quad=None,
                      cuda_stream: int = 0) -> None:
    _check(lib().rift_ile_geometry(h, int(intrinsic_id), int(n), _params6(params), _ptr(F), _ptr(Y), _ptr(shift),
                                   _ptr(quad), int(cuda_stream) or None), h)


def rift_ile_reduce(h, n_seg: int, n_per_seg: int, lnL, ln_weight=None, params=None, lo=None, hi=None,
                    n_bins: int = 0, merge: int = 0, want_hist: bool = False, cuda_stream: int = 0) -> dict:
    """Returns dict(lnZ, rel_err, n_eff, n_ess [n_seg] numpy fp64, hist [n_seg][6][n_bins] or None)."""
    out = [np.empty(n_seg, dtype=np.float64) for _ in range(4)]
    hist = np.empty((n_seg, 6, n_bins), dtype=np.float64) if want_hist else None
    lo_ = None if lo is None else np.ascontiguousarray(lo, dtype=np.float64)
    hi_ = None if hi is None else np.ascontiguousarray(hi, dtype=np.float64)
    _check(lib().rift_ile_reduce(h, int(n_seg), int(n_per_seg), _ptr(lnL), _ptr(ln_weight),
                                 None if params is None else _params6(params), _ptr(lo_), _ptr(hi_), int(n_bins),
                                 int(merge), *[o.ctypes.data for o in out], _ptr(hist), int(cuda_stream) or None), h)
    return dict(lnZ=out[0], rel_err=out[1], n_eff=out[2], n_ess=out[3], hist=hist)


def rift_ile_reduce_static(n_seg: int, n_per_seg: int, lnL, ln_weight, out, cuda_stream: int = 0) -> None:
    """Allocation-free reduce: out is a DEVICE fp64 [4][n_seg] array (lnZ, rel_err, n_eff, n_ess), filled asynchronously."""
    rc = lib().rift_ile_reduce_static(int(n_seg), int(n_per_seg), _ptr(lnL), _ptr(ln_weight), _ptr(out),
                                      int(cuda_stream) or None)
    if rc != RIFT_OK:
        raise RiftError(rc, f"{lib().rift_ile_strerror(rc).decode()} ({lib().rift_ile_reduce_static_error().decode()})")


class GmmHandle:
    """Opaque rift_gmm_t* with the shape needed to marshal arrays."""
    def __init__(self, ptr, n_dim, n_comp):
        self.ptr, self.n_dim, self.n_comp = ptr, n_dim, n_comp


def _xptrs(g: "GmmHandle", x):
    if len(x) != g.n_dim:
        raise ValueError("x must hold one device array per dimension")
    return (C.c_void_p * g.n_dim)(*[_ptr(v) for v in x])


def rift_gmm_create(n_dim: int, n_comp: int, lo, hi) -> GmmHandle:
    lo_ = np.ascontiguousarray(lo, dtype=np.float64)
    hi_ = np.ascontiguousarray(hi, dtype=np.float64)
    if lo_.size != n_dim or hi_.size != n_dim:
        raise ValueError("lo, hi must have n_dim entries")
    out = C.c_void_p()
    _check(lib().rift_gmm_create(int(n_dim), int(n_comp), lo_.ctypes.data, hi_.ctypes.data, C.byref(out)))
    return GmmHandle(out, int(n_dim), int(n_comp))


def rift_gmm_set_model(g: GmmHandle, mu, cov, pi, n_trained: float = 0.0) -> None:
    mu_ = np.ascontiguousarray(mu, dtype=np.float64).reshape(g.n_comp, g.n_dim)
    cov_ = np.ascontiguousarray(cov, dtype=np.float64).reshape(g.n_comp, g.n_dim, g.n_dim)
    pi_ = np.ascontiguousarray(pi, dtype=np.float64).reshape(g.n_comp)
    _check(lib().rift_gmm_set_model(g.ptr, mu_.ctypes.data, cov_.ctypes.data, pi_.ctypes.data, float(n_trained)))


def rift_gmm_get_model(g: GmmHandle):
    """(mu [K][d], cov [K][d][d], pi [K], n_trained)."""
    mu = np.empty((g.n_comp, g.n_dim))
    cov = np.empty((g.n_comp, g.n_dim, g.n_dim))
    pi = np.empty(g.n_comp)
    nt = C.c_double()
    _check(lib().rift_gmm_get_model(g.ptr, mu.ctypes.data, cov.ctypes.data, pi.ctypes.data, C.byref(nt)))
    return mu, cov, pi, nt.value


def rift_gmm_fit(g: GmmHandle, n: int, x, ln_w, n_iter: int, tol: float = 0.0, reg: float = 0.0, merge: int = 0,
                 cuda_stream: int = 0):
    """EM on device arrays x (one per dimension) with log-weights ln_w (or None); returns (iterations done, ln L)."""
    it, ll = C.c_int32(), C.c_double()
    _check(lib().rift_gmm_fit(g.ptr, int(n), _xptrs(g, x), _ptr(ln_w), int(n_iter), float(tol), float(reg), int(merge),
                              C.byref(it), C.byref(ll), int(cuda_stream) or None))
    return it.value, ll.value


def rift_gmm_fit_tempered(g: GmmHandle, n: int, x, ln_w, ess_min: float, n_iter: int, tol: float = 0.0, reg: float = 0.0,
                          merge: int = 0, cuda_stream: int = 0):
    """rift_gmm_fit on weights tempered so that their effective sample size reaches ess_min; returns (temper, iterations, ln L)."""
    it, ll, tp = C.c_int32(), C.c_double(), C.c_double()
    _check(lib().rift_gmm_fit_tempered(g.ptr, int(n), _xptrs(g, x), _ptr(ln_w), float(ess_min), int(n_iter), float(tol),
                                       float(reg), int(merge), C.byref(tp), C.byref(it), C.byref(ll), int(cuda_stream) or None))
    return tp.value, it.value, ll.value


def rift_gmm_draw(g: GmmHandle, n: int, seed: int, offset: int, x, ln_ps=None, want_failed: bool = False, cuda_stream: int = 0):
    nf = C.c_int64(0)
    _check(lib().rift_gmm_draw(g.ptr, int(n), int(seed), int(offset), _xptrs(g, x), _ptr(ln_ps),
                               C.byref(nf) if want_failed else None, int(cuda_stream) or None))
    return nf.value if want_failed else None


def rift_gmm_ln_density(g: GmmHandle, n: int, x, ln_ps, cuda_stream: int = 0) -> None:
    _check(lib().rift_gmm_ln_density(g.ptr, int(n), _xptrs(g, x), _ptr(ln_ps), int(cuda_stream) or None))


def rift_gmm_box_mass(g: GmmHandle) -> np.ndarray:
    Z = np.empty(g.n_comp)
    _check(lib().rift_gmm_box_mass(g.ptr, Z.ctypes.data))
    return Z


def rift_gmm_add(n: int, terms, out, cuda_stream: int = 0) -> None:
    """out = terms[0] + terms[1] + ... on the device."""
    arr = (C.c_void_p * len(terms))(*[_ptr(t) for t in terms])
    _check(lib().rift_gmm_add(int(n), len(terms), arr, _ptr(out), int(cuda_stream) or None))


def rift_gmm_destroy(g: GmmHandle) -> None:
    _check(lib().rift_gmm_destroy(g.ptr))


def rift_ile_rho_guess(h, n_points: int) -> np.ndarray:
    """rho_guess [n_points] (Eq. (D7), reading A14)."""
    out = np.empty(int(n_points), dtype=np.float64)
    _check(lib().rift_ile_rho_guess(h, out.ctypes.data), h)
    return out


def rift_sky_network_frame(loc_a_m, loc_b_m) -> np.ndarray:
    """R [3][3] (columns x', y', z') of the frame whose pole points from detector a to detector b."""
    a = np.ascontiguousarray(loc_a_m, dtype=np.float64)
    b = np.ascontiguousarray(loc_b_m, dtype=np.float64)
    R = np.empty((3, 3), dtype=np.float64)
    _check(lib().rift_sky_network_frame(a.ctypes.data, b.ctypes.data, R.ctypes.data))
    return R


def rift_sky_network_to_radec(n: int, R, gmst_rad: float, lam, beta, ra, dec, cuda_stream: int = 0) -> None:
    R_ = np.ascontiguousarray(R, dtype=np.float64)
    _check(lib().rift_sky_network_to_radec(int(n), R_.ctypes.data, float(gmst_rad), _ptr(lam), _ptr(beta), _ptr(ra), _ptr(dec),
                                           int(cuda_stream) or None))


def rift_sky_radec_to_network(n: int, R, gmst_rad: float, ra, dec, lam, beta, cuda_stream: int = 0) -> None:
    R_ = np.ascontiguousarray(R, dtype=np.float64)
    _check(lib().rift_sky_radec_to_network(int(n), R_.ctypes.data, float(gmst_rad), _ptr(ra), _ptr(dec), _ptr(lam), _ptr(beta),
                                           int(cuda_stream) or None))


def rift_ile_set_kernel(h, variant: int) -> None:
    _check(lib().rift_ile_set_kernel(h, int(variant)), h)


def rift_ile_set_option(h, option: int, value: int) -> None:
    _check(lib().rift_ile_set_option(h, int(option), int(value)), h)


def rift_ile_reserve(h, n_seg: int, n_per_seg: int, n_bins: int = 0) -> None:
    _check(lib().rift_ile_reserve(h, int(n_seg), int(n_per_seg), int(n_bins)), h)


def rift_ile_launch_count(h) -> int:
    return int(lib().rift_ile_launch_count(h))


def rift_ile_kernel_name(h) -> str:
    return lib().rift_ile_kernel_name(h).decode()


def rift_ile_profile(h, enable: bool) -> None:
    _check(lib().rift_ile_profile(h, int(bool(enable))), h)


def rift_ile_profile_read(h) -> dict:
    """dict(ms=[geometry, lnl, reduce, sort], launches=[...]) summed since the last read."""
    ms = (C.c_double * 4)()
    nl = (C.c_int64 * 4)()
    _check(lib().rift_ile_profile_read(h, ms, nl), h)
    return dict(ms=[float(x) for x in ms], launches=[int(x) for x in nl])


def rift_ile_fma_peak(mode: int, iters: int = 4096, cuda_stream: int = 0) -> float:
    """mode: 0 FFMA, 1 DFMA, 2 FFMA register tile, 3/4/5 FP64 mma.sync m8n8k4/m16n8k8/m16n8k16, 6 m8n8k4 + DFMA."""
    v = C.c_double()
    _check(lib().rift_ile_fma_peak(int(mode), int(iters), C.byref(v), int(cuda_stream) or None))
    return float(v.value)


# ---------------------------------------------------------------------------------------------- include/rift_ac.h
def rift_ac_create(n_dim: int, n_bins: int, lo, hi):
    """Adaptive-cartesian sampler handle (uniform bin masses).  lo, hi: host sequences of length n_dim."""
    lo_ = np.ascontiguousarray(lo, dtype=np.float64)
    hi_ = np.ascontiguousarray(hi, dtype=np.float64)
    if lo_.size != n_dim or hi_.size != n_dim:
        raise ValueError("lo, hi must have n_dim entries")
    h = C.c_void_p()
    _check(lib().rift_ac_create(int(n_dim), int(n_bins), lo_.ctypes.data, hi_.ctypes.data, C.byref(h)))
    return h


def rift_ac_draw(h, n: int, seed: int, offset: int, x, ln_ps, cuda_stream: int = 0) -> None:
    """x: a [n_dim][n] device tensor (contiguous rows) or a sequence of n_dim device arrays; ln_ps: device [n]."""
    rows = [x[d] for d in range(x.shape[0])] if hasattr(x, "shape") and not isinstance(x, (list, tuple)) else list(x)
    ptrs = (C.c_void_p * len(rows))(*[_ptr(r) for r in rows])
    _check(lib().rift_ac_draw(h, int(n), int(seed), int(offset), ptrs, _ptr(ln_ps), int(cuda_stream) or None))


def rift_ac_update(h, hist, floor_mix: float, temper: float = 1.0) -> None:
    hist_ = np.ascontiguousarray(hist, dtype=np.float64)
    _check(lib().rift_ac_update(h, hist_.ctypes.data, float(floor_mix), float(temper)))


def rift_ac_update_dims(h, hist, floor_mix: float, temper: float, adapt) -> None:
    """adapt: one flag per dimension (0 keeps the dimension's current masses), or None for all."""
    hist_ = np.ascontiguousarray(hist, dtype=np.float64)
    adapt_ = None if adapt is None else np.ascontiguousarray(adapt, dtype=np.int32)
    if adapt_ is not None and adapt_.size != hist_.shape[0]:
        raise ValueError("adapt must have one entry per dimension")
    _check(lib().rift_ac_update_dims(h, hist_.ctypes.data, float(floor_mix), float(temper),
                                     None if adapt_ is None else adapt_.ctypes.data))


def rift_ac_get_masses(h, n_dim: int, n_bins: int) -> np.ndarray:
    out = np.empty((n_dim, n_bins), dtype=np.float64)
    _check(lib().rift_ac_get_masses(h, out.ctypes.data))
    return out


def rift_ac_ile_ln_weight(n: int, params, d_min_mpc: float, d_max_mpc: float, ln_ps, ln_weight,
                          cuda_stream: int = 0) -> None:
    _check(lib().rift_ac_ile_ln_weight(int(n), _params6(params), float(d_min_mpc), float(d_max_mpc), _ptr(ln_ps),
                                       _ptr(ln_weight), int(cuda_stream) or None))


def rift_ac_destroy(h) -> None:
    _check(lib().rift_ac_destroy(h))
