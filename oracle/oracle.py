"""ctypes marshalling for oracle/rift_oracle.c (no arithmetic here beyond argument packing)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rift_oracle.c")
_SRC_DM = os.path.join(_HERE, "dmarg_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

__all__ = ["build", "lib", "num_threads", "antenna", "harmonics", "swsh_m2", "delays", "lnl_core",
           "logmeanexp", "eval_batch", "ReduceState", "reduce", "geometry_at", "dmarg_rule", "dmarg_core",
           "eval_batch_dmarg"]


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp -> oracle/liboracle.so (rebuilt when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_DM)):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
               _SRC, _SRC_DM, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_bp = C.POINTER(C.c_uint8)


def _d(a):
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_antenna_one.argtypes = [C.c_double] * 4 + [_dp, _dp]
        L.oracle_antenna_one.restype = None
        L.oracle_swsh_m2.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, _dp]
        L.oracle_swsh_m2.restype = C.c_int
        L.oracle_delay_one.argtypes = [C.c_double, C.c_double, C.c_double, _dp, C.c_double, _dp, _ip, _bp]
        L.oracle_delay_one.restype = None
        L.oracle_lnl_core.argtypes = [C.c_int] * 4 + [_dp, _dp, C.c_double, _ip, _dp, _dp, _dp, _dp, _dp]
        L.oracle_lnl_core.restype = C.c_double
        L.oracle_logmeanexp.argtypes = [C.c_int, _dp]
        L.oracle_logmeanexp.restype = C.c_double
        L.oracle_eval_batch.argtypes = ([C.c_int, _dp, _dp, C.c_double, C.c_int, _ip, _ip, C.c_int, C.c_int,
                                         C.c_double, C.c_double, _dp, _dp, _dp, C.c_int64] + [_dp] * 6
                                        + [_dp, _ip, _bp])
        L.oracle_eval_batch.restype = C.c_int
        L.oracle_reduce_new.argtypes = [C.c_int32, C.c_int]
        L.oracle_reduce_new.restype = C.c_void_p
        L.oracle_reduce_free.argtypes = [C.c_void_p]
        L.oracle_reduce_free.restype = None
        L.oracle_reduce_accumulate.argtypes = [C.c_void_p, C.c_int64, _dp, _dp, C.POINTER(_dp), _dp, _dp]
        L.oracle_reduce_accumulate.restype = None
        L.oracle_reduce_finalize.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp, _dp]
        L.oracle_reduce_finalize.restype = None
        L.oracle_dmarg_rule.argtypes = [C.c_double, C.c_double, C.c_double, C.c_int, _dp, _dp]
        L.oracle_dmarg_rule.restype = None
        L.oracle_dmarg_core.argtypes = [C.c_int, _dp] + [C.c_double] * 5 + [C.c_int]
        L.oracle_dmarg_core.restype = C.c_double
        L.oracle_eval_batch_dmarg.argtypes = ([C.c_int, _dp, _dp, C.c_double, C.c_int, _ip, _ip, C.c_int, C.c_int,
                                               C.c_double, C.c_double, _dp, _dp, _dp, C.c_int64] + [_dp] * 5
                                              + [C.c_double, C.c_double, C.c_double, C.c_int, _dp, _ip, _bp])
        L.oracle_eval_batch_dmarg.restype = C.c_int
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _c128(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.complex128)


def antenna(ra, dec, psi, gmst: float, response) -> np.ndarray:
    """F[n][K] complex = F+ + i Fx for each sample and detector (response: [K][3][3])."""
    ra, dec, psi = (np.atleast_1d(_f64(x)) for x in (ra, dec, psi))
    D = _f64(response).reshape(-1, 9)
    out = np.empty((ra.size, D.shape[0]), dtype=np.complex128)
    tmp = np.empty(2, dtype=np.float64)
    L = lib()
    for i in range(ra.size):
        for k in range(D.shape[0]):
            L.oracle_antenna_one(ra[i], dec[i], psi[i], gmst, _d(D[k]), _d(tmp))
            out[i, k] = complex(tmp[0], tmp[1])
    return out


def swsh_m2(l: int, m: int, theta: float, phi: float) -> complex:
    tmp = np.empty(2, dtype=np.float64)
    if lib().oracle_swsh_m2(int(l), int(m), float(theta), float(phi), _d(tmp)) != 0:
        raise ValueError((l, m))
    return complex(tmp[0], tmp[1])


def harmonics(iota, phi_ref, mode_l: Sequence[int], mode_m: Sequence[int]) -> np.ndarray:
    """Y[n][M] = -2Y_lm(iota, -phi_ref)."""
    iota, phi_ref = np.atleast_1d(_f64(iota)), np.atleast_1d(_f64(phi_ref))
    out = np.empty((iota.size, len(mode_l)), dtype=np.complex128)
    for i in range(iota.size):
        for a, (l, m) in enumerate(zip(mode_l, mode_m)):
            out[i, a] = swsh_m2(l, m, iota[i], -phi_ref[i])
    return out


def delays(ra, dec, gmst: float, location, delta_t: float) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """(dt[n][K] seconds, shift[n][K] int32, fragile[n][K] uint8)."""
    ra, dec = np.atleast_1d(_f64(ra)), np.atleast_1d(_f64(dec))
    r = _f64(location).reshape(-1, 3)
    dt = np.empty((ra.size, r.shape[0]), dtype=np.float64)
    sh = np.empty((ra.size, r.shape[0]), dtype=np.int32)
    fr = np.empty((ra.size, r.shape[0]), dtype=np.uint8)
    L = lib()
    d, s, f = C.c_double(), C.c_int32(), C.c_uint8()
    for i in range(ra.size):
        for k in range(r.shape[0]):
            L.oracle_delay_one(ra[i], dec[i], gmst, _d(r[k]), delta_t, C.byref(d), C.byref(s), C.byref(f))
            dt[i, k], sh[i, k], fr[i, k] = d.value, s.value, f.value
    return dt, sh, fr


def lnl_core(F, Y, c: float, shift, Q, U, V, n_tau: Optional[int] = None):
    """One sample from its coefficients: returns (lnL_tm, lnL_j[n_tau], quad)."""
    Q, U, V, F, Y = _c128(Q), _c128(U), _c128(V), _c128(F), _c128(Y)
    K, M, n_t = Q.shape
    n_tau = n_t if n_tau is None else int(n_tau)
    sh = np.ascontiguousarray(shift, dtype=np.int32)
    series = np.empty(n_tau, dtype=np.float64)
    quad = C.c_double()
    v = lib().oracle_lnl_core(K, M, n_t, n_tau, _d(F.view(np.float64)), _d(Y.view(np.float64)), float(c),
                              sh.ctypes.data_as(_ip), _d(Q.view(np.float64)), _d(U.view(np.float64)),
                              _d(V.view(np.float64)), _d(series), C.byref(quad))
    return float(v), series, quad.value


def logmeanexp(x) -> float:
    x = _f64(x)
    return float(lib().oracle_logmeanexp(int(x.size), _d(x)))


def eval_batch(location, response, gmst: float, mode_l, mode_m, delta_t: float, d_ref_mpc: float,
               Q, U, V, params, n_tau: Optional[int] = None, want_shifts: bool = True):
    """All samples of one intrinsic point.  params: [6][n].  Returns (lnL[n], shift[n][K], fragile[n])."""
    Q, U, V = _c128(Q), _c128(U), _c128(V)
    K, M, n_t = Q.shape
    n_tau = n_t if n_tau is None else int(n_tau)
    P = [_f64(p) for p in params]
    n = P[0].size
    r, D = _f64(location).reshape(K, 3), _f64(response).reshape(K, 9)
    ml = np.ascontiguousarray(mode_l, dtype=np.int32)
    mm = np.ascontiguousarray(mode_m, dtype=np.int32)
    lnL = np.empty(n, dtype=np.float64)
    sh = np.empty((n, K), dtype=np.int32)
    fr = np.empty(n, dtype=np.uint8)
    rc = lib().oracle_eval_batch(K, _d(r), _d(D), float(gmst), M, ml.ctypes.data_as(_ip), mm.ctypes.data_as(_ip),
                                 n_t, n_tau, float(delta_t), float(d_ref_mpc), _d(Q.view(np.float64)),
                                 _d(U.view(np.float64)), _d(V.view(np.float64)), n, *[_d(p) for p in P],
                                 _d(lnL), sh.ctypes.data_as(_ip), fr.ctypes.data_as(_bp))
    if rc != 0:
        raise ValueError("oracle_eval_batch: invalid arguments")
    return lnL, sh, fr


class ReduceState:
    """Mergeable sample-axis reduce state of one segment (Eq. (20)-(21))."""

    def __init__(self, n_bins: int = 0, want_hist: bool = False):
        self.n_bins = int(n_bins)
        self.want_hist = bool(want_hist and n_bins > 0)
        self._h = lib().oracle_reduce_new(self.n_bins, int(self.want_hist))

    def __del__(self):
        try:
            lib().oracle_reduce_free(self._h)
        except Exception:
            pass

    def accumulate(self, lnL, ln_w=None, params=None, lo=None, hi=None):
        lnL = _f64(lnL)
        lw = None if ln_w is None else _f64(ln_w)
        if self.want_hist and params is not None:
            P = [_f64(p) for p in params]
            arr = (_dp * 6)(*[_d(p) for p in P])
            lo_, hi_ = _f64(lo), _f64(hi)
            lib().oracle_reduce_accumulate(self._h, lnL.size, _d(lnL), None if lw is None else _d(lw), arr,
                                           _d(lo_), _d(hi_))
        else:
            lib().oracle_reduce_accumulate(self._h, lnL.size, _d(lnL), None if lw is None else _d(lw), None,
                                           None, None)

    def finalize(self):
        v = [C.c_double() for _ in range(4)]
        hist = np.zeros((6, self.n_bins), dtype=np.float64) if self.want_hist else None
        lib().oracle_reduce_finalize(self._h, *[C.byref(x) for x in v], None if hist is None else _d(hist))
        return dict(lnZ=v[0].value, rel_err=v[1].value, n_eff=v[2].value, n_ess=v[3].value, hist=hist)


def reduce(lnL, ln_w=None, params=None, lo=None, hi=None, n_bins: int = 0):
    st = ReduceState(n_bins, want_hist=params is not None)
    st.accumulate(lnL, ln_w, params, lo, hi)
    return st.finalize()


def geometry_at(theta, location, response, gmst, mode_l, mode_m, delta_t):
    """(F[K], Y[M], shift[K]) at one extrinsic point theta[6] (for the input generator)."""
    F = antenna(theta[0], theta[1], theta[2], gmst, response)[0]
    Y = harmonics(theta[3], theta[4], mode_l, mode_m)[0]
    _dt, sh, _fr = delays(theta[0], theta[1], gmst, location, delta_t)
    return F, Y, sh[0]


# ---------------------------------------------------------------------------------------------- dmarg_oracle.c (NEXT-2)
def dmarg_rule(d_min: float, d_max: float, alpha: float, n_panels: int):
    """(D[8 n_panels], W[8 n_panels]) of the composite Gauss-Legendre rule in ln D (W includes the prior density)."""
    D = np.empty(8 * n_panels, dtype=np.float64)
    W = np.empty(8 * n_panels, dtype=np.float64)
    lib().oracle_dmarg_rule(float(d_min), float(d_max), float(alpha), int(n_panels), _d(D), _d(W))
    return D, W


def dmarg_core(x, b: float, d_ref: float, d_min: float, d_max: float, alpha: float, n_panels: int) -> float:
    x = _f64(x)
    return float(lib().oracle_dmarg_core(int(x.size), _d(x), float(b), float(d_ref), float(d_min), float(d_max),
                                         float(alpha), int(n_panels)))


def eval_batch_dmarg(location, response, gmst: float, mode_l, mode_m, delta_t: float, d_ref_mpc: float, Q, U, V,
                     params5, d_min: float, d_max: float, n_panels: int, alpha: float = 2.0, n_tau: Optional[int] = None):
    """Distance-marginalised lnL of all samples of one intrinsic point.  params5: [5][n] (ra, dec, psi, iota, phi_ref).
    Returns (lnL[n], shift[n][K], fragile[n])."""
    Q, U, V = _c128(Q), _c128(U), _c128(V)
    K, M, n_t = Q.shape
    n_tau = n_t if n_tau is None else int(n_tau)
    P = [_f64(p) for p in params5[:5]]
    n = P[0].size
    r, D = _f64(location).reshape(K, 3), _f64(response).reshape(K, 9)
    ml = np.ascontiguousarray(mode_l, dtype=np.int32)
    mm = np.ascontiguousarray(mode_m, dtype=np.int32)
    lnL = np.empty(n, dtype=np.float64)
    sh = np.empty((n, K), dtype=np.int32)
    fr = np.empty(n, dtype=np.uint8)
    rc = lib().oracle_eval_batch_dmarg(K, _d(r), _d(D), float(gmst), M, ml.ctypes.data_as(_ip), mm.ctypes.data_as(_ip),
                                       n_t, n_tau, float(delta_t), float(d_ref_mpc), _d(Q.view(np.float64)),
                                       _d(U.view(np.float64)), _d(V.view(np.float64)), n, *[_d(p) for p in P],
                                       float(d_min), float(d_max), float(alpha), int(n_panels), _d(lnL),
                                       sh.ctypes.data_as(_ip), fr.ctypes.data_as(_bp))
    if rc != 0:
        raise ValueError("oracle_eval_batch_dmarg: invalid arguments")
    return lnL, sh, fr
