"""Seeded synthetic inputs for the ILE factored-likelihood hot path.

This module serves BOTH the CPU oracle (tests) and the CUDA library (tests, bench) and therefore
holds none of the method's arithmetic: no antenna pattern, no harmonics, no delays, no lnL.
Whatever the data recipe needs from the method (the complex coefficients F_k * Y_lm and the integer
delays of the injected "true" point) is PASSED IN by the caller, which obtains it either from the
oracle (tests) or from the CUDA geometry kernel (bench).

What it produces (BASELINE.json configs[0..4], readings A3(i), A7-A12 of SURVEY.md section 8(c),
restated in DESIGN.md section 4):

* detector constants (site position r_k in metres, response tensor D_k = (x x^T - y y^T)/2),
* mode lists,
* per intrinsic point: Q[K][M][N_t] (complex128), U[K][M][M] (Hermitian), V[K][M][M] (symmetric)
  following Eq. (D4a-c) with the literal one-sided 4*df recipe of configs[0],
* extrinsic samples (RA, dec, psi, iota, phi_ref, D) and their ln importance weights.

The paper's own workloads (GWOSC strain, lalsimulation waveforms, measured PSDs; PAPER.md:170,
:716, :508, :748) are not available here; these inputs stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional, Sequence, Tuple

import numpy as np

C_LIGHT = 299792458.0            # m/s
D_REF_MPC = 1000.0               # reading A7
D_MIN_MPC, D_MAX_MPC = 50.0, 2000.0
SEED_BASE = 221007912
F_LOW_HZ, F_HIGH_HZ, N_FREQ = 20.0, 1024.0, 4096   # configs[0]: "4096 bins over 20-1024 Hz"
PARAM_NAMES = ("ra", "dec", "psi", "iota", "phi_ref", "dist_mpc")

# ----------------------------------------------------------------------------------------------
# Detector geometry (reading G1: Earth-fixed frame, metres, arm unit vectors). Public site facts.
# ----------------------------------------------------------------------------------------------
_SITES = {
    "H1": dict(r=(-2.16141492636e6, -3.83469517889e6, 4.60035022664e6),
               x=(-0.22389266154, 0.79983062746, 0.55690487831),
               y=(-0.91397818574, 0.02609403989, -0.40492342125)),
    "L1": dict(r=(-7.42760447238e4, -5.49628371971e6, 3.22425701744e6),
               x=(-0.95457412153, -0.14158077340, -0.26218911324),
               y=(0.29774156894, -0.48791033647, -0.82054461286)),
    "V1": dict(r=(4.54637409900e6, 8.42989697626e5, 4.37857696241e6),
               x=(-0.70045821479, 0.20848948619, 0.68256166277),
               y=(-0.05379255368, -0.96908180549, 0.24080451708)),
}


def response_tensor(xarm: Sequence[float], yarm: Sequence[float]) -> np.ndarray:
    """D = (x (x) x - y (x) y) / 2, symmetric and traceless for unit orthogonal arms."""
    x = np.asarray(xarm, dtype=np.float64)
    y = np.asarray(yarm, dtype=np.float64)
    return 0.5 * (np.outer(x, x) - np.outer(y, y))


def site(name: str) -> Tuple[np.ndarray, np.ndarray]:
    """(location[3] in metres, response[3][3]) for H1 / L1 / V1."""
    s = _SITES[name]
    return np.asarray(s["r"], dtype=np.float64), response_tensor(s["x"], s["y"])


def synthetic_site(rng: np.random.Generator) -> Tuple[np.ndarray, np.ndarray]:
    """Reading A11: a site on a spherical Earth (R = 6.371e6 m) with orthogonal arms in the local
    horizontal plane; sin(lat) ~ U[-1,1], lon ~ U[-pi,pi), x-arm azimuth ~ U[0,2pi)."""
    R = 6.371e6
    sin_lat = rng.uniform(-1.0, 1.0)
    lon = rng.uniform(-math.pi, math.pi)
    az = rng.uniform(0.0, 2.0 * math.pi)
    cos_lat = math.sqrt(max(0.0, 1.0 - sin_lat * sin_lat))
    up = np.array([cos_lat * math.cos(lon), cos_lat * math.sin(lon), sin_lat])
    east = np.array([-math.sin(lon), math.cos(lon), 0.0])
    north = np.cross(up, east)
    xarm = math.cos(az) * east + math.sin(az) * north
    yarm = -math.sin(az) * east + math.cos(az) * north
    return R * up, response_tensor(xarm, yarm)


# ----------------------------------------------------------------------------------------------
# Configs
# ----------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Config:
    index: int
    name: str
    detectors: Tuple[str, ...]          # "H1","L1","V1" or "S0","S1" (seeded synthetic sites)
    modes: Tuple[Tuple[int, int], ...]
    f_s: float
    t_window: float
    n_points: int
    n_samples: int
    psd: str                            # "flat" | "analytic"
    proposal: str                       # "prior" | "gauss_sky"
    mode_amp_decay: bool                # amplitude x 0.5^(l-2)
    rho: float = 12.0                   # reading A7
    gmst: float = 0.0

    @property
    def n_det(self) -> int:
        return len(self.detectors)

    @property
    def n_modes(self) -> int:
        return len(self.modes)

    @property
    def n_t(self) -> int:               # reading A10: N_t = 2*round(T_w f_s)+1  (411, 3277)
        return 2 * int(round(self.t_window * self.f_s)) + 1

    @property
    def delta_t(self) -> float:
        return 1.0 / self.f_s

    def flop_per_eval(self) -> int:     # window term + quadratic term
        return 4 * self.n_det * self.n_modes * self.n_t + 8 * self.n_det * self.n_modes ** 2


def _modes_l(ls: Sequence[int]) -> Tuple[Tuple[int, int], ...]:
    return tuple((l, m) for l in ls for m in range(-l, l + 1))


CONFIGS: Dict[int, Config] = {
    0: Config(0, "C0 tiny", ("H1", "L1"), ((2, -2), (2, 2)), 4096.0, 0.05, 1, 4096, "flat", "prior", False),
    1: Config(1, "C1", ("H1", "L1", "V1"), _modes_l([2]), 4096.0, 0.05, 16, 100_000, "analytic", "prior", False),
    2: Config(2, "C2 higher modes", ("H1", "L1", "V1"), _modes_l([2, 3, 4]), 4096.0, 0.05, 64, 1_000_000,
              "analytic", "gauss_sky", True),
    3: Config(3, "C3 streaming", ("H1", "L1", "V1"), _modes_l([2]), 4096.0, 0.05, 1024, 100_000,
              "analytic", "prior", False),
    # reading A11: 9 modes = (2,m) for all m plus (3,+-2),(3,+-3)
    4: Config(4, "C4 long window", ("H1", "L1", "V1", "S0", "S1"),
              _modes_l([2]) + ((3, -3), (3, -2), (3, 2), (3, 3)), 16384.0, 0.1, 8, 4_000_000,
              "analytic", "prior", True),
}


def with_overrides(cfg: Config, **kw) -> Config:
    d = {f: getattr(cfg, f) for f in cfg.__dataclass_fields__}
    d.update(kw)
    return Config(**d)


def detector_arrays(cfg: Config) -> Tuple[np.ndarray, np.ndarray]:
    """(location[K][3], response[K][3][3]); synthetic sites are seeded by the config index."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 * cfg.index + 900))
    loc, resp = [], []
    for name in cfg.detectors:
        r, d = site(name) if name in _SITES else synthetic_site(rng)
        loc.append(r)
        resp.append(d)
    return np.ascontiguousarray(loc, dtype=np.float64), np.ascontiguousarray(resp, dtype=np.float64)


def mode_arrays(cfg: Config) -> Tuple[np.ndarray, np.ndarray]:
    l = np.array([lm[0] for lm in cfg.modes], dtype=np.int32)
    m = np.array([lm[1] for lm in cfg.modes], dtype=np.int32)
    return l, m


# ----------------------------------------------------------------------------------------------
# Spectra, noise, Q/U/V (literal recipe "LIT", readings A3(i), A8, A9)
# ----------------------------------------------------------------------------------------------
def freq_grid() -> Tuple[np.ndarray, float]:
    df = (F_HIGH_HZ - F_LOW_HZ) / N_FREQ
    return F_LOW_HZ + df * np.arange(N_FREQ, dtype=np.float64), df


def psd(kind: str, f: np.ndarray) -> np.ndarray:
    if kind == "flat":
        return np.ones_like(f)
    if kind == "analytic":
        x = f / 200.0
        return x ** -4 + 1.0 + x ** 2
    raise ValueError(kind)


def point_rng(cfg: Config, point: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + 1000 * cfg.index + point + stream))


def prior_draw(rng: np.random.Generator, n: int) -> np.ndarray:
    """n draws from the extrinsic prior (reading A18). Returns float64 [6][n] in PARAM_NAMES order."""
    out = np.empty((6, n), dtype=np.float64)
    out[0] = rng.uniform(0.0, 2.0 * math.pi, n)
    out[1] = np.arcsin(rng.uniform(-1.0, 1.0, n))
    out[2] = rng.uniform(0.0, math.pi, n)
    out[3] = np.arccos(rng.uniform(-1.0, 1.0, n))
    out[4] = rng.uniform(0.0, 2.0 * math.pi, n)
    u = rng.uniform(0.0, 1.0, n)
    out[5] = np.cbrt(u * (D_MAX_MPC ** 3 - D_MIN_MPC ** 3) + D_MIN_MPC ** 3)
    return out


def true_point(cfg: Config, point: int) -> np.ndarray:
    """The injected extrinsic point of an intrinsic point: one prior draw from the point's seed."""
    return prior_draw(point_rng(cfg, point, stream=250), 1)[:, 0].copy()


_DFT_CACHE: Dict[Tuple[int, float], np.ndarray] = {}


def _dft_matrix(n_t: int, f_s: float) -> np.ndarray:
    """exp(2 pi i f_n t_j), t_j = (j - (N_t-1)/2)/f_s; cached per (N_t, f_s)."""
    key = (n_t, f_s)
    if key not in _DFT_CACHE:
        f, _df = freq_grid()
        t = (np.arange(n_t, dtype=np.float64) - (n_t - 1) / 2.0) / f_s
        _DFT_CACHE.clear()
        _DFT_CACHE[key] = np.exp(2j * math.pi * np.outer(t, f))
    return _DFT_CACHE[key]


@dataclass
class PointData:
    Q: np.ndarray        # [K][M][N_t] complex128, centre sample = t_ref
    U: np.ndarray        # [K][M][M] complex128 Hermitian
    V: np.ndarray        # [K][M][M] complex128 symmetric
    rho: float           # sqrt(sum_k 4 df sum_f |d_k|^2 / S) of the noise-free data after scaling
    scale: float         # the scalar applied to every h_lm (reading A7)


@dataclass
class Spectra:
    h: np.ndarray        # [K][M][N_FREQ] complex128: the modes h_lm(f) per detector (reading B1), already scaled (A7)
    d: np.ndarray        # [K][N_FREQ] complex128: the data of every detector
    w: np.ndarray        # [K][N_FREQ] float64: inner-product weights 4 df / S(f) (the one-sided recipe of configs[0])
    f: np.ndarray        # [N_FREQ] Hz
    rho: float
    scale: float


def make_spectra(cfg: Config, point: int, coeff_true: np.ndarray, shift_true: np.ndarray, c_true: float,
                 noise: bool = True) -> Spectra:
    """Frequency series of one intrinsic point by the literal recipe of BASELINE.json configs[0] (the inputs of
    Eq. (D4a-c)): modes, data, inner-product weights.

    coeff_true[k][lm] : complex, the coefficient of h_lm in detector k's data (the caller passes
                        F_k * Y_lm at the true point; this module does not know what it means).
    shift_true[k]     : integer delay of detector k in samples; the data carry the phase ramp
                        exp(-2 pi i f shift/f_s) so that Q_k peaks shift_true[k] samples after t_ref.
    c_true            : D_ref / D_true.
    """
    K, M = cfg.n_det, cfg.n_modes
    coeff_true = np.asarray(coeff_true, dtype=np.complex128).reshape(K, M)
    shift_true = np.asarray(shift_true, dtype=np.int64).reshape(K)
    f, df = freq_grid()
    S = psd(cfg.psd, f)
    rng = point_rng(cfg, point)

    # h_lm(f): amplitude f^(-7/6) (1 + 0.3 N(0,1)), phase U[0, 2pi), drawn per detector and mode.
    amp = f ** (-7.0 / 6.0) * (1.0 + 0.3 * rng.standard_normal((K, M, N_FREQ)))
    pha = rng.uniform(0.0, 2.0 * math.pi, (K, M, N_FREQ))
    h = amp * np.exp(1j * pha)
    if cfg.mode_amp_decay:
        decay = np.array([0.5 ** (l - 2) for (l, _m) in cfg.modes])
        h *= decay[None, :, None]

    # noise-free data, then one scalar on every h_lm so that its optimal SNR is cfg.rho (A7)
    ramp = np.exp(-2j * math.pi * f[None, :] * (shift_true[:, None] / cfg.f_s))
    d0 = c_true * np.einsum("km,kmf->kf", coeff_true, h) * ramp
    rho0 = math.sqrt(float(np.sum(4.0 * df * np.abs(d0) ** 2 / S)))
    scale = cfg.rho / rho0 if rho0 > 0 else 1.0
    h *= scale
    d = d0 * scale
    if noise:
        sig = np.sqrt(S / (4.0 * df))                      # reading A8: Re and Im each N(0, S/(4 df))
        d = d + sig * (rng.standard_normal((K, N_FREQ)) + 1j * rng.standard_normal((K, N_FREQ)))
    w = np.broadcast_to(4.0 * df / S, (K, N_FREQ)).copy()
    return Spectra(np.ascontiguousarray(h), np.ascontiguousarray(d), w, f, cfg.rho if rho0 > 0 else 0.0, scale)


def make_point(cfg: Config, point: int, coeff_true: np.ndarray, shift_true: np.ndarray,
               c_true: float, noise: bool = True) -> PointData:
    """Q, U, V of one intrinsic point from make_spectra's series, on the host (numpy): the generator of the parity tests.
    (bench.py builds the same arrays on the device with rift_ile_precompute.)"""
    K, M, n_t = cfg.n_det, cfg.n_modes, cfg.n_t
    sp = make_spectra(cfg, point, coeff_true, shift_true, c_true, noise)
    h, d, f = sp.h, sp.d, sp.f
    df = (F_HIGH_HZ - F_LOW_HZ) / N_FREQ
    S = psd(cfg.psd, f)

    # U = 4 df sum h* h'/S ; V = 4 df sum h h'/S   (configs[0])
    hw = h / S
    U = 4.0 * df * np.einsum("kaf,kbf->kab", np.conj(h), hw)
    V = 4.0 * df * np.einsum("kaf,kbf->kab", h, hw)
    U = 0.5 * (U + np.conj(np.swapaxes(U, 1, 2)))          # exactly Hermitian / symmetric
    V = 0.5 * (V + np.swapaxes(V, 1, 2))

    # Q(t_j) = 4 df sum_n exp(2 pi i f_n t_j) h*(f_n) d(f_n) / S(f_n), t_j = (j - (N_t-1)/2)/f_s (A9)
    E = _dft_matrix(n_t, cfg.f_s)                          # [N_t][N_FREQ]
    W = (np.conj(h) * (d / S)[:, None, :]).reshape(K * M, N_FREQ)
    Q = (4.0 * df) * (W @ E.T)                             # [K*M][N_t]
    return PointData(np.ascontiguousarray(Q.reshape(K, M, n_t)), np.ascontiguousarray(U),
                     np.ascontiguousarray(V), sp.rho, sp.scale)


# ----------------------------------------------------------------------------------------------
# Extrinsic samples and importance weights
# ----------------------------------------------------------------------------------------------
def _truncnorm(rng: np.random.Generator, mu: float, sigma: float, lo: float, hi: float, n: int):
    """Inverse-CDF draws from N(mu, sigma^2) truncated to [lo, hi]; returns (x, ln pdf(x))."""
    from scipy.special import ndtr, ndtri
    a, b = ndtr((lo - mu) / sigma), ndtr((hi - mu) / sigma)
    u = rng.uniform(0.0, 1.0, n)
    x = mu + sigma * ndtri(a + u * (b - a))
    x = np.clip(x, lo, hi)
    lnp = -0.5 * ((x - mu) / sigma) ** 2 - math.log(sigma * math.sqrt(2.0 * math.pi)) - math.log(b - a)
    return x, lnp


def draw_samples(cfg: Config, point: int, n: Optional[int] = None,
                 theta_true: Optional[np.ndarray] = None) -> Tuple[np.ndarray, np.ndarray]:
    """Extrinsic samples of one intrinsic point: (params[6][n] float64, ln_weight[n] float64).

    "prior": prior draws, ln w = 0.  "gauss_sky" (C2, reading A12): RA, dec from truncated normals
    (sigma = 0.3 rad) about the true point, ln w = ln[cos(dec)/(4 pi)] - ln p_s(RA) - ln p_s(dec);
    the other four dimensions are prior draws.
    """
    n = cfg.n_samples if n is None else int(n)
    rng = point_rng(cfg, point, stream=500)
    params = prior_draw(rng, n)
    ln_w = np.zeros(n, dtype=np.float64)
    if cfg.proposal == "gauss_sky":
        if theta_true is None:
            theta_true = true_point(cfg, point)
        ra0, dec0 = float(theta_true[0]), float(theta_true[1])
        ra, lnp_ra = _truncnorm(rng, ra0, 0.3, ra0 - math.pi, ra0 + math.pi, n)
        dec, lnp_dec = _truncnorm(rng, dec0, 0.3, -0.5 * math.pi, 0.5 * math.pi, n)
        params[0] = np.mod(ra, 2.0 * math.pi)
        params[1] = dec
        ln_w = np.log(np.maximum(np.cos(dec), 1e-300) / (4.0 * math.pi)) - lnp_ra - lnp_dec
    elif cfg.proposal != "prior":
        raise ValueError(cfg.proposal)
    return np.ascontiguousarray(params), ln_w


HIST_LO = np.array([0.0, -0.5 * math.pi, 0.0, 0.0, 0.0, D_MIN_MPC])
HIST_HI = np.array([2.0 * math.pi, 0.5 * math.pi, math.pi, math.pi, 2.0 * math.pi, D_MAX_MPC])


# ----------------------------------------------------------------------------------------------
# Whole-config assembly
# ----------------------------------------------------------------------------------------------
GeometryFn = Callable[[np.ndarray], Tuple[np.ndarray, np.ndarray, np.ndarray]]
"""geometry_fn(theta[6]) -> (F[K] complex, Y[M] complex, shift[K] int) at one extrinsic point;
supplied by the caller (oracle in tests, the CUDA geometry kernel in bench.py)."""


@dataclass
class ConfigInputs:
    cfg: Config
    det_location: np.ndarray
    det_response: np.ndarray
    mode_l: np.ndarray
    mode_m: np.ndarray
    Q: np.ndarray            # [P][K][M][N_t] complex128
    U: np.ndarray            # [P][K][M][M]
    V: np.ndarray
    theta_true: np.ndarray   # [P][6]
    points: List[PointData] = field(default_factory=list)


def build_inputs(cfg: Config, geometry_fn: GeometryFn, n_points: Optional[int] = None,
                 noise: bool = True, point_ids: Optional[Sequence[int]] = None) -> ConfigInputs:
    """point_ids: the seeds' point indices (default 0..P-1); a multi-GPU run gives every rank its own ids."""
    P = cfg.n_points if n_points is None else int(n_points)
    if point_ids is None:
        point_ids = list(range(P))
    P = len(point_ids)
    loc, resp = detector_arrays(cfg)
    ml, mm = mode_arrays(cfg)
    K, M, n_t = cfg.n_det, cfg.n_modes, cfg.n_t
    Q = np.empty((P, K, M, n_t), dtype=np.complex128)
    U = np.empty((P, K, M, M), dtype=np.complex128)
    V = np.empty((P, K, M, M), dtype=np.complex128)
    th = np.empty((P, 6), dtype=np.float64)
    pts = []
    for p, pid in enumerate(point_ids):
        th[p] = true_point(cfg, pid)
        F, Y, shift = geometry_fn(th[p])
        coeff = np.asarray(F).reshape(K, 1) * np.asarray(Y).reshape(1, M)
        pd = make_point(cfg, pid, coeff, shift, D_REF_MPC / th[p, 5], noise=noise)
        Q[p], U[p], V[p] = pd.Q, pd.U, pd.V
        pts.append(PointData(None, None, None, pd.rho, pd.scale))
    return ConfigInputs(cfg, loc, resp, ml, mm, Q, U, V, th, pts)
