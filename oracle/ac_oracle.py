"""Oracle of the adaptive-cartesian (AC) sampler -- TEST INFRASTRUCTURE, not the product.

Plain numpy, fp64, written from PAPER.md section IV.C.2 (:336-358): a separable sampling prior p_s(theta) = prod_k p_{s,k}
whose adaptive dimensions are histograms with a fixed number of bins (Eq. (22), :348; n_bins = 100, :350), refreshed from the
recent history of weighted samples; the Monte Carlo estimate is Eq. (3), :55.  Readings:
  C1  the histogram is built from the integrand-weighted samples (SURVEY.md reading A13), optionally tempered, and mixed with a
      uniform floor so that the support never collapses:  m' = (1 - floor) h^temper / sum(h^temper) + floor / n_bins;
  C2  draws are inverse-CDF: bin b = the last bin with cdf[b] <= u, position uniform inside the bin; the random numbers are a
      counter-based hash (splitmix64 finaliser) of (seed, sample index, dimension), so that any implementation reproduces them.
Shares no code with paper_2210_07912_b200 and never imports it.
"""
from __future__ import annotations

import math

import numpy as np

__all__ = ["hash_u01", "uniform_masses", "cdf_of", "draw", "update", "ln_prior_ile"]

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def hash_u01(seed: int, index: np.ndarray) -> np.ndarray:
    """u in [0, 1) with 53 random bits from splitmix64(seed + (index + 1) * 0x9E3779B97F4A7C15)."""
    with np.errstate(over="ignore"):
        z = (np.uint64(seed) + (np.asarray(index, dtype=np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform_masses(n_dim: int, n_bins: int) -> np.ndarray:
    return np.full((n_dim, n_bins), 1.0 / n_bins)


def cdf_of(masses: np.ndarray) -> np.ndarray:
    """cdf[d][b] = sum of the masses of the bins before b, accumulated left to right (cdf[d][0] = 0)."""
    n_dim, n_bins = masses.shape
    cdf = np.zeros((n_dim, n_bins))
    for d in range(n_dim):
        acc = 0.0
        for b in range(n_bins):
            cdf[d, b] = acc
            acc = acc + masses[d, b]
    return cdf


def draw(masses: np.ndarray, lo, hi, n: int, seed: int, offset: int = 0):
    """n draws from the product of histograms.  Returns (x [n_dim][n], ln p_s [n], bins [n_dim][n])."""
    masses = np.asarray(masses, dtype=np.float64)
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    n_dim, n_bins = masses.shape
    cdf = cdf_of(masses)
    i = np.arange(n, dtype=np.uint64) + np.uint64(offset)
    x = np.empty((n_dim, n))
    bins = np.empty((n_dim, n), dtype=np.int32)
    ln_ps = np.zeros(n)
    for d in range(n_dim):
        u = hash_u01(seed, i * np.uint64(n_dim) + np.uint64(d))
        b = np.searchsorted(cdf[d], u, side="right") - 1          # last bin with cdf[b] <= u
        b = np.clip(b, 0, n_bins - 1)
        w = (hi[d] - lo[d]) / n_bins
        frac = (u - cdf[d, b]) / masses[d, b]
        frac = np.minimum(frac, np.nextafter(1.0, 0.0))           # rounding of the cdf must not push x out of its bin
        x[d] = (b.astype(np.float64) + frac) * w + lo[d]
        bins[d] = b
        ln_ps = ln_ps + np.log(masses[d, b] / w)
    return x, ln_ps, bins


def update(hist: np.ndarray, floor: float, temper: float = 1.0) -> np.ndarray:
    """New bin masses from normalised weighted histograms (reading C1)."""
    hist = np.asarray(hist, dtype=np.float64)
    n_dim, n_bins = hist.shape
    out = np.empty_like(hist)
    for d in range(n_dim):
        h = np.power(np.maximum(hist[d], 0.0), temper)
        s = 0.0
        for b in range(n_bins):
            s = s + h[b]
        if not (s > 0.0) or not math.isfinite(s):
            out[d] = 1.0 / n_bins
        else:
            out[d] = (1.0 - floor) * (h / s) + floor / n_bins
    return out


def ln_prior_ile(params: np.ndarray, d_min: float, d_max: float) -> np.ndarray:
    """ln p(theta) of the extrinsic priors (SURVEY.md reading A18): RA, psi, phi uniform; dec ~ cos(dec)/2; iota ~ sin(iota)/2;
    distance ~ 3 D^2 / (d_max^3 - d_min^3) on [d_min, d_max]; -inf outside the support."""
    ra, dec, psi, iota, phi, dist = (np.asarray(p, dtype=np.float64) for p in params)
    two_pi = 2.0 * math.pi
    with np.errstate(divide="ignore", invalid="ignore"):
        lp = (-math.log(two_pi) + np.log(np.cos(dec) / 2.0) - math.log(math.pi) + np.log(np.sin(iota) / 2.0)
              - math.log(two_pi) + np.log(3.0 * dist * dist / (d_max ** 3 - d_min ** 3)))
    ok = ((ra >= 0) & (ra < two_pi) & (np.abs(dec) <= math.pi / 2) & (psi >= 0) & (psi < math.pi) & (iota >= 0)
          & (iota <= math.pi) & (phi >= 0) & (phi < two_pi) & (dist >= d_min) & (dist <= d_max))
    return np.where(ok & np.isfinite(lp), lp, -np.inf)
