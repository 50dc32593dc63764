"""gmm_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle of the Gaussian-mixture adaptive sampler of SURVEY.md section 8(f) NEXT-4: PAPER.md section IV.C.1 (:315-334, Eq. (19)-
(21)) and Appendix A (:562-625, Eq. (A1)-(A13)), plain numpy / scipy in fp64, one group of n_dim = 1 or 2 correlated dimensions
("pairwise-correlated") over a rectangular domain [lo, hi).  Shares no code with paper_2210_07912_b200 and never imports it.

Readings:
  G1  Eq. (A2)-(A3) as printed cancel the sample weight w_n (it multiplies numerator and denominator of p_nk), which would make
      the M-step ignore the weights.  We take the weighted EM the text describes ("for each sample x_n and its corresponding
      sample weight w_n"): r_nk = N(x_n|mu_k,Sigma_k) pi_k / sum_j N(x_n|mu_j,Sigma_j) pi_j, p_nk = w_n r_nk with the weights
      normalised to sum_n w_n = 1, so that (A6) reads pi_k = sum_n p_nk; ln L = sum_n w_n ln sum_k N_k pi_k (Eq. (A1) with the
      weights as exponents).  Weights arrive as logarithms (ln omega_i of the reduce): w_n = exp(ln_w_n - max) / sum.
  G2  Sigma_k of Eq. (A5) is centred on the NEW mean of Eq. (A4); `reg` (default 0) is added to its diagonal.
  G3  Online update: the new model is trained on the new batch starting from the old model's parameters; Eq. (A11) prints pi_k
      for pi_i.  The matching of Eq. (A8) is a search over all permutations (n_comp <= 8).
  G4  Eq. (A12) prints lambda^(1/2) phi x; with phi holding the eigenvectors as columns the map with covariance Sigma is
      x' = phi lambda^(1/2) x + mu =: A x + mu.  Eigenvalues ascending, each eigenvector signed so that its component of largest
      magnitude is positive (the first on a tie): any orthogonal choice gives the same distribution, one choice gives the same
      draws.  Eq. (A13): r = A^-1, the proposal box is the bounding box of r (corner - mu) over the corners of the domain.
  G5  Truncated components ("truncated normal distributions p_{n,t} in place of normal distributions p_n in our mixture"):
      p_s(x) = sum_k pi_k N(x|mu_k,Sigma_k) / Z_k on the domain, Z_k the component's mass inside it; a draw picks its
      component once and repeats the box proposal until it lands in the domain (at most max_tries = 64 times; a sample that
      never does is set to the domain-clipped mean and counted).  The univariate truncated normals are inverse-CDF draws.
  G6  Random numbers: the counter-based hash of oracle/ac_oracle.py (splitmix64 finaliser of seed + (c + 1) * golden ratio)
      with counter c = (sample * max_tries + try) * 4 + j, j = 0 for the component of try 0, j = 1 + dimension for z_j.
  G7  Tempering (not in the paper; a safeguard of the adaptive loop): the fit may be run on weights w_n^temper, temper the
      largest value in [0, 1] found by 20 bisection steps from [0, 1] whose effective sample size (sum w^t)^2 / sum w^(2t)
      reaches ess_min (1 if the plain weights already do).
Pins: tests/test_gmm_oracle_pins.py (P32-P40).
"""
from __future__ import annotations

import itertools
import math

import numpy as np
from scipy import integrate, special

from .ac_oracle import hash_u01

__all__ = ["tempered_ess", "temper_for_ess", "normalise_ln_weights", "ln_normal", "e_step", "m_step", "fit", "match_components", "merge", "transform", "z_box",
           "box_mass", "draw", "ln_density", "MAX_TRIES"]

MAX_TRIES = 64


def tempered_ess(ln_w, beta: float) -> float:
    ln_w = np.asarray(ln_w, dtype=np.float64)
    v = ln_w[np.isfinite(ln_w)]
    w = np.exp(beta * (v - np.max(v)))
    return float(np.sum(w) ** 2 / np.sum(w * w))


def temper_for_ess(ln_w, ess_min: float) -> float:
    """G7."""
    if ess_min <= 0 or tempered_ess(ln_w, 1.0) >= ess_min:
        return 1.0
    lo, hi = 0.0, 1.0
    for _ in range(20):
        mid = 0.5 * (lo + hi)
        if tempered_ess(ln_w, mid) >= ess_min:
            lo = mid
        else:
            hi = mid
    return lo


def normalise_ln_weights(ln_w) -> np.ndarray:
    ln_w = np.asarray(ln_w, dtype=np.float64)
    w = np.exp(ln_w - np.max(ln_w))
    return w / np.sum(w)


def ln_normal(x, mu, cov) -> np.ndarray:
    """ln N(x | mu, cov) for x [n][d]."""
    x = np.asarray(x, dtype=np.float64)
    d = x.shape[1]
    cov = np.asarray(cov, dtype=np.float64).reshape(d, d)
    r = x - np.asarray(mu, dtype=np.float64)[None, :]
    sol = np.linalg.solve(cov, r.T).T
    return -0.5 * np.sum(r * sol, axis=1) - 0.5 * math.log(np.linalg.det(cov)) - 0.5 * d * math.log(2.0 * math.pi)


def e_step(x, w, mu, cov, pi):
    """Eq. (A2)-(A3) under G1: (r [n][K], ln L)."""
    K = len(pi)
    with np.errstate(divide="ignore"):
        lp = np.stack([ln_normal(x, mu[k], cov[k]) + math.log(pi[k]) if pi[k] > 0 else np.full(len(x), -np.inf)
                       for k in range(K)], axis=1)
    m = np.max(lp, axis=1, keepdims=True)
    lse = m[:, 0] + np.log(np.sum(np.exp(lp - m), axis=1))
    r = np.exp(lp - lse[:, None])
    return r, float(np.sum(w * lse))


def m_step(x, w, r, reg: float = 0.0):
    """Eq. (A4)-(A6) with p_nk = w_n r_nk, sum_n w_n = 1."""
    x = np.asarray(x, dtype=np.float64)
    n, d = x.shape
    K = r.shape[1]
    p = w[:, None] * r
    s0 = np.sum(p, axis=0)
    mu = np.zeros((K, d))
    cov = np.zeros((K, d, d))
    for k in range(K):
        mu[k] = np.sum(p[:, k, None] * x, axis=0) / s0[k]
        c = x - mu[k][None, :]
        cov[k] = (p[:, k, None, None] * c[:, :, None] * c[:, None, :]).sum(axis=0) / s0[k] + reg * np.eye(d)
    return mu, cov, s0 / np.sum(w)


def fit(x, ln_w, mu0, cov0, pi0, n_iter: int, tol: float = 0.0, reg: float = 0.0):
    """EM from (mu0, cov0, pi0): E-step, M-step, ... until |ln L - ln L_prev| < tol or n_iter M-steps are done.
    Returns (mu, cov, pi, iterations done, ln L of the last E-step)."""
    x = np.asarray(x, dtype=np.float64)
    w = normalise_ln_weights(ln_w)
    mu, cov, pi = np.array(mu0, dtype=np.float64), np.array(cov0, dtype=np.float64), np.array(pi0, dtype=np.float64)
    prev = None
    it = 0
    ll = -np.inf
    while it < n_iter:
        r, ll = e_step(x, w, mu, cov, pi)
        if prev is not None and abs(ll - prev) < tol:
            break
        mu, cov, pi = m_step(x, w, r, reg)
        prev = ll
        it += 1
    return mu, cov, pi, it, ll


def _mahalanobis(a, b, cov_inv) -> float:
    d = np.asarray(a) - np.asarray(b)
    return math.sqrt(max(0.0, float(d @ cov_inv @ d)))


def match_components(mu_old, cov_old, mu_new, cov_new):
    """Eq. (A8): perm[i] = the old component j matched to new component i, minimising the summed symmetric Mahalanobis
    distance over all permutations (the first minimum in lexicographic order)."""
    K = len(mu_old)
    inv_old = [np.linalg.inv(np.asarray(c)) for c in cov_old]
    inv_new = [np.linalg.inv(np.asarray(c)) for c in cov_new]
    cost = np.array([[_mahalanobis(mu_old[j], mu_new[i], inv_new[i]) + _mahalanobis(mu_new[i], mu_old[j], inv_old[j])
                      for j in range(K)] for i in range(K)])
    best, best_perm = None, None
    for perm in itertools.permutations(range(K)):
        c = sum(cost[i, perm[i]] for i in range(K))
        if best is None or c < best:
            best, best_perm = c, perm
    return list(best_perm)


def merge(mu_old, cov_old, pi_old, n_old: float, mu_new, cov_new, pi_new, n_new: float):
    """Eq. (A8)-(A11) under G3; the result is indexed like the old model."""
    K = len(pi_old)
    perm = match_components(mu_old, cov_old, mu_new, cov_new)
    mu = np.zeros_like(np.asarray(mu_old, dtype=np.float64))
    cov = np.zeros_like(np.asarray(cov_old, dtype=np.float64))
    pi = np.zeros(K)
    for i in range(K):
        j = perm[i]
        a, b = n_old * pi_old[j], n_new * pi_new[i]
        mj, mi = np.asarray(mu_old[j], dtype=np.float64), np.asarray(mu_new[i], dtype=np.float64)
        m = (a * mj + b * mi) / (a + b)
        cov[j] = ((a * np.asarray(cov_old[j]) + b * np.asarray(cov_new[i])) / (a + b)
                  + (a * np.outer(mj, mj) + b * np.outer(mi, mi)) / (a + b) - np.outer(m, m))
        mu[j] = m
        pi[j] = (a + b) / (n_old + n_new)
    return mu, cov, pi


def transform(cov) -> np.ndarray:
    """A = phi lambda^(1/2) of Eq. (A12) under G4."""
    cov = np.atleast_2d(np.asarray(cov, dtype=np.float64))
    lam, phi = np.linalg.eigh(cov)
    for j in range(phi.shape[1]):
        i = int(np.argmax(np.abs(phi[:, j]) > np.max(np.abs(phi[:, j])) * (1 - 1e-12)))
        if phi[i, j] < 0:
            phi[:, j] = -phi[:, j]
    return phi * np.sqrt(lam)[None, :]


def z_box(mu, A, lo, hi):
    """Eq. (A13): bounding box of A^-1 (corner - mu) over the corners of the domain."""
    d = len(mu)
    r = np.linalg.inv(A)
    corners = np.array([[(hi if (c >> j) & 1 else lo)[j] for j in range(d)] for c in range(1 << d)], dtype=np.float64)
    t = (corners - np.asarray(mu)[None, :]) @ r.T
    return t.min(axis=0), t.max(axis=0)


def _Phi(t):
    return special.ndtr(t)


def box_mass(mu, cov, lo, hi) -> float:
    """Z = integral of N(x | mu, cov) over [lo, hi]: the definition, by scipy's adaptive quadrature over x_1 of the exact
    conditional integral over x_2 (n_dim = 2), or the difference of two normal CDFs (n_dim = 1)."""
    mu, lo, hi = (np.asarray(v, dtype=np.float64) for v in (mu, lo, hi))
    cov = np.atleast_2d(np.asarray(cov, dtype=np.float64))
    if len(mu) == 1:
        s = math.sqrt(cov[0, 0])
        return float(_Phi((hi[0] - mu[0]) / s) - _Phi((lo[0] - mu[0]) / s))
    s1 = math.sqrt(cov[0, 0])
    slope = cov[0, 1] / cov[0, 0]
    sc = math.sqrt(cov[1, 1] - cov[0, 1] ** 2 / cov[0, 0])

    def f(x1):
        m = mu[1] + slope * (x1 - mu[0])
        return math.exp(-0.5 * ((x1 - mu[0]) / s1) ** 2) / (s1 * math.sqrt(2 * math.pi)) * (
            _Phi((hi[1] - m) / sc) - _Phi((lo[1] - m) / sc))
    a, b = max(lo[0], mu[0] - 12 * s1), min(hi[0], mu[0] + 12 * s1)
    if b <= a:
        return 0.0
    brk = [p for p in (mu[0] + (lo[1] - mu[1]) / slope, mu[0] + (hi[1] - mu[1]) / slope) if a < p < b] if slope != 0 else []
    val, _err = integrate.quad(f, a, b, points=brk or None, epsabs=1e-15, epsrel=1e-13, limit=400)
    return float(val)


def draw(n: int, seed: int, offset: int, mu, cov, pi, lo, hi):
    """(x [n][d], n_failed) under G4-G6 for samples offset .. offset + n - 1."""
    mu = np.asarray(mu, dtype=np.float64)
    K, d = mu.shape
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    A = [transform(np.asarray(cov[k]).reshape(d, d)) for k in range(K)]
    zb = [z_box(mu[k], A[k], lo, hi) for k in range(K)]
    cum = np.cumsum(np.asarray(pi, dtype=np.float64))
    x = np.empty((n, d))
    failed = 0
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    uc = hash_u01(seed, idx * np.uint64(MAX_TRIES * 4))
    for i in range(n):
        k = int(np.searchsorted(cum, uc[i], side="right"))
        k = min(k, K - 1)
        pa, pb = _Phi(zb[k][0]), _Phi(zb[k][1])
        done = False
        for t in range(MAX_TRIES):
            c = (int(idx[i]) * MAX_TRIES + t) * 4
            u = hash_u01(seed, np.array([c + 1 + j for j in range(d)], dtype=np.uint64))
            z = special.ndtri(pa + u * (pb - pa))
            xi = mu[k] + A[k] @ z
            if np.all(xi >= lo) and np.all(xi < hi):
                x[i] = xi
                done = True
                break
        if not done:
            x[i] = np.clip(mu[k], lo, np.nextafter(hi, lo))
            failed += 1
    return x, failed


def ln_density(x, mu, cov, pi, lo, hi) -> np.ndarray:
    """ln p_s(x) of G5 (-inf outside the domain)."""
    x = np.asarray(x, dtype=np.float64)
    mu = np.asarray(mu, dtype=np.float64)
    K, d = mu.shape
    lo, hi = np.asarray(lo, dtype=np.float64), np.asarray(hi, dtype=np.float64)
    with np.errstate(divide="ignore"):
        lp = np.stack([ln_normal(x, mu[k], np.asarray(cov[k]).reshape(d, d)) + math.log(pi[k])
                       - math.log(box_mass(mu[k], np.asarray(cov[k]).reshape(d, d), lo, hi)) if pi[k] > 0
                       else np.full(len(x), -np.inf) for k in range(K)], axis=1)
    m = np.max(lp, axis=1, keepdims=True)
    out = m[:, 0] + np.log(np.sum(np.exp(lp - m), axis=1))
    inside = np.all((x >= lo[None, :]) & (x < hi[None, :]), axis=1)
    return np.where(inside, out, -np.inf)
