"""precompute_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Oracle of SURVEY.md section 8(f) NEXT-3: the mode / data inner products held fixed per intrinsic point, Eq. (D4a-c)
(PAPER.md:769-776), as plain numpy in complex128.  With the inner product written as a weighted sum over a caller-supplied
list of frequencies (reading E1 of DESIGN.md section 13: w_k(f_n) = 4 df / S_k(f_n) over f_n > 0 is the one-sided recipe of
BASELINE.json configs[0]; w = 2 df / S over +-f the two-sided Eq. (D4a); either is the caller's choice of f and w):

    Q[k, a, j] = sum_n w[k, n] exp(2 pi i f[n] t_j) conj(h[k, a, n]) d[k, n],     t_j = (j - (n_t - 1)/2) delta_t
    U[k, a, b] = sum_n w[k, n] conj(h[k, a, n]) h[k, b, n]
    V[k, a, b] = sum_n w[k, n] h[k, a, n] h[k, b, n]

h: [K][M][N_f] (per detector and mode, reading B1), d: [K][N_f], w: [K][N_f], f: [N_f].  No symmetrisation, no FFT, no
blocking: the definition.  Pins: tests/test_precompute_oracle_pins.py (P23 brute force, P24 numpy.fft on an FFT grid, P25 a
delayed copy peaks at its delay with height U_aa, P26 Hermitian / symmetric / positive).
"""
from __future__ import annotations

import numpy as np


def window_times(n_t: int, delta_t: float) -> np.ndarray:
    return (np.arange(n_t, dtype=np.float64) - (n_t - 1) / 2.0) * delta_t


def quv(h, d, w, f, n_t: int, delta_t: float):
    """(Q[K][M][n_t], U[K][M][M], V[K][M][M]) of one intrinsic point."""
    h = np.asarray(h, dtype=np.complex128)
    d = np.asarray(d, dtype=np.complex128)
    w = np.asarray(w, dtype=np.float64)
    f = np.asarray(f, dtype=np.float64)
    E = np.exp(2j * np.pi * np.outer(window_times(n_t, delta_t), f))            # [n_t][N_f]
    X = w[:, None, :] * np.conj(h) * d[:, None, :]                              # [K][M][N_f]
    Q = np.einsum("jn,kan->kaj", E, X)
    U = np.einsum("kn,kan,kbn->kab", w, np.conj(h), h)
    V = np.einsum("kn,kan,kbn->kab", w, h, h)
    return Q, U, V
