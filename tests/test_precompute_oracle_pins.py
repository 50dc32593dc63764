"""Pins of oracle/precompute_oracle.py (Eq. (D4a-c))."""
import math

import numpy as np

from oracle import precompute_oracle as po
from paper_2210_07912_b200 import synth


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def test_p23_brute_force_on_a_tiny_input():
    rng = np.random.default_rng(1)
    K, M, NF, n_t, dt = 2, 3, 5, 7, 0.01
    h, d, w, f = _rand(rng, K, M, NF), _rand(rng, K, NF), rng.uniform(0.5, 2.0, (K, NF)), rng.uniform(20.0, 90.0, NF)
    Q, U, V = po.quv(h, d, w, f, n_t, dt)
    for k in range(K):
        for a in range(M):
            for j in range(n_t):
                t = (j - (n_t - 1) / 2.0) * dt
                acc = 0j
                for n in range(NF):
                    acc += w[k, n] * complex(math.cos(2 * math.pi * f[n] * t), math.sin(2 * math.pi * f[n] * t)) \
                        * h[k, a, n].conjugate() * d[k, n]
                assert abs(Q[k, a, j] - acc) < 1e-13 * max(1.0, abs(acc))
            for b in range(M):
                u = sum(w[k, n] * h[k, a, n].conjugate() * h[k, b, n] for n in range(NF))
                v = sum(w[k, n] * h[k, a, n] * h[k, b, n] for n in range(NF))
                assert abs(U[k, a, b] - u) < 1e-13 and abs(V[k, a, b] - v) < 1e-13


def test_p24_library_fft_on_an_fft_grid():
    """f_n = n df, delta_t = 1/(N df): Q(t_j) = N ifft(w h* d)[j - (n_t-1)/2 mod N]."""
    rng = np.random.default_rng(2)
    K, M, N, df = 1, 2, 256, 0.25
    n_t, dt = 31, 1.0 / (N * df)
    h, d, w = _rand(rng, K, M, N), _rand(rng, K, N), rng.uniform(0.5, 2.0, (K, N))
    f = df * np.arange(N)
    Q, _U, _V = po.quv(h, d, w, f, n_t, dt)
    for a in range(M):
        ref = N * np.fft.ifft(w[0] * np.conj(h[0, a]) * d[0])
        idx = (np.arange(n_t) - (n_t - 1) // 2) % N
        assert np.max(np.abs(Q[0, a] - ref[idx])) < 1e-11 * np.max(np.abs(ref))


def test_p25_delayed_copy_peaks_at_its_delay():
    rng = np.random.default_rng(3)
    f, df = synth.freq_grid()
    K, M, n_t, dt = 1, 2, 411, 1.0 / 4096.0
    h = _rand(rng, K, M, f.size) * f ** (-7.0 / 6.0)
    w = np.broadcast_to(4.0 * df / synth.psd("analytic", f), (K, f.size)).copy()
    j0 = 37                                                   # samples after the window centre
    d = h[:, 0, :] * np.exp(-2j * np.pi * f * (j0 * dt))
    Q, U, _V = po.quv(h, d, w, f, n_t, dt)
    peak = (n_t - 1) // 2 + j0
    assert abs(Q[0, 0, peak] - U[0, 0, 0]) < 1e-12 * abs(U[0, 0, 0]) and abs(U[0, 0, 0].imag) < 1e-12 * U[0, 0, 0].real
    assert np.argmax(np.abs(Q[0, 0])) == peak
    assert np.all(np.abs(Q[0, 0]) <= U[0, 0, 0].real * (1 + 1e-12))   # Cauchy-Schwarz: unit-modulus phases
    assert abs(Q[0, 1, peak] - U[0, 1, 0]) < 1e-12 * abs(U[0, 0, 0])  # <h_1 | h_0> at the aligned time


def test_p26_symmetries_and_the_recipe_of_synth():
    rng = np.random.default_rng(4)
    K, M, NF = 2, 4, 64
    h, d, w, f = _rand(rng, K, M, NF), _rand(rng, K, NF), rng.uniform(0.5, 2.0, (K, NF)), rng.uniform(20.0, 500.0, NF)
    _Q, U, V = po.quv(h, d, w, f, 9, 1e-3)
    assert np.max(np.abs(U - np.conj(np.swapaxes(U, 1, 2)))) < 1e-12
    assert np.max(np.abs(V - np.swapaxes(V, 1, 2))) < 1e-12
    assert np.all(np.linalg.eigvalsh(U[0]) > 0)
    # the generator of the timing configs (synth.make_point) builds exactly these sums (and symmetrises U, V)
    cfg = synth.with_overrides(synth.CONFIGS[1], n_points=1)
    coeff = _rand(rng, cfg.n_det, cfg.n_modes)
    sp = synth.make_spectra(cfg, 0, coeff, np.array([3, -5, 11]), 0.8)
    pd = synth.make_point(cfg, 0, coeff, np.array([3, -5, 11]), 0.8)
    Q2, U2, V2 = po.quv(sp.h, sp.d, sp.w, sp.f, cfg.n_t, cfg.delta_t)
    assert np.max(np.abs(Q2 - pd.Q)) < 1e-10 * np.max(np.abs(pd.Q))
    assert np.max(np.abs(U2 - pd.U)) < 1e-11 * np.max(np.abs(pd.U)) and np.max(np.abs(V2 - pd.V)) < 1e-11 * np.max(np.abs(pd.V))
