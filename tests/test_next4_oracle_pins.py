"""Pins of oracle/sky_oracle.py (rotated network-frame sky; rho_guess, Eq. (D7)
PAPER.md:790 with reading A14) against what the geometry and the mathematics fix -- no GPU, no product code."""
import numpy as np

from oracle import sky_oracle as so
from paper_2210_07912_b200 import synth

C_LIGHT = 299792458.0


def _sites():
    loc, _resp = synth.detector_arrays(synth.CONFIGS[1])          # H1, L1, V1
    return loc


def test_p27_pole_is_the_baseline_and_the_frame_is_a_rotation():
    loc = _sites()
    for a, b in ((0, 1), (0, 2), (2, 1)):
        R = so.network_frame(loc[a], loc[b])
        base = (loc[b] - loc[a]) / np.linalg.norm(loc[b] - loc[a])
        assert np.allclose(R.T @ R, np.eye(3), atol=1e-14) and abs(np.linalg.det(R) - 1.0) < 1e-14
        assert np.allclose(R[:, 2], base, atol=1e-15)
        # nominal north pole: beta = pi/2 points along the baseline, whatever lambda is
        for gmst in (0.0, 1.234):
            ra, dec = so.network_to_radec(np.array([0.3, 2.0]), np.array([np.pi / 2, np.pi / 2]), R, gmst)
            n = so.sky_unit_vector(ra, dec, gmst)
            assert np.allclose(n, base[None, :], atol=1e-7)          # asin near 1 loses half the digits
        # x' is perpendicular to the Earth's axis: lambda = 0, beta = 0 lies in the equatorial plane
        ra, dec = so.network_to_radec(np.array([0.0]), np.array([0.0]), R, 0.0)
        assert abs(dec[0]) < 1e-15
    # baseline along the axis: the frame is the identity
    assert np.allclose(so.network_frame([0, 0, -1.0], [0, 0, 2.0]), np.eye(3))


def test_p28_delay_difference_depends_on_nominal_declination_only(oracle):
    """tau_a - tau_b = -(r_a - r_b).n / c = |r_b - r_a| sin(beta) / c, from the oracle's own (pinned) delay of step a3: the
    posterior of a two-detector network lies along lines of constant beta, which is why the paper offers the frame."""
    loc = _sites()
    rng = np.random.default_rng(5)
    for gmst in (0.0, 2.5):
        R = so.network_frame(loc[0], loc[1])
        L = np.linalg.norm(loc[1] - loc[0])
        lam = rng.uniform(0, 2 * np.pi, 200)
        beta = np.arcsin(rng.uniform(-1, 1, 200))
        ra, dec = so.network_to_radec(lam, beta, R, gmst)
        assert np.all((ra >= 0) & (ra < 2 * np.pi)) and np.all(np.abs(dec) <= np.pi / 2)
        dt, _sh, _fr = oracle.delays(ra, dec, gmst, loc[:2], 1.0 / 4096)
        assert np.max(np.abs((dt[:, 0] - dt[:, 1]) - L * np.sin(beta) / C_LIGHT)) < 1e-15
        # same beta, other lambda: same difference
        ra2, dec2 = so.network_to_radec(lam[::-1], beta, R, gmst)
        dt2, _s, _f = oracle.delays(ra2, dec2, gmst, loc[:2], 1.0 / 4096)
        assert np.max(np.abs((dt2[:, 0] - dt2[:, 1]) - (dt[:, 0] - dt[:, 1]))) < 1e-15


def test_p29_round_trip_and_solid_angle():
    loc = _sites()
    R = so.network_frame(loc[0], loc[2])
    rng = np.random.default_rng(6)
    gmst = 0.7
    ra = rng.uniform(0, 2 * np.pi, 1000)
    dec = np.arcsin(rng.uniform(-1, 1, 1000))
    lam, beta = so.radec_to_network(ra, dec, R, gmst)
    ra2, dec2 = so.network_to_radec(lam, beta, R, gmst)
    d = np.abs(ra2 - ra)
    assert np.max(np.minimum(d, 2 * np.pi - d)) < 1e-9 and np.max(np.abs(dec2 - dec)) < 1e-9
    # angles between pairs of directions are preserved (an isometry of the sphere keeps the isotropic prior isotropic)
    n = so.sky_unit_vector(ra, dec, gmst)
    v = np.stack([np.cos(beta) * np.cos(lam), np.cos(beta) * np.sin(lam), np.sin(beta)], axis=-1)
    assert np.max(np.abs(n[:500] @ n[500:].T - v[:500] @ v[500:].T)) < 1e-12
    # a uniform (lambda, sin beta) grid maps to directions whose mean vanishes and whose second moment is I/3
    g_l, g_s = np.meshgrid((np.arange(64) + 0.5) * 2 * np.pi / 64, (np.arange(64) + 0.5) * 2 / 64 - 1, indexing="ij")
    ra_g, dec_g = so.network_to_radec(g_l.ravel(), np.arcsin(g_s.ravel()), R, gmst)
    ng = so.sky_unit_vector(ra_g, dec_g, gmst)
    assert np.max(np.abs(ng.mean(axis=0))) < 1e-12
    assert np.max(np.abs(ng.T @ ng / ng.shape[0] - np.eye(3) / 3)) < 1e-3


def _single_mode_case(rng, K, M, n_t, delta_t, amps, delays_samples):
    """Noise-free data d_k = A_k h_{k,0} delayed by an integer number of samples: Q_{k,0} peaks at |A_k| U_{k,00}."""
    n_f = 257
    f = 20.0 + np.arange(n_f) * 0.75
    h = (rng.normal(size=(K, M, n_f)) + 1j * rng.normal(size=(K, M, n_f))) * f ** (-7.0 / 6.0)
    w = 4.0 * (f[1] - f[0]) / (1.0 + (f / 200.0) ** 2)
    t = (np.arange(n_t) - (n_t - 1) / 2.0) * delta_t
    Q = np.zeros((K, M, n_t), dtype=np.complex128)
    U = np.zeros((K, M, M), dtype=np.complex128)
    for k in range(K):
        d = amps[k] * h[k, 0] * np.exp(-2j * np.pi * f * delays_samples[k] * delta_t)
        for a in range(M):
            Q[k, a] = np.array([np.sum(w * np.conj(h[k, a]) * d * np.exp(2j * np.pi * f * tj)) for tj in t])
            for b in range(M):
                U[k, a, b] = np.sum(w * np.conj(h[k, a]) * h[k, b])
    return Q, U


def test_p30_noise_free_single_mode_signal_gives_rho_over_2p3():
    rng = np.random.default_rng(7)
    amps = np.array([0.7 - 0.2j, 1.3 + 0.4j])
    Q, U = _single_mode_case(rng, 2, 1, 65, 1.0 / 512, amps, [5, -9])
    rho2 = sum(abs(amps[k]) ** 2 * U[k, 0, 0].real for k in range(2))          # optimal SNR^2 of the network
    assert abs(so.rho_guess(Q, U) - np.sqrt(rho2) / 2.3) < 1e-12 * np.sqrt(rho2)
    # the peak sits at the injected delay (Cauchy-Schwarz: nowhere else is |Q| as large)
    assert np.argmax(np.abs(Q[0, 0])) == 32 + 5 and np.argmax(np.abs(Q[1, 0])) == 32 - 9


def test_p31_brute_force_and_zero_diagonal():
    rng = np.random.default_rng(8)
    Q = rng.normal(size=(3, 4, 50)) + 1j * rng.normal(size=(3, 4, 50))
    U = rng.normal(size=(3, 4, 4)) + 1j * rng.normal(size=(3, 4, 4))
    U[1, 2, 2] = 0.0                                               # a mode absent from one detector: its term is left out
    tot = 0.0
    for k in range(3):
        for a in range(4):
            if U[k, a, a] != 0:
                tot += max(abs(q) ** 2 for q in Q[k, a]) / abs(U[k, a, a])
    assert abs(so.rho_guess(Q, U) - np.sqrt(tot) / 2.3) < 1e-13
    # scaling: data twice as loud doubles rho_guess; a louder template leaves it unchanged (Q ~ h, U ~ h^2)
    assert abs(so.rho_guess(2 * Q, U) - 2 * so.rho_guess(Q, U)) < 1e-12
    assert abs(so.rho_guess(3 * Q, 9 * U) - so.rho_guess(Q, U)) < 1e-12
