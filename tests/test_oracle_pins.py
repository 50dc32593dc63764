"""Pins P1-P12: the oracle against what the paper and the mathematics fix.

Nothing here retypes an oracle formula: harmonics are checked against closed forms, orthonormality
and sum rules; the antenna pattern against sky averages and rotation covariance; delays against
site baselines; the factored likelihood against the direct definition Eq. (D1) evaluated from
frequency series (numpy); the time marginal, layout and reduce steps against invariants, App. B's
closed forms and brute force; the whole integral against tensor-product quadrature.
"""
import math
import os

import numpy as np
import pytest

from paper_2210_07912_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
TWO_PI = 2.0 * math.pi


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


# ------------------------------------------------------------------------------------------ P1
def test_p1_l2_closed_forms(oracle):
    rng = np.random.default_rng(1)
    for row in _rows("swsh_l2.txt"):
        m, num, den, p1, ps, sign = (int(x) for x in row)
        for _ in range(20):
            t, p = rng.uniform(0, math.pi), rng.uniform(0, TWO_PI)
            ref = math.sqrt(num / (den * math.pi)) * (1 + sign * math.cos(t)) ** p1 * math.sin(t) ** ps \
                * np.exp(1j * m * p)
            assert abs(oracle.swsh_m2(2, m, t, p) - ref) < 1e-14


def test_p1_higher_closed_forms(oracle):
    # textbook forms: (3,3), (3,-3), (3,2), (3,0), (4,4)
    t, p = 0.83, 2.1
    c, s = math.cos(t), math.sin(t)
    ref = {
        (3, 3): -math.sqrt(21 / (2 * math.pi)) * math.cos(t / 2) ** 5 * math.sin(t / 2) * np.exp(3j * p),
        (3, -3): math.sqrt(21 / (2 * math.pi)) * math.cos(t / 2) * math.sin(t / 2) ** 5 * np.exp(-3j * p),
        (3, 2): math.sqrt(7 / math.pi) * math.cos(t / 2) ** 4 * (-2 + 3 * c) / 2 * np.exp(2j * p),
        (3, 0): 0.25 * math.sqrt(105 / (2 * math.pi)) * c * s * s,
        (4, 4): 3 * math.sqrt(7 / math.pi) * math.cos(t / 2) ** 6 * math.sin(t / 2) ** 2 * np.exp(4j * p),
    }
    for (l, m), v in ref.items():
        assert abs(oracle.swsh_m2(l, m, t, p) - v) < 1e-13, (l, m)


def test_p1_orthonormal_and_sum_rule(oracle):
    # Gauss-Legendre in cos(theta) x uniform phi: exact for these trigonometric polynomials
    # (products of two harmonics of l <= 8: degree <= 16 in cos(theta), |m - m'| <= 16 < 24 in phi).  Every l the library
    # accepts (2 <= l <= 8, include/rift_ile.h) is covered.
    xs, ws = np.polynomial.legendre.leggauss(24)
    nphi = 36
    phis = TWO_PI * np.arange(nphi) / nphi
    modes = [(l, m) for l in range(2, 9) for m in range(-l, l + 1)]
    vals = np.array([[[oracle.swsh_m2(l, m, math.acos(x), p) for p in phis] for x in xs] for (l, m) in modes])
    gram = np.einsum("atp,btp,t->ab", np.conj(vals), vals, ws) * (TWO_PI / nphi)
    assert np.max(np.abs(gram - np.eye(len(modes)))) < 1e-12
    # sum_m |Y_lm|^2 = (2l+1)/(4 pi) at every angle
    for l in range(2, 9):
        for theta in (0.0, 0.3, 1.234, 2.9, math.pi):
            tot = sum(abs(oracle.swsh_m2(l, m, theta, 0.5)) ** 2 for m in range(-l, l + 1))
            assert abs(tot - (2 * l + 1) / (4 * math.pi)) < 1e-13


def test_p1_face_on_and_reflection(oracle):
    for l, m in [(2, 2), (2, 1), (2, 0), (2, -1), (2, -2)]:
        v = oracle.swsh_m2(l, m, 0.0, 0.7)
        if m == 2:
            assert abs(abs(v) - math.sqrt(5 / (4 * math.pi))) < 1e-15
        else:
            assert abs(v) < 1e-15
    rng = np.random.default_rng(3)
    for l in range(2, 9):
        for m in range(-l, l + 1):
            t, p = rng.uniform(0, math.pi), rng.uniform(0, TWO_PI)
            lhs = oracle.swsh_m2(l, -m, t, p)
            rhs = (-1) ** l * np.conj(oracle.swsh_m2(l, m, math.pi - t, p))
            assert abs(lhs - rhs) < 1e-13


def test_harmonics_use_minus_phi_ref(oracle):
    # the likelihood uses -2Y_lm(iota, -phi_ref): BASELINE.json north_star
    Y = oracle.harmonics([0.9], [0.4], [2, 3], [2, -1])[0]
    assert abs(Y[0] - oracle.swsh_m2(2, 2, 0.9, -0.4)) == 0.0
    assert abs(Y[1] - oracle.swsh_m2(3, -1, 0.9, -0.4)) == 0.0


# ------------------------------------------------------------------------------------------ P2
def test_p2_response_tensors():
    for name in ("H1", "L1", "V1"):
        r, D = synth.site(name)
        assert abs(np.trace(D)) < 1e-7
        assert abs(np.sum(D * D) - 0.5) < 1e-6
        assert np.allclose(D, D.T)
        assert 6.35e6 < np.linalg.norm(r) < 6.39e6


def test_p2_sky_average_is_one_fifth(oracle):
    _r, D = synth.site("H1")
    xs, ws = np.polynomial.legendre.leggauss(8)
    nra, npsi = 12, 8
    ra = TWO_PI * np.arange(nra) / nra
    psi = math.pi * np.arange(npsi) / npsi
    acc_p = acc_c = 0.0
    for x, w in zip(xs, ws):
        for a in ra:
            F = oracle.antenna(np.full(npsi, a), np.full(npsi, math.asin(x)), psi, 0.3, D[None])[:, 0]
            acc_p += w * np.sum(F.real ** 2)
            acc_c += w * np.sum(F.imag ** 2)
    norm = 2.0 * nra * npsi
    assert abs(acc_p / norm - 0.2) < 1e-10
    assert abs(acc_c / norm - 0.2) < 1e-10


def test_p2_psi_rotation_and_zenith(oracle):
    rng = np.random.default_rng(5)
    loc, resp = synth.detector_arrays(synth.CONFIGS[1])
    for _ in range(10):
        ra, dec, psi = rng.uniform(0, TWO_PI), math.asin(rng.uniform(-1, 1)), rng.uniform(0, math.pi)
        F0 = oracle.antenna(ra, dec, 0.0, 0.0, resp)[0]
        Fp = oracle.antenna(ra, dec, psi, 0.0, resp)[0]
        assert np.max(np.abs(Fp - np.exp(-2j * psi) * F0)) < 1e-14
    # a source at H1's zenith: |F| ~ 1 (0.99999, arms orthogonal to 1e-6)
    r, D = synth.site("H1")
    u = r / np.linalg.norm(r)
    F = oracle.antenna(math.atan2(u[1], u[0]), math.asin(u[2]), 0.2, 0.0, D[None])[0, 0]
    assert abs(abs(F) - 1.0) < 2e-5
    # GMST rotates the sky: F(ra, gmst) = F(ra - gmst, 0)
    assert abs(oracle.antenna(1.0, 0.3, 0.4, 0.25, D[None])[0, 0] - oracle.antenna(0.75, 0.3, 0.4, 0.0, D[None])[0, 0]) < 1e-15


# ------------------------------------------------------------------------------------------ P3
def test_p3_delays(oracle):
    gold = {r[0]: float(r[1]) for r in _rows("site_geometry.txt")}
    loc, _ = synth.detector_arrays(synth.CONFIGS[1])
    names = ["H1", "L1", "V1"]
    dt_s = 1.0 / 4096.0
    # source along r_H1: dt_H1 = -|r|/c
    u = loc[0] / np.linalg.norm(loc[0])
    dt, sh, _ = oracle.delays(math.atan2(u[1], u[0]), math.asin(u[2]), 0.0, loc, dt_s)
    assert abs(dt[0, 0] * 1e3 + gold["H1-geocentre"]) < 1e-3
    assert abs(dt[0, 0] + np.linalg.norm(loc[0]) / synth.C_LIGHT) < 1e-15
    # random sky: bounds, baselines, nearest-sample rounding
    rng = np.random.default_rng(7)
    ra, dec = rng.uniform(0, TWO_PI, 4000), np.arcsin(rng.uniform(-1, 1, 4000))
    dt, sh, fr = oracle.delays(ra, dec, 0.0, loc, dt_s)
    for k in range(3):
        assert np.all(np.abs(dt[:, k]) <= np.linalg.norm(loc[k]) / synth.C_LIGHT + 1e-15)
    assert np.all(np.abs(sh * dt_s - dt) <= 0.5 * dt_s + 1e-15)
    assert fr.sum() == 0
    for (a, b) in [(0, 1), (0, 2), (1, 2)]:
        base_ms = np.linalg.norm(loc[a] - loc[b]) / synth.C_LIGHT * 1e3
        assert abs(base_ms - gold[f"{names[a]}-{names[b]}"]) < 1e-3
        assert np.max(np.abs(dt[:, a] - dt[:, b])) * 1e3 <= base_ms + 1e-9
    # the extremum is reached along the baseline
    b = (loc[0] - loc[1]) / np.linalg.norm(loc[0] - loc[1])
    dt, _, _ = oracle.delays(math.atan2(b[1], b[0]), math.asin(b[2]), 0.0, loc, dt_s)
    assert abs(abs(dt[0, 0] - dt[0, 1]) * 1e3 - gold["H1-L1"]) < 1e-3
    # sign: a source overhead of a site arrives there BEFORE the geocentre
    assert dt[0, 0] - dt[0, 1] < 0
    # half-up rounding and GMST
    dtg, shg, _ = oracle.delays(1.3, 0.2, 0.4, loc, dt_s)
    dt0, sh0, _ = oracle.delays(0.9, 0.2, 0.0, loc, dt_s)
    assert np.max(np.abs(dtg - dt0)) < 1e-15
    assert np.all(shg == np.floor(dtg / dt_s + 0.5).astype(np.int32))


# ------------------------------------------------------------------------------------------ P4, P5
def _real_strain_toy(rng, K, M, nf, n_t, df, delta_t, F, Y, c, shifts, noise_amp):
    """Reading A3(ii): self-consistent real strain.  a(f) = h~_lm(+f), b(f) = conj h~_lm(-f), f > 0."""
    f = df * (1 + np.arange(nf))
    S = 0.5 + rng.uniform(0, 1, (K, nf))
    a = rng.standard_normal((M, nf)) + 1j * rng.standard_normal((M, nf))
    b = 0.3 * (rng.standard_normal((M, nf)) + 1j * rng.standard_normal((M, nf)))
    centre = (n_t - 1) // 2

    def htilde(k, Fk, Yv, cc, t):           # detector-k strain at f > 0 for a template arriving at time t
        return 0.5 * cc * (Fk * (Yv @ a) + np.conj(Fk) * (np.conj(Yv) @ b)) * np.exp(-2j * np.pi * f * t)

    d = np.array([htilde(k, F[k], Y, c, shifts[k] * delta_t) for k in range(K)])
    d = d + noise_amp * (rng.standard_normal((K, nf)) + 1j * rng.standard_normal((K, nf)))
    U = np.empty((K, M, M), complex)
    V = np.empty((K, M, M), complex)
    Q = np.empty((K, M, n_t), complex)
    t = (np.arange(n_t) - centre) * delta_t
    E = np.exp(2j * np.pi * np.outer(t, f))
    for k in range(K):
        U[k] = 2 * df * (np.einsum("af,bf->ab", np.conj(a), a / S[k]) + np.einsum("af,bf->ab", b, np.conj(b) / S[k]))
        V[k] = 2 * df * (np.einsum("af,bf->ab", np.conj(b), a / S[k]) + np.einsum("af,bf->ab", a, np.conj(b) / S[k]))
        for m in range(M):
            Q[k, m] = 2 * df * (E @ (np.conj(a[m]) * d[k] / S[k]) + np.conj(E) @ (b[m] * np.conj(d[k]) / S[k]))
    inner = lambda k, x, y: 4 * df * np.real(np.sum(np.conj(x) * y / S[k]))   # <x|y> for real series
    return dict(f=f, S=S, a=a, b=b, d=d, U=U, V=V, Q=Q, htilde=htilde, inner=inner, centre=centre)


def test_p4_factored_form_equals_definition_d1(oracle):
    rng = np.random.default_rng(11)
    K, M, nf, n_t, n_tau = 3, 4, 48, 41, 9
    df, delta_t = 1.0, 1.0 / 256.0
    F = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    Y = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    c = 1.7
    data_shift = np.array([2, -3, 1])
    toy = _real_strain_toy(rng, K, M, nf, n_t, df, delta_t, F, Y, 0.9, data_shift, noise_amp=0.7)
    # evaluate at DIFFERENT coefficients / distance / shifts than the injected ones
    F2 = F + 0.3 * (rng.standard_normal(K) + 1j * rng.standard_normal(K))
    Y2 = Y + 0.3 * (rng.standard_normal(M) + 1j * rng.standard_normal(M))
    s2 = np.array([4, -6, 0], dtype=np.int32)
    _tm, series, quad = oracle.lnl_core(F2, Y2, c, s2, toy["Q"], toy["U"], toy["V"], n_tau=n_tau)
    j0 = (n_t - n_tau) // 2
    for j in range(n_tau):
        direct = 0.0
        for k in range(K):
            t_k = (j0 + s2[k] + j - toy["centre"]) * delta_t
            h = toy["htilde"](k, F2[k], Y2, c, t_k)
            r = h - toy["d"][k]
            direct += -0.5 * (toy["inner"](k, r, r) - toy["inner"](k, toy["d"][k], toy["d"][k]))
        assert abs(series[j] - direct) < 1e-10 * max(1.0, abs(direct)), (j, series[j], direct)
    assert quad > 0


def test_p5_zero_noise_peak_is_half_rho_squared(oracle):
    rng = np.random.default_rng(13)
    cfg = synth.CONFIGS[1]
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    theta = synth.true_point(cfg, 0)
    delta_t = 1.0 / 256.0
    F, Y, _ = oracle.geometry_at(theta, loc, resp, 0.0, ml, mm, delta_t)
    shifts = np.array([3, -2, 5], dtype=np.int32)
    c = synth.D_REF_MPC / theta[5]
    n_t = 33
    toy = _real_strain_toy(rng, 3, 5, 64, n_t, 1.0, delta_t, F, Y, c, shifts, noise_amp=0.0)
    rho2 = sum(toy["inner"](k, toy["d"][k], toy["d"][k]) for k in range(3))
    tm, series, _q = oracle.lnl_core(F, Y, c, shifts, toy["Q"], toy["U"], toy["V"])
    centre = (n_t - 1) // 2
    assert abs(series[centre] - 0.5 * rho2) < 1e-11 * rho2
    assert np.argmax(series) == centre
    assert np.all(series <= 0.5 * rho2 + 1e-9)
    assert tm <= 0.5 * rho2 and tm >= 0.5 * rho2 - math.log(n_t) - 1e-9


def test_p5_literal_recipe_closed_form(oracle):
    """Reading A3(i): the literal one-sided recipe of configs[0] does NOT give rho^2/2; noise-free, at the
    injected point it gives c^2 sum_k (3/4 |F_k|^2 Y^dag U_k Y - 1/4 Re F_k^2 Y^T V_k Y)."""
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=8.0)
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    theta = synth.true_point(cfg, 0)
    F, Y, sh = oracle.geometry_at(theta, loc, resp, cfg.gmst, ml, mm, cfg.delta_t)
    c = synth.D_REF_MPC / theta[5]
    pd = synth.make_point(cfg, 0, np.outer(F, Y), sh, c, noise=False)
    _tm, series, _q = oracle.lnl_core(F, Y, c, sh, pd.Q, pd.U, pd.V)
    expect = 0.0
    for k in range(cfg.n_det):
        yuy = np.conj(Y) @ pd.U[k] @ Y
        yvy = Y @ pd.V[k] @ Y
        expect += c * c * (0.75 * abs(F[k]) ** 2 * yuy.real - 0.25 * (F[k] ** 2 * yvy).real)
    centre = (cfg.n_t - 1) // 2
    assert abs(series[centre] - expect) < 1e-9 * abs(expect)
    assert np.argmax(series) == centre


# ------------------------------------------------------------------------------------------ P6
def test_p6_distance_parabola(oracle):
    rng = np.random.default_rng(17)
    K, M, n_t = 2, 3, 15
    Q = rng.standard_normal((K, M, n_t)) + 1j * rng.standard_normal((K, M, n_t))
    A = rng.standard_normal((K, M, M)) + 1j * rng.standard_normal((K, M, M))
    U = np.einsum("kab,kcb->kac", A, np.conj(A))            # Hermitian positive definite
    B = rng.standard_normal((K, M, M)) + 1j * rng.standard_normal((K, M, M))
    V = 0.1 * (B + np.swapaxes(B, 1, 2))
    F = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    Y = rng.standard_normal(M) + 1j * rng.standard_normal(M)
    s = np.zeros(K, dtype=np.int32)
    ser = {c: oracle.lnl_core(F, Y, c, s, Q, U, V)[1] for c in (1.0, 2.0, 3.7)}
    quad = {c: oracle.lnl_core(F, Y, c, s, Q, U, V)[2] for c in (1.0, 2.0)}
    b = quad[1.0]
    assert abs(quad[2.0] - 4 * b) < 1e-12 * abs(b)
    a = ser[1.0] + b                                         # lnL_j(c) = c a_j - c^2 b   (Eq. (D5))
    assert np.max(np.abs(ser[3.7] - (3.7 * a - 3.7 ** 2 * b))) < 1e-11 * (1 + np.max(np.abs(a)))
    j = int(np.argmax(a))
    cstar = a[j] / (2 * b)
    peak = oracle.lnl_core(F, Y, cstar, s, Q, U, V)[1][j]
    assert abs(peak - a[j] ** 2 / (4 * b)) < 1e-11 * abs(peak)


# ------------------------------------------------------------------------------------------ P7, P8
def _random_problem(rng, K, M, n_t):
    Q = rng.standard_normal((K, M, n_t)) + 1j * rng.standard_normal((K, M, n_t))
    A = rng.standard_normal((K, M, M)) + 1j * rng.standard_normal((K, M, M))
    U = 0.05 * np.einsum("kab,kcb->kac", A, np.conj(A))
    B = rng.standard_normal((K, M, M)) + 1j * rng.standard_normal((K, M, M))
    V = 0.01 * (B + np.swapaxes(B, 1, 2))
    F = 0.5 * (rng.standard_normal(K) + 1j * rng.standard_normal(K))
    Y = 0.5 * (rng.standard_normal(M) + 1j * rng.standard_normal(M))
    s = rng.integers(-7, 8, K).astype(np.int32)
    return Q, U, V, F, Y, s


def test_p7_time_marginal_invariants(oracle):
    rng = np.random.default_rng(19)
    K, M, n_t = 3, 4, 37
    Q, U, V, F, Y, s = _random_problem(rng, K, M, n_t)
    c = 1.3
    # constant-in-time Q: the marginal equals the (constant) lnL
    Qc = np.repeat(Q[:, :, :1], n_t, axis=2)
    tm, series, _ = oracle.lnl_core(F, Y, c, s, Qc, U, V)
    assert np.max(np.abs(series - series[0])) < 1e-13
    assert abs(tm - series[0]) < 1e-13
    # a common circular shift of every Q leaves the marginal unchanged (N_tau = N_t, reading A4)
    tm0, ser0, _ = oracle.lnl_core(F, Y, c, s, Q, U, V)
    for n in (1, 5, -11, n_t):
        tm1, ser1, _ = oracle.lnl_core(F, Y, c, s, np.roll(Q, n, axis=2), U, V)
        assert abs(tm1 - tm0) < 1e-12
        assert np.max(np.abs(np.roll(ser0, n) - ser1)) < 1e-12
    # shifting only detector k's Q by n == shifting s_k by -n
    for k, n in ((0, 3), (2, -4)):
        Q2 = Q.copy()
        Q2[k] = np.roll(Q[k], n, axis=1)
        s2 = s.copy()
        s2[k] -= n
        a = oracle.lnl_core(F, Y, c, s, Q2, U, V)[1]
        b = oracle.lnl_core(F, Y, c, s2, Q, U, V)[1]
        assert np.max(np.abs(a - b)) < 1e-13
    # guard-band window: n_tau < n_t reads the central n_tau samples of the circular series
    n_tau = 21
    j0 = (n_t - n_tau) // 2
    tm_w, ser_w, _ = oracle.lnl_core(F, Y, c, s, Q, U, V, n_tau=n_tau)
    assert np.max(np.abs(ser_w - ser0[j0:j0 + n_tau])) == 0.0
    # brute-force definition of the series for one j
    j = 5
    x = sum((np.conj(F[k] * Y[a]) * Q[k, a, (j + s[k]) % n_t]).real for k in range(K) for a in range(M))
    q = 0.25 * c * c * sum(abs(F[k]) ** 2 * (np.conj(Y) @ U[k] @ Y).real + (F[k] ** 2 * (Y @ V[k] @ Y)).real
                           for k in range(K))
    assert abs(ser0[j] - (c * x - q)) < 1e-12


def test_p8_layout_invariants(oracle):
    rng = np.random.default_rng(23)
    K, M, n_t = 3, 5, 29
    Q, U, V, F, Y, s = _random_problem(rng, K, M, n_t)
    c = 0.8
    tm0, ser0, q0 = oracle.lnl_core(F, Y, c, s, Q, U, V)
    pm = rng.permutation(M)
    tm1, ser1, q1 = oracle.lnl_core(F, Y[pm], c, s, Q[:, pm], U[:, pm][:, :, pm], V[:, pm][:, :, pm])
    assert abs(tm1 - tm0) < 1e-12 and abs(q1 - q0) < 1e-12
    pk = rng.permutation(K)
    tm2, ser2, q2 = oracle.lnl_core(F[pk], Y, c, s[pk], Q[pk], U[pk], V[pk])
    assert abs(tm2 - tm0) < 1e-12 and abs(q2 - q0) < 1e-12
    # a transposed U must CHANGE the answer (so a transposition mistake is visible)
    assert abs(oracle.lnl_core(F, Y, c, s, Q, np.swapaxes(U, 1, 2), V)[2] - q0) > 1e-6
    # rescaling Q -> sQ, (U,V) -> s^2 (U,V), c -> c/s
    sc = 3.0
    tm3, _, _ = oracle.lnl_core(F, Y, c / sc, s, sc * Q, sc * sc * U, sc * sc * V)
    assert abs(tm3 - tm0) < 1e-11


def test_eval_batch_composes_geometry_and_core(oracle):
    cfg = synth.CONFIGS[0]
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    rng = np.random.default_rng(29)
    n_t = 21
    Q, U, V, _F, _Y, _s = _random_problem(rng, cfg.n_det, cfg.n_modes, n_t)
    params = synth.prior_draw(rng, 16)
    lnL, sh, _fr = oracle.eval_batch(loc, resp, 0.1, ml, mm, 1.0 / 512.0, 1000.0, Q, U, V, params)
    for i in (0, 7, 15):
        F = oracle.antenna(params[0, i], params[1, i], params[2, i], 0.1, resp)[0]
        Y = oracle.harmonics(params[3, i], params[4, i], ml, mm)[0]
        _dt, s, _ = oracle.delays(params[0, i], params[1, i], 0.1, loc, 1.0 / 512.0)
        assert np.all(s[0] == sh[i])
        tm, _, _ = oracle.lnl_core(F, Y, 1000.0 / params[5, i], s[0], Q, U, V)
        assert lnL[i] == tm
    bad = params.copy()
    bad[5, 3] = -1.0
    bad[0, 4] = np.nan
    lnL2, _, _ = oracle.eval_batch(loc, resp, 0.1, ml, mm, 1.0 / 512.0, 1000.0, Q, U, V, bad)
    assert np.isnan(lnL2[3]) and np.isnan(lnL2[4])
    ok = np.ones(16, bool)
    ok[[3, 4]] = False
    assert np.all(lnL2[ok] == lnL[ok])


# ------------------------------------------------------------------------------------------ P9
def _lme_longdouble(x):
    x = np.asarray(x, dtype=np.longdouble)
    m = np.max(x)
    if not np.isfinite(m):
        return float(m)
    return float(m + np.log(np.sum(np.exp(x - m))) - np.log(np.longdouble(x.size)))


def test_p9_logsumexp_range(oracle):
    rng = np.random.default_rng(31)
    x = rng.uniform(-900.0, 450.0, 411)                  # spread > 800: exp() alone would overflow / underflow
    assert abs(oracle.logmeanexp(x) - _lme_longdouble(x)) < 1e-12 * 450
    x = np.full(411, -np.inf)
    x[17] = 3.25
    assert abs(oracle.logmeanexp(x) - (3.25 - math.log(411))) < 1e-14
    assert oracle.logmeanexp(np.full(5, -np.inf)) == -np.inf
    assert math.isnan(oracle.logmeanexp(np.array([1.0, np.nan])))
    x = np.array([800.0, 799.0, -800.0])
    assert abs(oracle.logmeanexp(x) - (800 + math.log1p(math.exp(-1.0) + math.exp(-1600.0)) - math.log(3))) < 1e-12
    # rho = 30: peak lnL = 450 through the whole core
    n_t = 51
    Q = np.zeros((1, 1, n_t), complex)
    Q[0, 0, 25] = 900.0
    U = np.array([[[900.0 * 2]]], complex)
    V = np.zeros((1, 1, 1), complex)
    tm, ser, _ = oracle.lnl_core([1.0], [1.0], 1.0, [0], Q, U, V)
    assert abs(ser[25] - 450.0) < 1e-12 and abs(ser[0] + 450.0) < 1e-12
    assert abs(tm - _lme_longdouble(ser)) < 1e-12 * 450 and np.isfinite(tm)


# ------------------------------------------------------------------------------------------ P10, P11
def test_p10_reduce_special_cases(oracle):
    r = oracle.reduce(np.array([2.5]), np.array([-0.5]))
    assert abs(r["lnZ"] - 2.0) < 1e-15 and r["n_eff"] == 1.0 and r["n_ess"] == 1.0 and r["rel_err"] == 0.0
    rng = np.random.default_rng(37)
    lw = rng.standard_normal(1000)
    r = oracle.reduce(np.zeros(1000), lw)                 # lnL = 0  =>  lnZ = ln mean w
    assert abs(r["lnZ"] - math.log(np.mean(np.exp(lw)))) < 1e-13
    r = oracle.reduce(np.full(64, -3.0))                  # equal lnL => n_eff = n_ess = N, zero error
    assert abs(r["n_eff"] - 64) < 1e-12 and abs(r["n_ess"] - 64) < 1e-12 and r["rel_err"] < 1e-7
    assert abs(r["lnZ"] + 3.0) < 1e-14
    # definitions (B1), (B2) and the unbiased variance of the mean (reading A20), by brute force
    lnL = 5 * rng.standard_normal(500)
    w = np.exp(lnL + lw[:500])
    r = oracle.reduce(lnL, lw[:500])
    assert abs(r["lnZ"] - math.log(w.mean())) < 1e-12
    assert abs(r["n_eff"] - w.sum() / w.max()) < 1e-10
    assert abs(r["n_ess"] - w.sum() ** 2 / np.sum(w * w)) < 1e-10
    assert abs(r["rel_err"] - math.sqrt(np.var(w, ddof=1) / w.size) / w.mean()) < 1e-12
    # the printed (B3) differs from it only at O(1/N^2) relative
    printed = (-(w.mean() ** 2) + np.sum(w * w) / (w.size - 1)) / w.size / w.mean() ** 2
    assert abs(printed - r["rel_err"] ** 2) < 2.0 / w.size * printed


def test_p10_merge_equals_one_pass_and_histograms(oracle):
    rng = np.random.default_rng(41)
    n, nb = 3000, 10
    params = synth.prior_draw(rng, n)
    lnL = 8 * rng.standard_normal(n)
    lw = 0.3 * rng.standard_normal(n)
    one = oracle.reduce(lnL, lw, params, synth.HIST_LO, synth.HIST_HI, nb)
    st = oracle.ReduceState(nb, want_hist=True)
    for a, b in ((0, 700), (700, 701), (701, n)):         # the maximum moves between chunks
        st.accumulate(lnL[a:b], lw[a:b], params[:, a:b], synth.HIST_LO, synth.HIST_HI)
    two = st.finalize()
    for key in ("lnZ", "rel_err", "n_eff", "n_ess"):
        assert abs(one[key] - two[key]) < 1e-11 * max(1.0, abs(one[key])), key
    assert np.max(np.abs(one["hist"] - two["hist"])) < 1e-12
    # Eq. (20): with equal-size chunks the pooled mean is the running average of chunk integrals
    I1 = math.exp(oracle.reduce(lnL[:1500], lw[:1500])["lnZ"])
    I2 = math.exp(oracle.reduce(lnL[1500:], lw[1500:])["lnZ"])
    assert abs(math.exp(one["lnZ"]) - (1 * I1 + I2) / 2) < 1e-12 * math.exp(one["lnZ"])
    # histograms: normalised, and equal to numpy's weighted histogram
    w = np.exp(lnL + lw - np.max(lnL + lw))
    for d in range(6):
        assert abs(one["hist"][d].sum() - 1.0) < 1e-12
        ref, _ = np.histogram(params[d], bins=nb, range=(synth.HIST_LO[d], synth.HIST_HI[d]), weights=w)
        assert np.max(np.abs(one["hist"][d] - ref / w.sum())) < 1e-12
    # out-of-range values are clamped to the end bins
    p2 = params.copy()
    p2[5, :10] = 1e9
    p2[5, 10:20] = -5.0
    h = oracle.reduce(lnL, lw, p2, synth.HIST_LO, synth.HIST_HI, nb)["hist"]
    assert abs(h[5].sum() - 1.0) < 1e-12


def test_p11_appendix_b_toy(oracle):
    rng = np.random.default_rng(43)
    N = 400_000
    for row in _rows("appendix_b_toy.txt"):
        alpha, var = float(row[0]), float(row[1])
        x = rng.uniform(0, 1, N) ** (1.0 / alpha)          # x ~ p_s = alpha x^(alpha-1)
        lw = -np.log(alpha) - (alpha - 1) * np.log(x)
        r = oracle.reduce(np.zeros(N), lw)
        # <w> = 1 within 5 sigma of the closed-form variance
        assert abs(math.exp(r["lnZ"]) - 1.0) < 5 * math.sqrt(var / N)
        # N rel_err^2 -> V(w)/<w>^2
        tol = 0.05 if alpha < 1.4 else 0.2                  # alpha = 1.5: fourth moment diverges, slow convergence
        assert abs(N * r["rel_err"] ** 2 / var - 1.0) < tol
        assert abs(N / r["n_ess"] - 1.0 - var) < tol * (1 + var)
    # median n_eff over repeated draws vs Eq. (B5), alpha = 3
    alpha, N, reps = 3.0, 20_000, 400
    neff = []
    for _ in range(reps):
        x = rng.uniform(0, 1, N) ** (1.0 / alpha)
        neff.append(oracle.reduce(np.zeros(N), -np.log(alpha) - (alpha - 1) * np.log(x))["n_eff"])
    b5 = N * alpha * (N / math.log(2)) ** (-(alpha - 1) / alpha)
    assert abs(np.median(neff) / b5 - 1.0) < 0.15


# ------------------------------------------------------------------------------------------ P12
def test_p12_direct_quadrature_of_the_extrinsic_integral(oracle):
    """C0 geometry at low amplitude (rho = 2.5) on a short window: tensor-product quadrature of
    int L p dtheta against the Monte-Carlo lnZ of Eq. (3).  Catches normalisation mistakes."""
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=2.5, f_s=512.0, t_window=0.03)
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    inp = synth.build_inputs(cfg, lambda th: oracle.geometry_at(th, loc, resp, cfg.gmst, ml, mm, cfg.delta_t))
    Q, U, V = inp.Q[0], inp.U[0], inp.V[0]
    ev = lambda p: oracle.eval_batch(loc, resp, cfg.gmst, ml, mm, cfg.delta_t, synth.D_REF_MPC, Q, U, V, p)[0]

    # Monte Carlo with prior draws (ln w = 0)
    n_mc = 400_000
    params = synth.prior_draw(np.random.default_rng(47), n_mc)
    mc = oracle.reduce(ev(params))

    # quadrature: trapezoid (periodic) in RA, psi, phi; Gauss-Legendre in sin(dec), cos(iota), D
    n_ra, n_sd, n_psi, n_ci, n_phi, n_d = 48, 20, 6, 10, 8, 12
    xs, wsd = np.polynomial.legendre.leggauss(n_sd)
    xc, wci = np.polynomial.legendre.leggauss(n_ci)
    xd, wd = np.polynomial.legendre.leggauss(n_d)
    D = 0.5 * (synth.D_MAX_MPC - synth.D_MIN_MPC) * xd + 0.5 * (synth.D_MAX_MPC + synth.D_MIN_MPC)
    pD = 3 * D ** 2 / (synth.D_MAX_MPC ** 3 - synth.D_MIN_MPC ** 3) * 0.5 * (synth.D_MAX_MPC - synth.D_MIN_MPC) * wd
    ra = TWO_PI * np.arange(n_ra) / n_ra
    psi = math.pi * np.arange(n_psi) / n_psi
    phi = TWO_PI * np.arange(n_phi) / n_phi
    g = np.meshgrid(ra, np.arcsin(xs), psi, np.arccos(xc), phi, D, indexing="ij")
    wgt = np.einsum("a,b,c,d,e,f->abcdef", np.full(n_ra, 1.0 / n_ra), 0.5 * wsd, np.full(n_psi, 1.0 / n_psi),
                    0.5 * wci, np.full(n_phi, 1.0 / n_phi), pD).ravel()
    assert abs(wgt.sum() - 1.0) < 1e-12
    lnL = ev(np.array([x.ravel() for x in g]))
    m = lnL.max()
    lnZ_quad = m + math.log(np.sum(wgt * np.exp(lnL - m)))
    assert abs(mc["lnZ"] - lnZ_quad) < max(4 * mc["rel_err"], 5e-3), (mc, lnZ_quad)
    assert abs(lnZ_quad) > 0.02      # the integrand is not trivially flat
