"""Pins of oracle/dmarg_oracle.c (distance marginalisation): the oracle
against closed forms, a library integrator, its own convergence and the 6-D Monte Carlo evidence of the plain oracle."""
import math

import numpy as np
import pytest

from paper_2210_07912_b200 import synth

from helpers import build, oracle_eval

D_REF, D_MIN, D_MAX = synth.D_REF_MPC, synth.D_MIN_MPC, synth.D_MAX_MPC


def test_p19_rule_is_normalised_and_positive(oracle):
    for alpha in (2.0, 0.0, -1.0, -2.0):
        for n_panels in (1, 8, 64):
            D, W = oracle.dmarg_rule(D_MIN, D_MAX, alpha, n_panels)
            assert np.all(np.diff(D) > 0) and D[0] > D_MIN and D[-1] < D_MAX and np.all(W > 0)
            if n_panels >= 8:
                assert abs(W.sum() - 1.0) < 1e-12, (alpha, n_panels)      # int p(D) dD = 1
    # x = 0, b = 0: the integrand is the prior, the marginal likelihood is 1
    assert abs(oracle.dmarg_core(np.zeros(5), 0.0, D_REF, D_MIN, D_MAX, 2.0, 64)) < 1e-12


@pytest.mark.parametrize("x,b", [(30.0, 10.0), (150.0, 80.0), (3.0, 0.2), (-20.0, 5.0), (400.0, 8.0), (0.3, 40.0)])
def test_p19_closed_form_uniform_in_c(oracle, x, b):
    """alpha = -2: p(D) dD is proportional to dc (c = D_ref/D), so one tau gives a Gaussian integral in c,
    int_{c2}^{c1} exp(c x - c^2 b) dc = sqrt(pi/b)/2 exp(x^2/4b) [erf(sqrt(b)(c1 - mu)) - erf(sqrt(b)(c2 - mu))], mu = x/2b --
    peak inside the range, at its edges and outside it."""
    c1, c2, mu = D_REF / D_MIN, D_REF / D_MAX, x / (2.0 * b)
    from scipy.special import erfc, erfcx  # noqa: F401
    sb = math.sqrt(b)
    # difference of error functions, written so that it survives a peak far outside the range
    lo, hi = sb * (c2 - mu), sb * (c1 - mu)
    if lo > 0:
        diff = erfc(lo) - erfc(hi)
    elif hi < 0:
        diff = erfc(-hi) - erfc(-lo)
    else:
        diff = math.erf(hi) - math.erf(lo)
    ln_int = 0.5 * math.log(math.pi / b) - math.log(2.0) + x * x / (4.0 * b) + math.log(diff)
    want = ln_int - math.log(D_REF) - math.log(1.0 / D_MIN - 1.0 / D_MAX)
    got = oracle.dmarg_core([x], b, D_REF, D_MIN, D_MAX, -2.0, 2048)
    assert abs(got - want) < 1e-9 * max(1.0, abs(want)), (got, want)


@pytest.mark.parametrize("b", [0.5, 20.0, 120.0])
def test_p20_library_integrator_d2_prior(oracle, b):
    """alpha = 2 (the d_L^2 prior), three tau: scipy.integrate.quad on the same integrand."""
    from scipy.integrate import quad
    xs = np.array([2.0 * b * 1.3, 2.0 * b * 0.9 - 4.0, -1.0])              # peaks at c = 1.3, ~0.9, none
    norm = 3.0 / (D_MAX ** 3 - D_MIN ** 3)
    ref = max(float(np.max(c * xs) - c * c * b) for c in np.linspace(D_REF / D_MAX, D_REF / D_MIN, 4000))
    tot = 0.0
    for x in xs:
        f = lambda D: norm * D * D * math.exp(D_REF / D * x - (D_REF / D) ** 2 * b - ref)   # noqa: E731
        mu = x / (2.0 * b)
        pts = [D_REF / mu] if mu > D_REF / D_MAX and mu < D_REF / D_MIN else None
        val, _err = quad(f, D_MIN, D_MAX, points=pts, limit=400, epsabs=0.0, epsrel=1e-12)
        tot += val
    want = ref + math.log(tot / len(xs))
    got = oracle.dmarg_core(xs, b, D_REF, D_MIN, D_MAX, 2.0, 1024)
    assert abs(got - want) < 1e-9 * max(1.0, abs(want)), (got, want)


def test_p21_convergence_in_the_number_of_panels(oracle):
    """The rule converges fast in the number of panels; the error of the 64-node rule the CUDA path defaults to is recorded
    here for a quiet and a loud signal (DESIGN.md section 12 quotes these numbers)."""
    rng = np.random.default_rng(4)
    for rho, tol64 in ((5.0, 1e-6), (12.0, 5e-3), (30.0, 1.5)):
        b = 0.5 * rho * rho                                              # peak at c = 1: x = 2 b, lnL_max = b = rho^2/2
        x = 2.0 * b * (1.0 - 0.5 * rng.uniform(0, 1, 40) ** 2)
        ref = oracle.dmarg_core(x, b, D_REF, D_MIN, D_MAX, 2.0, 4096)
        errs = [abs(oracle.dmarg_core(x, b, D_REF, D_MIN, D_MAX, 2.0, n) - ref) for n in (8, 32, 128, 512)]
        assert errs[0] < tol64, (rho, errs)
        assert errs[2] < 1e-9 and errs[3] < 1e-10, (rho, errs)
        assert errs[1] <= errs[0] + 1e-12


def test_p22_five_dimensional_evidence_matches_six_dimensional(oracle):
    """Marginalising the distance inside the likelihood and integrating the other five parameters by Monte Carlo must give
    the evidence of the 6-D Monte Carlo integral of the plain oracle (same intrinsic point, same priors) within errors."""
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=4.0)
    inp = build(oracle, cfg)
    n6, n5 = 400_000, 12_000
    p6 = synth.prior_draw(np.random.default_rng(11), n6)
    r6 = oracle.reduce(oracle_eval(oracle, inp, 0, p6)[0])
    p5 = synth.prior_draw(np.random.default_rng(12), n5)
    l5 = oracle.eval_batch_dmarg(inp.det_location, inp.det_response, cfg.gmst, inp.mode_l, inp.mode_m, cfg.delta_t, D_REF,
                                 inp.Q[0], inp.U[0], inp.V[0], p5[:5], D_MIN, D_MAX, 32)[0]
    r5 = oracle.reduce(l5)
    sig = math.hypot(r6["rel_err"], r5["rel_err"])
    assert abs(r6["lnZ"] - r5["lnZ"]) < 3.0 * sig + 1e-3, (r6["lnZ"], r5["lnZ"], sig)
    assert r5["n_ess"] / n5 > 2.0 * r6["n_ess"] / n6                      # fewer dimensions: better sampling efficiency
