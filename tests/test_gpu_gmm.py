"""GPU parity of the Gaussian-mixture adaptive sampler (include/rift_gmm.h, PAPER.md section
IV.C.1 and Appendix A) against oracle/gmm_oracle.py on the same seeded inputs: EM iteration by iteration, the online merge, the
component masses, the density, the truncated draws (same counter-based random numbers), and an adaptive integration loop."""
import math

import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from oracle import gmm_oracle as go

pytestmark = pytest.mark.gpu

TOL_EM = 1e-9                # sums of 1e4-1e5 terms in another order, then divisions (relative, on means / covariances / weights)
TOL_DRAW = 1e-11             # normcdfinv vs scipy's ndtri through A z + mu (absolute, on O(1) coordinates)
TOL_LNP = 1e-9               # ln p_s: the component masses Z_k by Gauss-Legendre vs adaptive quadrature


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _data(rng, n, d):
    mus = [np.array([-1.0, 0.5])[:d], np.array([1.5, 1.2])[:d], np.array([0.3, -0.8])[:d]]
    covs = [np.array([[0.4, 0.25], [0.25, 0.3]])[:d, :d], np.array([[0.15, -0.05], [-0.05, 0.5]])[:d, :d], np.eye(2)[:d, :d] * 0.1]
    k = rng.choice(3, size=n, p=[0.5, 0.3, 0.2])
    x = np.stack([rng.multivariate_normal(mus[j], covs[j]) for j in k])
    return x


def _init(d):
    mu0 = np.array([[-0.5, 0.0], [1.0, 1.0], [0.0, -0.5]])[:, :d]
    cov0 = np.array([np.eye(d) * 0.5] * 3)
    return mu0, cov0, np.array([0.3, 0.4, 0.3])


@pytest.mark.parametrize("d,n,weighted", [(2, 60_001, True), (1, 4_099, True), (2, 777, False)])
def test_em_matches_oracle_iteration_by_iteration(torch, d, n, weighted):
    rng = np.random.default_rng(100 + n)
    x = _data(rng, n, d)
    ln_w = rng.normal(0.0, 2.0, n) + 700.0 if weighted else None            # a large common offset must not matter
    if weighted:
        ln_w[5] = -np.inf
        ln_w[6] = np.nan                                                     # treated as weight 0
    lo, hi = x.min(axis=0) - 1.0, x.max(axis=0) + 1.0
    mu0, cov0, pi0 = _init(d)
    xs = [_dev(torch, x[:, j]) for j in range(d)]
    lw = None if ln_w is None else _dev(torch, ln_w)
    lw_o = np.zeros(n) if ln_w is None else np.where(np.isnan(ln_w), -np.inf, ln_w)
    for iters, reg in ((1, 0.0), (4, 1e-6), (9, 0.0)):
        g = rift.rift_gmm_create(d, 3, lo, hi)
        rift.rift_gmm_set_model(g, mu0, cov0, pi0)
        it, ll = rift.rift_gmm_fit(g, n, xs, lw, iters, 0.0, reg)
        mu, cov, pi, nt = rift.rift_gmm_get_model(g)
        mu_o, cov_o, pi_o, it_o, ll_o = go.fit(x, lw_o, mu0, cov0, pi0, iters, 0.0, reg)
        assert it == it_o == iters and nt == n
        assert abs(ll - ll_o) < TOL_EM * max(1.0, abs(ll_o))
        assert np.max(np.abs(mu - mu_o)) < TOL_EM and np.max(np.abs(cov - cov_o)) < TOL_EM and np.max(np.abs(pi - pi_o)) < TOL_EM
        rift.rift_gmm_destroy(g)
    # the tolerance stops both at the same iteration, and repeating the call gives the same bits (fixed reduction order)
    g = rift.rift_gmm_create(d, 3, lo, hi)
    rift.rift_gmm_set_model(g, mu0, cov0, pi0)
    it, ll = rift.rift_gmm_fit(g, n, xs, lw, 300, 1e-7, 0.0)
    first = rift.rift_gmm_get_model(g)
    it_o = go.fit(x, lw_o, mu0, cov0, pi0, 300, 1e-7, 0.0)[3]
    assert it == it_o and 1 < it < 300
    rift.rift_gmm_set_model(g, mu0, cov0, pi0)
    rift.rift_gmm_fit(g, n, xs, lw, 300, 1e-7, 0.0)
    again = rift.rift_gmm_get_model(g)
    assert all(np.array_equal(a, b) for a, b in zip(first[:3], again[:3]))
    rift.rift_gmm_destroy(g)


def test_tempered_fit_matches_oracle(torch):
    rng = np.random.default_rng(17)
    d, n = 2, 50_000
    x = _data(rng, n, d)
    ln_w = rng.normal(0.0, 7.0, n) - 300.0
    ln_w[11] = -np.inf
    lo, hi = x.min(axis=0) - 1.0, x.max(axis=0) + 1.0
    mu0, cov0, pi0 = _init(d)
    xs, lw = [_dev(torch, x[:, j]) for j in range(d)], _dev(torch, ln_w)
    for ess_min in (500.0, 1.0, 1e9):
        g = rift.rift_gmm_create(d, 3, lo, hi)
        rift.rift_gmm_set_model(g, mu0, cov0, pi0)
        temper, it, ll = rift.rift_gmm_fit_tempered(g, n, xs, lw, ess_min, 5, 0.0, 1e-6)
        t_o = go.temper_for_ess(ln_w, ess_min)
        assert temper == t_o, (temper, t_o)                 # the same 20 bisection decisions
        assert (ess_min == 1.0) == (temper == 1.0) and (ess_min == 1e9) == (temper == 0.0)
        mu, cov, pi, _nt = rift.rift_gmm_get_model(g)
        mu_o, cov_o, pi_o, it_o, ll_o = go.fit(x, np.where(np.isfinite(ln_w), t_o * np.where(np.isfinite(ln_w), ln_w, 0.0), -np.inf), mu0, cov0, pi0, 5, 0.0,
                                                1e-6)
        assert it == it_o and abs(ll - ll_o) < TOL_EM * max(1.0, abs(ll_o))
        assert np.max(np.abs(mu - mu_o)) < TOL_EM and np.max(np.abs(cov - cov_o)) < TOL_EM and np.max(np.abs(pi - pi_o)) < TOL_EM
        rift.rift_gmm_destroy(g)


def test_online_update_merges_like_the_oracle(torch):
    rng = np.random.default_rng(7)
    d, n1, n2 = 2, 20_000, 12_345
    x1, x2 = _data(rng, n1, d), _data(rng, n2, d) + 0.05
    lw1, lw2 = rng.normal(0, 1, n1), rng.normal(0, 1, n2)
    lo, hi = np.array([-6.0, -6.0]), np.array([6.0, 6.0])
    mu0, cov0, pi0 = _init(d)
    g = rift.rift_gmm_create(d, 3, lo, hi)
    rift.rift_gmm_set_model(g, mu0, cov0, pi0)
    rift.rift_gmm_fit(g, n1, [_dev(torch, x1[:, j]) for j in range(d)], _dev(torch, lw1), 5)
    rift.rift_gmm_fit(g, n2, [_dev(torch, x2[:, j]) for j in range(d)], _dev(torch, lw2), 5, merge=1)
    mu, cov, pi, nt = rift.rift_gmm_get_model(g)
    a = go.fit(x1, lw1, mu0, cov0, pi0, 5)
    b = go.fit(x2, lw2, a[0], a[1], a[2], 5)                                 # G3: trained from the old model's parameters
    mu_o, cov_o, pi_o = go.merge(a[0], a[1], a[2], n1, b[0], b[1], b[2], n2)
    assert nt == n1 + n2 and abs(pi.sum() - 1.0) < 1e-12
    assert np.max(np.abs(mu - mu_o)) < TOL_EM and np.max(np.abs(cov - cov_o)) < TOL_EM and np.max(np.abs(pi - pi_o)) < TOL_EM
    # a permuted new model is matched back: set the old model, fit from a permuted start, merge
    perm = [2, 0, 1]
    rift.rift_gmm_set_model(g, a[0], a[1], a[2], n1)
    h2 = rift.rift_gmm_create(d, 3, lo, hi)
    rift.rift_gmm_set_model(h2, a[0][perm], a[1][perm], a[2][perm], 0)
    rift.rift_gmm_fit(h2, n2, [_dev(torch, x2[:, j]) for j in range(d)], _dev(torch, lw2), 5)
    mu_p, cov_p, pi_p, _ = rift.rift_gmm_get_model(h2)
    assert go.match_components(a[0], a[1], mu_p, cov_p) == perm
    mo = go.merge(a[0], a[1], a[2], n1, mu_p, cov_p, pi_p, n2)
    assert np.max(np.abs(mo[0] - mu_o)) < 1e-8                               # the same merged model whatever the order was
    rift.rift_gmm_destroy(h2)
    rift.rift_gmm_destroy(g)


MODELS = {
    "2d": (np.array([[0.2, 0.1], [1.2, 0.9], [-0.3, 1.0]]),
           np.array([[[0.5, 0.35], [0.35, 0.4]], [[0.2, -0.1], [-0.1, 0.3]], [[0.05, 0.0], [0.0, 0.6]]]),
           np.array([0.5, 0.3, 0.2]), np.array([-0.5, -0.6]), np.array([1.6, 1.4])),
    "2d_tight": (np.array([[0.0, 0.0], [0.5, 0.45]]),
                 np.array([[[1.0, 0.99 * 0.5], [0.99 * 0.5, 0.25]], [[0.01, 0.0], [0.0, 0.01]]]),
                 np.array([0.7, 0.3]), np.array([-1.0, -1.0]), np.array([1.0, 1.0])),
    "1d": (np.array([[0.5], [2.5]]), np.array([[[0.64]], [[0.09]]]), np.array([0.7, 0.3]), np.array([0.0]), np.array([3.0])),
}


@pytest.mark.parametrize("name", list(MODELS))
def test_masses_density_and_draws_match_oracle(torch, name):
    mu, cov, pi, lo, hi = MODELS[name]
    K, d = mu.shape
    g = rift.rift_gmm_create(d, K, lo, hi)
    rift.rift_gmm_set_model(g, mu, cov, pi)
    Z = rift.rift_gmm_box_mass(g)
    Z_o = np.array([go.box_mass(mu[k], cov[k], lo, hi) for k in range(K)])
    assert np.max(np.abs(Z - Z_o) / Z_o) < 1e-9
    # draws: same counters, same component, same proposal -> the same points up to the inverse normal CDF's rounding
    n, seed, off = 3000, 12345, 1_000_000_007
    xs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(d)]
    lnp = torch.empty(n, dtype=torch.float64, device="cuda")
    failed = rift.rift_gmm_draw(g, n, seed, off, xs, lnp, want_failed=True)
    torch.cuda.synchronize()
    x = np.stack([v.cpu().numpy() for v in xs], axis=1)
    x_o, failed_o = go.draw(n, seed, off, mu, cov, pi, lo, hi)
    assert failed == failed_o == 0
    assert np.all((x >= lo) & (x < hi))
    diff = np.max(np.abs(x - x_o), axis=1)
    assert np.mean(diff < TOL_DRAW) > 0.999          # an acceptance within rounding of the domain's edge may differ: none expected
    assert np.max(diff) < TOL_DRAW
    lnp_o = go.ln_density(x_o, mu, cov, pi, lo, hi)
    assert np.max(np.abs(lnp.cpu().numpy() - lnp_o)) < TOL_LNP
    # the density entry point, inside and outside the domain
    rng = np.random.default_rng(1)
    pts = rng.uniform(lo - 0.3, hi + 0.3, size=(5000, d))
    out = torch.empty(5000, dtype=torch.float64, device="cuda")
    rift.rift_gmm_ln_density(g, 5000, [_dev(torch, pts[:, j]) for j in range(d)], out)
    torch.cuda.synchronize()
    ref = go.ln_density(pts, mu, cov, pi, lo, hi)
    got = out.cpu().numpy()
    assert np.array_equal(np.isneginf(got), np.isneginf(ref)) and np.any(np.isneginf(ref))
    fin = np.isfinite(ref)
    assert np.max(np.abs(got[fin] - ref[fin])) < TOL_LNP
    # a second call continues the stream
    xs2 = [torch.empty(100, dtype=torch.float64, device="cuda") for _ in range(d)]
    rift.rift_gmm_draw(g, 100, seed, off + 2900, xs2)
    torch.cuda.synchronize()
    assert np.array_equal(np.stack([v.cpu().numpy() for v in xs2], axis=1), x[2900:])
    rift.rift_gmm_destroy(g)


def test_adaptive_loop_integrates_a_correlated_gaussian(torch):
    """The paper's integrator test in miniature (Fig. 6, :332): a narrow, strongly correlated Gaussian 'likelihood' in a wide
    box.  Draw from p_s, weight by L / p_s, refit (merged online), repeat: the evidence estimate converges to the closed form
    (the Gaussian's mass inside the box) and the effective sample size grows far beyond that of the uniform start."""
    lo, hi = np.array([-10.0, -10.0]), np.array([10.0, 10.0])
    m_true, c_true = np.array([1.0, -2.0]), np.array([[0.04, 0.054], [0.054, 0.09]])          # correlation 0.9
    exact = go.box_mass(m_true, c_true, lo, hi)
    g = rift.rift_gmm_create(2, 2, lo, hi)
    n = 200_000
    xs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    lnp = torch.empty(n, dtype=torch.float64, device="cuda")
    prec = torch.from_numpy(np.linalg.inv(c_true)).cuda()
    ln_norm = -0.5 * math.log(np.linalg.det(c_true)) - math.log(2 * math.pi)
    ess = []
    for it in range(6):
        rift.rift_gmm_draw(g, n, 99, it * n, xs, lnp)
        d0, d1 = xs[0] - m_true[0], xs[1] - m_true[1]
        lnL = ln_norm - 0.5 * (prec[0, 0] * d0 * d0 + 2 * prec[0, 1] * d0 * d1 + prec[1, 1] * d1 * d1)
        lnw = lnL - lnp
        w = torch.exp(lnw - lnw.max())
        ess.append(float(w.sum() ** 2 / (w * w).sum()))
        est = float(torch.exp(lnw).mean())
        rift.rift_gmm_fit(g, n, xs, lnw, 20, 1e-8, 1e-9, merge=1 if it > 0 else 0)
    assert ess[0] < 0.01 * n and ess[-1] > 0.5 * n, ess
    assert abs(est - exact) < 5e-3 * exact, (est, exact)
    rift.rift_gmm_destroy(g)


def test_gmm_loop_on_the_ile_likelihood_matches_prior_sampling(torch, oracle):
    """The configuration the paper recommends for loud signals (:807), end to end on the hot path: GMM sampling in the rotated
    network-frame sky with distance marginalisation (gmm_loop.integrate) gives the same evidence as plain prior sampling of the
    same distance-marginalised likelihood, with a far larger effective sample size per evaluation."""
    from paper_2210_07912_b200 import gmm_loop, synth
    from helpers import build, create
    cfg = synth.with_overrides(synth.CONFIGS[0], n_points=1, rho=9.0)
    inp = build(oracle, cfg, n_points=1)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    s = torch.cuda.current_stream().cuda_stream
    d_min, d_max, n_dist = synth.D_MIN_MPC, synth.D_MAX_MPC, 128
    # reference: 4e6 prior draws of the five parameters, pooled
    n_ref, ref = 1_000_000, None
    for r in range(4):
        params, _ = synth.draw_samples(cfg, 800 + r, n_ref)
        p = torch.from_numpy(np.ascontiguousarray(params[:5])).cuda()
        lnL = torch.empty(n_ref, dtype=torch.float64, device="cuda")
        rift.rift_ile_eval_batch_dmarg(h, [0], n_ref, p, d_min, d_max, n_dist, lnL, None, s)
        ref = rift.rift_ile_reduce(h, 1, n_ref, lnL, None, merge=1 if r else 0, cuda_stream=s)
    R = rift.rift_sky_network_frame(inp.det_location[0], inp.det_location[1])
    samplers = gmm_loop.create_samplers(n_comp_sky=3, n_comp_1d=1)
    res = gmm_loop.integrate(h, samplers, 0, R, cfg.gmst, d_min, d_max, n_dist, 200_000, n_eff_target=1e9, max_rounds=8,
                             seed=5, cuda_stream=s)
    gmm_loop.destroy_samplers(samplers)
    rift.rift_ile_destroy(h)
    assert res["rounds"] == 8 and res["n_evals"] == 1_600_000
    sigma = math.hypot(res["rel_err"], float(ref["rel_err"][0]))
    assert abs(res["lnZ"] - float(ref["lnZ"][0])) < 4.0 * sigma + 0.02, (res, ref)
    # efficiency: effective samples per evaluation at least 5x those of prior sampling
    assert res["n_ess"] / res["n_evals"] > 5.0 * float(ref["n_ess"][0]) / (4 * n_ref), (res, ref)


def test_rosenbrock_evidence_of_fig7_with_the_gmm_integrator(torch, oracle):
    """Fig. 7 (:356) with the GMM integrator: the evidence of the two-dimensional Rosenbrock likelihood, -5.804
    (tests/golden/fig7_rosenbrock.txt), from 1e6 evaluations in batches of 1e4 -- a curved, strongly correlated ridge, which a
    correlated mixture follows where a separable sampler cannot.  Draws, densities, EM refits (merged online) and the pooled
    evidence (Eq. (20)-(21)) come from the library; only the integrand is the test's."""
    import os
    from paper_2210_07912_b200 import synth
    from helpers import build, create
    path = os.path.join(os.path.dirname(__file__), "golden", "fig7_rosenbrock.txt")
    gold = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")][0]
    ln_z, n_total, n = float(gold[0]), int(gold[1]), int(gold[2])
    inp = build(oracle, synth.CONFIGS[0])
    h = create(rift, inp, rift.RIFT_PREC_MIXED)                             # only its reduce is used
    stream = torch.cuda.current_stream().cuda_stream
    L = 5.0
    g = rift.rift_gmm_create(2, 6, [-L, -L], [L, L])
    xs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    lps = torch.empty(n, dtype=torch.float64, device="cuda")
    lom = torch.empty(n, dtype=torch.float64, device="cuda")
    pooled = None
    for it in range(n_total // n):
        rift.rift_gmm_draw(g, n, 78, it * n, xs, lps, cuda_stream=stream)
        lnL = -((1.0 - xs[0]) ** 2 + 100.0 * (xs[1] - xs[0] * xs[0]) ** 2)
        lw = -math.log((2 * L) ** 2) - lps
        pooled = rift.rift_ile_reduce(h, 1, n, lnL, lw, cuda_stream=stream, merge=0 if it == 0 else 1)
        rift.rift_gmm_add(n, [lnL, lw], lom, stream)
        rift.rift_gmm_fit_tempered(g, n, xs, lom, 300.0, 10, 1e-6, 1e-6, merge=1 if it > 0 else 0, cuda_stream=stream)
    rel = float(pooled["rel_err"][0])
    assert rel < 0.03, pooled
    assert abs(float(pooled["lnZ"][0]) - ln_z) < 4 * rel + 5e-4, pooled    # the paper prints three decimals
    # the correlated mixture follows the curved ridge: two orders of magnitude more effective samples than the separable
    # histogram sampler of NEXT-1 reaches on the same budget (golden file: the paper's n_ESS ~ 1400 for AC; observed 4.4e5)
    assert pooled["n_ess"][0] > 100.0 * float(gold[3]), (pooled, gold)
    rift.rift_gmm_destroy(g)
    rift.rift_ile_destroy(h)


def test_fig6_correlated_three_dimensional_gaussian_with_pairwise_groups(torch, oracle):
    """Fig. 6 (:332): weighted samples of a correlated three-dimensional Gaussian likelihood after a fixed number of evaluations;
    the one-dimensional cumulative distributions they imply are compared with the true ones.  The sampler is a product of a
    correlated pair (x0, x1) and a single dimension x2 (the pairwise-correlated form: the x2 correlations are left to the
    weights), refitted every round with the online merge."""
    from scipy import stats
    from paper_2210_07912_b200 import synth
    from helpers import build, create
    inp = build(oracle, synth.CONFIGS[0])
    h = create(rift, inp, rift.RIFT_PREC_MIXED)                             # only its reduce is used
    stream = torch.cuda.current_stream().cuda_stream
    L, n, rounds = 6.0, 20_000, 20
    mu = np.array([0.5, -1.0, 1.5])
    sd = np.array([0.4, 0.7, 0.5])
    corr = np.array([[1.0, 0.85, 0.3], [0.85, 1.0, 0.2], [0.3, 0.2, 1.0]])
    cov = corr * np.outer(sd, sd)
    prec = torch.from_numpy(np.linalg.inv(cov)).cuda()
    ln_norm = -0.5 * math.log(np.linalg.det(cov)) - 1.5 * math.log(2 * math.pi)
    g01 = rift.rift_gmm_create(2, 2, [-L, -L], [L, L])
    g2 = rift.rift_gmm_create(1, 1, [-L], [L])
    x = torch.empty((3, n), dtype=torch.float64, device="cuda")
    lp = torch.empty((2, n), dtype=torch.float64, device="cuda")
    lom = torch.empty(n, dtype=torch.float64, device="cuda")
    keep_x, keep_w = [], []
    pooled = None
    for it in range(rounds):
        rift.rift_gmm_draw(g01, n, 31, it * n, [x[0], x[1]], lp[0], cuda_stream=stream)
        rift.rift_gmm_draw(g2, n, 32, it * n, [x[2]], lp[1], cuda_stream=stream)
        d = x - torch.from_numpy(mu).cuda()[:, None]
        lnL = ln_norm - 0.5 * torch.einsum("in,ij,jn->n", d, prec, d)
        lw = -3.0 * math.log(2 * L) - lp[0] - lp[1]
        pooled = rift.rift_ile_reduce(h, 1, n, lnL, lw, cuda_stream=stream, merge=0 if it == 0 else 1)
        rift.rift_gmm_add(n, [lnL, lw], lom, stream)
        for g, rows in ((g01, [x[0], x[1]]), (g2, [x[2]])):
            rift.rift_gmm_fit_tempered(g, n, rows, lom, 300.0, 10, 1e-6, 1e-6, merge=1 if it > 0 else 0, cuda_stream=stream)
        if it >= rounds // 2:                                                # the adapted half of the run, as the figure's samples
            keep_x.append(x.cpu().numpy().copy())
            keep_w.append(np.exp((lnL + lw).cpu().numpy()))
    # evidence: the Gaussian's mass in the box (1 to 1e-12) over the prior volume
    rel = float(pooled["rel_err"][0])
    assert rel < 0.01 and abs(float(pooled["lnZ"][0]) + 3.0 * math.log(2 * L)) < 4 * rel + 1e-3, pooled
    assert pooled["n_ess"][0] > 0.03 * rounds * n, pooled      # pooled over ALL rounds: the wide first rounds weigh it down
    # one-dimensional weighted CDFs against the true marginals
    X, W = np.concatenate(keep_x, axis=1), np.concatenate(keep_w)
    for dim in range(3):
        order = np.argsort(X[dim])
        cdf = np.cumsum(W[order]) / W.sum()
        true = stats.norm.cdf(X[dim][order], mu[dim], sd[dim])
        assert np.max(np.abs(cdf - true)) < 0.01, (dim, np.max(np.abs(cdf - true)))
    # the pair's mixture has found the correlation
    m, c, p, _ = rift.rift_gmm_get_model(g01)
    mix_cov = sum(p[k] * (c[k] + np.outer(m[k], m[k])) for k in range(2)) - np.outer(p @ m, p @ m)
    assert abs(mix_cov[0, 1] / np.sqrt(mix_cov[0, 0] * mix_cov[1, 1]) - 0.85) < 0.05
    rift.rift_gmm_destroy(g01)
    rift.rift_gmm_destroy(g2)
    rift.rift_ile_destroy(h)
