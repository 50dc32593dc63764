"""Pins of oracle/gmm_oracle.py (section IV.C.1 :315-334 and Appendix A :562-625)
against closed forms, library routines the oracle does not call (numpy.cov, sklearn's EM, scipy's truncnorm and multivariate
normal CDF) and invariants -- no GPU, no product code."""
import warnings

import numpy as np
import pytest
from scipy import stats

from oracle import gmm_oracle as go


def _mix(rng, n, mus, covs, pis):
    k = rng.choice(len(pis), size=n, p=pis)
    return np.stack([rng.multivariate_normal(mus[j], covs[j]) for j in k])


def test_p32_single_component_m_step_is_the_weighted_sample_moments():
    rng = np.random.default_rng(1)
    for d in (1, 2):
        x = rng.normal(size=(500, d)) * 1.7 + 3.0
        ln_w = rng.normal(size=500)
        w = go.normalise_ln_weights(ln_w)
        assert abs(w.sum() - 1.0) < 1e-15
        r, _ll = go.e_step(x, w, np.zeros((1, d)), np.eye(d)[None], np.ones(1))
        assert np.allclose(r, 1.0)
        mu, cov, pi = go.m_step(x, w, r)
        assert np.allclose(mu[0], np.average(x, axis=0, weights=w), rtol=1e-13)
        assert np.allclose(cov[0], np.atleast_2d(np.cov(x.T, aweights=w, bias=True)), rtol=1e-12)
        assert abs(pi[0] - 1.0) < 1e-15
    # ln N against scipy
    x = rng.normal(size=(20, 2))
    c = np.array([[2.0, 0.6], [0.6, 0.5]])
    assert np.allclose(go.ln_normal(x, [0.3, -1.0], c), stats.multivariate_normal([0.3, -1.0], c).logpdf(x), rtol=1e-12)


@pytest.mark.parametrize("d", [1, 2])
def test_p33_em_matches_sklearn_iteration_by_iteration(d):
    """Equal weights: Eq. (A3)-(A6) are the textbook EM, which sklearn implements (the oracle never calls it)."""
    from sklearn.mixture import GaussianMixture
    rng = np.random.default_rng(2)
    mus = [np.full(d, -2.0), np.full(d, 2.5), np.array([0.0] * d)]
    covs = [np.eye(d) * 0.5, np.eye(d) * 1.5, np.eye(d) * 0.2]
    x = _mix(rng, 1500, mus, covs, [0.5, 0.3, 0.2])
    mu0 = np.array([m + 0.5 for m in mus])
    cov0 = np.array([np.eye(d)] * 3)
    pi0 = np.array([0.4, 0.4, 0.2])
    for iters in (1, 3, 7):
        with warnings.catch_warnings():
            warnings.simplefilter("ignore")
            gm = GaussianMixture(3, covariance_type="full", tol=0.0, reg_covar=1e-6, max_iter=iters, means_init=mu0,
                                 weights_init=pi0, precisions_init=np.array([np.linalg.inv(c) for c in cov0])).fit(x)
        mu, cov, pi, it, _ll = go.fit(x, np.zeros(len(x)), mu0, cov0, pi0, iters, 0.0, 1e-6)
        assert it == iters
        assert np.allclose(mu, gm.means_, rtol=1e-9, atol=1e-11) and np.allclose(cov, gm.covariances_, rtol=1e-9, atol=1e-11)
        assert np.allclose(pi, gm.weights_, rtol=1e-9)


def test_p34_weights_act_as_multiplicities_and_loglik_never_decreases():
    rng = np.random.default_rng(3)
    x = _mix(rng, 300, [np.array([-1.0, 0.0]), np.array([2.0, 1.0])], [np.eye(2) * 0.3, np.array([[1.0, 0.7], [0.7, 1.0]])], [0.6, 0.4])
    mult = rng.integers(1, 4, size=300)
    mu0, cov0, pi0 = np.array([[-0.5, 0.2], [1.0, 0.5]]), np.array([np.eye(2)] * 2), np.array([0.5, 0.5])
    a = go.fit(x, np.log(mult.astype(float)), mu0, cov0, pi0, 6)
    b = go.fit(np.repeat(x, mult, axis=0), np.zeros(int(mult.sum())), mu0, cov0, pi0, 6)
    for u, v in zip(a[:3], b[:3]):
        assert np.allclose(u, v, rtol=1e-10, atol=1e-12)
    # a common factor on the weights changes nothing
    c = go.fit(x, np.log(mult.astype(float)) + 123.0, mu0, cov0, pi0, 6)
    for u, v in zip(a[:3], c[:3]):
        assert np.allclose(u, v, rtol=1e-12, atol=1e-14)
    lls = [go.fit(x, np.log(mult.astype(float)), mu0, cov0, pi0, k)[4] for k in range(1, 12)]
    assert all(l2 >= l1 - 1e-12 for l1, l2 in zip(lls, lls[1:]))
    # the tolerance stops the iteration early
    it = go.fit(x, np.zeros(300), mu0, cov0, pi0, 500, tol=1e-6)[3]
    assert 2 <= it < 500


def test_p35_merge_of_exact_moments_is_the_pooled_moments_and_matching_undoes_a_permutation():
    rng = np.random.default_rng(4)
    xa, xb = rng.normal(size=(400, 2)) @ np.array([[1.0, 0.4], [0.0, 0.7]]) + 1.0, rng.normal(size=(250, 2)) * 0.5 - 0.3
    mom = lambda x: (x.mean(axis=0)[None], np.cov(x.T, bias=True)[None], np.ones(1))
    mu, cov, pi = go.merge(*mom(xa), 400, *mom(xb), 250)
    allx = np.concatenate([xa, xb])
    assert np.allclose(mu[0], allx.mean(axis=0), rtol=1e-13) and np.allclose(cov[0], np.cov(allx.T, bias=True), rtol=1e-12)
    assert abs(pi[0] - 1.0) < 1e-15
    # three components, the new model a slightly moved, permuted copy of the old one
    mu_o = np.array([[0.0, 0.0], [3.0, 1.0], [-2.0, 2.0]])
    cov_o = np.array([np.eye(2), np.array([[1.0, 0.5], [0.5, 2.0]]), np.eye(2) * 0.3])
    pi_o = np.array([0.5, 0.3, 0.2])
    for perm in ([2, 0, 1], [1, 2, 0], [0, 1, 2]):
        mu_n, cov_n, pi_n = mu_o[perm] + 0.05, cov_o[perm] * 1.1, pi_o[perm]
        assert go.match_components(mu_o, cov_o, mu_n, cov_n) == perm
        m, c, p = go.merge(mu_o, cov_o, pi_o, 1000, mu_n, cov_n, pi_n, 1000)
        assert np.allclose(m, mu_o + 0.025) and np.allclose(p, pi_o) and abs(p.sum() - 1) < 1e-15


def test_p36_transform_and_proposal_box():
    rng = np.random.default_rng(5)
    for _ in range(20):
        b = rng.normal(size=(2, 2))
        cov = b @ b.T + 0.1 * np.eye(2)
        A = go.transform(cov)
        assert np.allclose(A @ A.T, cov, rtol=1e-12)
        lam = np.sum(A * A, axis=0)
        assert lam[0] <= lam[1] and abs(A[:, 0] @ A[:, 1]) < 1e-12 * lam[1]
        for j in range(2):
            assert A[np.argmax(np.abs(A[:, j])), j] > 0
        mu, lo, hi = rng.normal(size=2), np.array([-1.0, -2.0]), np.array([1.5, 0.5])
        zl, zh = go.z_box(mu, A, lo, hi)
        pts = rng.uniform(lo, hi, size=(200, 2))
        z = (pts - mu) @ np.linalg.inv(A).T
        assert np.all(z >= zl - 1e-12) and np.all(z <= zh + 1e-12)          # the proposal box contains the whole domain
    assert np.allclose(go.transform(np.array([[4.0]])), [[2.0]])
    assert np.allclose(go.transform(np.diag([4.0, 1.0])), [[0.0, 2.0], [1.0, 0.0]])  # ascending eigenvalues, positive signs


def test_p37_box_mass():
    lo, hi = np.array([-1.0, -0.5]), np.array([2.0, 1.5])
    # independent dimensions: a product of one-dimensional masses
    z = go.box_mass([0.2, 0.1], np.diag([1.0, 0.25]), lo, hi)
    z1 = go.box_mass([0.2], [[1.0]], lo[:1], hi[:1]) * go.box_mass([0.1], [[0.25]], lo[1:], hi[1:])
    assert abs(z - z1) < 1e-13
    assert abs(go.box_mass([0.0, 0.0], [[1.0, 0.9], [0.9, 1.0]], [-50, -50], [50, 50]) - 1.0) < 1e-12
    assert abs(go.box_mass([0.0, 0.0], [[1.0, 0.9], [0.9, 1.0]], [0, -50], [50, 50]) - 0.5) < 1e-12
    assert abs(go.box_mass([0.0, 0.0], [[1.0, 0.5], [0.5, 1.0]], [0, 0], [60, 60]) - (0.25 + np.arcsin(0.5) / (2 * np.pi))) < 1e-12
    # scipy's multivariate normal CDF (Genz), by inclusion-exclusion
    rng = np.random.default_rng(6)
    for rho in (0.3, -0.8, 0.99):
        cov = np.array([[1.3, rho * np.sqrt(1.3 * 0.6)], [rho * np.sqrt(1.3 * 0.6), 0.6]])
        mu = rng.normal(size=2) * 0.5
        mvn = stats.multivariate_normal(mu, cov)
        F = lambda a, b: mvn.cdf([a, b])
        ref = F(hi[0], hi[1]) - F(lo[0], hi[1]) - F(hi[0], lo[1]) + F(lo[0], lo[1])
        assert abs(go.box_mass(mu, cov, lo, hi) - ref) < 2e-6


def test_p38_draws_follow_the_truncated_mixture():
    # one dimension: the draws are exactly scipy's truncated normal (Kolmogorov-Smirnov on the mixture CDF)
    mu, cov, pi = np.array([[0.5], [2.5]]), np.array([[[0.64]], [[0.09]]]), np.array([0.7, 0.3])
    lo, hi = np.array([0.0]), np.array([3.0])
    x, failed = go.draw(4000, 9, 0, mu, cov, pi, lo, hi)
    assert failed == 0 and np.all((x >= lo) & (x < hi))
    cdf = lambda t: sum(pi[k] * stats.truncnorm.cdf(t, (lo[0] - mu[k, 0]) / np.sqrt(cov[k, 0, 0]), (hi[0] - mu[k, 0]) / np.sqrt(cov[k, 0, 0]),
                                                     loc=mu[k, 0], scale=np.sqrt(cov[k, 0, 0])) for k in range(2))
    assert stats.kstest(x[:, 0], cdf).pvalue > 1e-3
    # a later call continues the same stream
    x2, _ = go.draw(100, 9, 3900, mu, cov, pi, lo, hi)
    assert np.array_equal(x2, x[3900:])
    # the density is normalised on the domain and matches the truncated mixture
    t = np.linspace(0, 3, 30001)[:-1] + 0.5e-4
    p = np.exp(go.ln_density(t[:, None], mu, cov, pi, lo, hi))
    assert abs(p.sum() * 1e-4 - 1.0) < 1e-7
    ref = sum(pi[k] * stats.truncnorm.pdf(t, (lo[0] - mu[k, 0]) / np.sqrt(cov[k, 0, 0]), (hi[0] - mu[k, 0]) / np.sqrt(cov[k, 0, 0]),
                                          loc=mu[k, 0], scale=np.sqrt(cov[k, 0, 0])) for k in range(2))
    assert np.max(np.abs(p - ref)) < 1e-12
    assert np.all(np.isneginf(go.ln_density(np.array([[-0.1], [3.0]]), mu, cov, pi, lo, hi)))


def test_p39_two_dimensional_draws_and_importance_identity():
    """Correlated pair in a box that cuts the Gaussians: draws stay inside, p_s integrates to 1 on the domain, and
    E_{p_s}[f / p_s] = integral of f (the identity Eq. (3) rests on) for f = a correlated Gaussian 'likelihood'."""
    mu = np.array([[0.2, 0.1], [1.2, 0.9]])
    cov = np.array([[[0.5, 0.35], [0.35, 0.4]], [[0.2, -0.1], [-0.1, 0.3]]])
    pi = np.array([0.6, 0.4])
    lo, hi = np.array([-0.5, -0.6]), np.array([1.6, 1.4])
    x, failed = go.draw(6000, 21, 0, mu, cov, pi, lo, hi)
    assert failed == 0 and np.all((x >= lo) & (x < hi))
    g1, g2 = np.meshgrid(lo[0] + (np.arange(420) + 0.5) * 0.005, lo[1] + (np.arange(400) + 0.5) * 0.005, indexing="ij")
    grid = np.stack([g1.ravel(), g2.ravel()], axis=1)
    p = np.exp(go.ln_density(grid, mu, cov, pi, lo, hi))
    assert abs(p.sum() * 0.005 ** 2 - 1.0) < 2e-4                           # midpoint rule; the box edges cut the density
    f = stats.multivariate_normal([0.5, 0.4], [[0.3, 0.2], [0.2, 0.25]])
    exact = go.box_mass([0.5, 0.4], [[0.3, 0.2], [0.2, 0.25]], lo, hi)
    wts = f.pdf(x) / np.exp(go.ln_density(x, mu, cov, pi, lo, hi))
    est, err = wts.mean(), wts.std() / np.sqrt(len(wts))
    assert abs(est - exact) < 5 * err and err < 0.02 * exact
    # sample moments of the draws against moments of p_s on the grid
    m_grid = (p[:, None] * grid).sum(axis=0) * 0.005 ** 2
    assert np.max(np.abs(x.mean(axis=0) - m_grid)) < 5 * np.max(x.std(axis=0)) / np.sqrt(len(x))


def test_p40_tempering_reaches_the_requested_effective_sample_size():
    rng = np.random.default_rng(9)
    ln_w = rng.normal(0.0, 6.0, 20000)                 # a few samples carry all the weight
    assert go.tempered_ess(ln_w, 1.0) < 50 and abs(go.tempered_ess(ln_w, 0.0) - 20000) < 1e-6
    ess = [go.tempered_ess(ln_w, b) for b in np.linspace(0, 1, 21)]
    assert all(a >= b for a, b in zip(ess, ess[1:]))   # monotone: the bisection is well defined
    for target in (100.0, 1000.0, 15000.0):
        b = go.temper_for_ess(ln_w, target)
        assert 0.0 < b < 1.0 and go.tempered_ess(ln_w, b) >= target > go.tempered_ess(ln_w, b + 2.0 ** -19)
    assert go.temper_for_ess(ln_w, 1.0) == 1.0 and go.temper_for_ess(ln_w, 0.0) == 1.0
    assert go.temper_for_ess(ln_w, 1e9) == 0.0         # unreachable: all weights equal
    # the equal-weight closed form: ESS of N(0, s^2) log-weights tempered by b is about n exp(-(b s)^2)
    b = go.temper_for_ess(ln_w, 20000 * np.exp(-1.0))
    assert abs(b * 6.0 - 1.0) < 0.05
