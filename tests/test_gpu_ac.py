"""GPU tests of the on-device adaptive-cartesian sampler (include/rift_ac.h; section IV.C.2, :336-358):
element-wise parity of the draw, the histogram refresh and the ILE prior weights with oracle/ac_oracle.py, and the closed
loop draw -> rift_ile_eval_batch -> rift_ile_reduce -> update on a synthetic intrinsic point."""
import math

import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from paper_2210_07912_b200 import synth
from oracle import ac_oracle as ac

from helpers import build, create

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def test_draw_update_and_weights_match_the_oracle(torch):
    rng = np.random.default_rng(4)
    n_dim, n_bins, n = 6, 100, 10_007
    lo, hi = synth.HIST_LO, synth.HIST_HI
    h = rift.rift_ac_create(n_dim, n_bins, lo, hi)
    x = torch.zeros((n_dim, n), dtype=torch.float64, device="cuda")
    lps = torch.zeros(n, dtype=torch.float64, device="cuda")
    masses = ac.uniform_masses(n_dim, n_bins)
    for rnd, (floor, temper) in enumerate([(None, None), (0.1, 1.0), (0.02, 0.5)]):
        if floor is not None:
            hist = rng.random((n_dim, n_bins)) ** 4
            hist[2, 30:60] = 0.0
            hist /= hist.sum(axis=1, keepdims=True)
            rift.rift_ac_update(h, hist, floor, temper)
            masses = ac.update(hist, floor, temper)
            assert np.max(np.abs(rift.rift_ac_get_masses(h, n_dim, n_bins) - masses)) < 1e-15
        rift.rift_ac_draw(h, n, seed=77, offset=1000 * rnd, x=x, ln_ps=lps)
        torch.cuda.synchronize()
        xo, lpo, bo = ac.draw(masses, lo, hi, n, seed=77, offset=1000 * rnd)
        xg = x.cpu().numpy()
        w = (hi - lo) / n_bins
        bg = np.floor((xg - lo[:, None]) / w[:, None]).astype(np.int32)
        assert np.mean(bg == bo) > 0.9999                                   # the same bins (up to samples on a bin edge)
        assert np.max(np.abs(xg - xo) / (hi - lo)[:, None]) < 1e-14
        assert np.max(np.abs(lps.cpu().numpy() - lpo)) < 1e-12
        # ILE prior weights
        lw = torch.zeros(n, dtype=torch.float64, device="cuda")
        rift.rift_ac_ile_ln_weight(n, x, synth.D_MIN_MPC, synth.D_MAX_MPC, lps, lw)
        torch.cuda.synchronize()
        ref = ac.ln_prior_ile(xo, synth.D_MIN_MPC, synth.D_MAX_MPC) - lpo
        got = lw.cpu().numpy()
        fin = np.isfinite(ref)
        assert np.array_equal(np.isfinite(got), fin)
        assert np.max(np.abs(got[fin] - ref[fin])) < 1e-11
    rift.rift_ac_destroy(h)
    with pytest.raises(rift.RiftError):
        rift.rift_ac_create(3, 100, [0, 0, 0], [1, 0, 1])                     # hi <= lo


def test_closed_loop_on_a_synthetic_point(torch, oracle):
    """Adapted sampling of one intrinsic point (C0 recipe at rho = 6): the sample-size measures n_eff, n_ESS (Eq. (B1)-(B2),
    :637-641) rise several-fold over prior sampling at equal cost, and the pooled evidence (Eq. (3), (20)-(21)) agrees with a large
    prior-sampled run within the Monte Carlo errors both report (Eq. (B3))."""
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=6.0)
    inp = build(oracle, cfg)
    h = create(rift, inp, rift.RIFT_PREC_MIXED)
    stream = torch.cuda.current_stream().cuda_stream
    lo, hi, nb = synth.HIST_LO, synth.HIST_HI, 100

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a)).cuda()

    # reference: 2e6 prior draws
    n_ref = 2_000_000
    p_ref = dev(synth.prior_draw(np.random.default_rng(123), n_ref))
    lnL = torch.empty(n_ref, dtype=torch.float64, device="cuda")
    rift.rift_ile_eval_batch(h, [0], n_ref, p_ref, lnL, None, stream)
    ref = rift.rift_ile_reduce(h, 1, n_ref, lnL, None, cuda_stream=stream)
    assert ref["n_eff"][0] > 20, ref

    n = 100_000
    s = rift.rift_ac_create(6, nb, lo, hi)
    x = torch.empty((6, n), dtype=torch.float64, device="cuda")
    lps = torch.empty(n, dtype=torch.float64, device="cuda")
    lw = torch.empty(n, dtype=torch.float64, device="cuda")
    lnL = torch.empty(n, dtype=torch.float64, device="cuda")
    neff, rounds = [], 10
    for it in range(rounds):
        rift.rift_ac_draw(s, n, seed=2210, offset=it * n, x=x, ln_ps=lps, cuda_stream=stream)
        rift.rift_ac_ile_ln_weight(n, x, synth.D_MIN_MPC, synth.D_MAX_MPC, lps, lw, stream)
        rift.rift_ile_eval_batch(h, [0], n, x, lnL, None, stream)
        one = rift.rift_ile_reduce(h, 1, n, lnL, lw, x, lo, hi, nb, merge=0, want_hist=True, cuda_stream=stream)
        neff.append(float(one["n_eff"][0]))
        rift.rift_ac_update(s, one["hist"][0], 0.1, 0.75)
    # pooled evidence with the adapted sampler frozen: five fresh rounds merged by rift_ile_reduce (Eq. (20)-(21))
    first = True
    for it in range(rounds, rounds + 5):
        rift.rift_ac_draw(s, n, seed=2210, offset=it * n, x=x, ln_ps=lps, cuda_stream=stream)
        rift.rift_ac_ile_ln_weight(n, x, synth.D_MIN_MPC, synth.D_MAX_MPC, lps, lw, stream)
        rift.rift_ile_eval_batch(h, [0], n, x, lnL, None, stream)
        pooled = rift.rift_ile_reduce(h, 1, n, lnL, lw, cuda_stream=stream, merge=0 if first else 1)
        first = False
    cost = (5 * n) / n_ref                                                 # prior-sampled sizes scaled to equal cost
    assert neff[-1] > 5 * neff[0], neff                                    # separable histograms: 27 -> ~250 here
    assert pooled["n_eff"][0] > 2 * ref["n_eff"][0] * cost, (pooled, ref)   # n_eff (B1) hinges on the single largest weight
    assert pooled["n_ess"][0] > 5 * ref["n_ess"][0] * cost, (pooled, ref)   # n_ESS (B2): 5.5e3 against 3.6e2 here
    sigma = math.hypot(pooled["rel_err"][0], ref["rel_err"][0])
    assert abs(pooled["lnZ"][0] - ref["lnZ"][0]) < 5 * sigma + 0.02, (pooled, ref, sigma)
    rift.rift_ac_destroy(s)
    rift.rift_ile_destroy(h)


def test_rosenbrock_evidence_of_fig7_on_device(torch, oracle):
    """Fig. 7 (:356): the AC integrator recovers the evidence of the two-dimensional Rosenbrock likelihood, -5.804
    (tests/golden/fig7_rosenbrock.txt, reading C3), from 1e6 evaluations in batches of 1e4.  The draws, their densities,
    the weighted histograms and the pooled evidence (Eq. (20)-(21)) all come from the library; only the integrand is the
    test's."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "fig7_rosenbrock.txt")
    gold = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")][0]
    ln_z, n_total, n = float(gold[0]), int(gold[1]), int(gold[2])
    inp = build(oracle, synth.CONFIGS[0])
    h_round, h_pool = create(rift, inp, rift.RIFT_PREC_MIXED), create(rift, inp, rift.RIFT_PREC_MIXED)
    stream = torch.cuda.current_stream().cuda_stream
    L, nb = 5.0, 100
    s = rift.rift_ac_create(2, nb, [-L, -L], [L, L])
    x = torch.empty((2, n), dtype=torch.float64, device="cuda")
    lps = torch.empty(n, dtype=torch.float64, device="cuda")
    six = [x[0], x[1], x[0], x[0], x[0], x[0]]                             # reduce histograms six rows; the first two are ours
    lo6, hi6 = [-L] * 6, [L] * 6
    for it in range(n_total // n):
        rift.rift_ac_draw(s, n, seed=78, offset=it * n, x=x, ln_ps=lps, cuda_stream=stream)
        lnL = -((1.0 - x[0]) ** 2 + 100.0 * (x[1] - x[0] * x[0]) ** 2)
        lw = -math.log((2 * L) ** 2) - lps
        one = rift.rift_ile_reduce(h_round, 1, n, lnL, lw, six, lo6, hi6, nb, merge=0, want_hist=True, cuda_stream=stream)
        pooled = rift.rift_ile_reduce(h_pool, 1, n, lnL, lw, cuda_stream=stream, merge=0 if it == 0 else 1)
        rift.rift_ac_update(s, one["hist"][0][:2], 0.1, 0.75)
    rel = float(pooled["rel_err"][0])
    assert rel < 0.03, pooled
    assert abs(float(pooled["lnZ"][0]) - ln_z) < 4 * rel + 5e-4, pooled    # the paper prints three decimals
    assert pooled["n_ess"][0] > 0.5 * float(gold[3]) and pooled["n_eff"][0] > 0.4 * float(gold[4]), pooled
    rift.rift_ac_destroy(s)
    rift.rift_ile_destroy(h_round)
    rift.rift_ile_destroy(h_pool)


def test_round_loop_sky_only_to_n_eff_target_then_frozen(torch, oracle):
    """The production settings of :452 through paper_2210_07912_b200.ac_loop: rounds until the pooled n_eff reaches 10, only
    the sky adapted (rift_ac_update_dims), then the same sampler frozen for a second pass, as a worker does for the later
    points of its batch."""
    from paper_2210_07912_b200 import ac_loop
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=6.0)
    inp = build(oracle, cfg)
    h = create(rift, inp, rift.RIFT_PREC_MIXED)
    stream = torch.cuda.current_stream().cuda_stream
    lo, hi, nb = synth.HIST_LO, synth.HIST_HI, 100
    n_ref = 2_000_000
    p_ref = torch.from_numpy(np.ascontiguousarray(synth.prior_draw(np.random.default_rng(123), n_ref))).cuda()
    lnL = torch.empty(n_ref, dtype=torch.float64, device="cuda")
    rift.rift_ile_eval_batch(h, [0], n_ref, p_ref, lnL, None, stream)
    ref = rift.rift_ile_reduce(h, 1, n_ref, lnL, None, cuda_stream=stream)

    s = rift.rift_ac_create(6, nb, lo, hi)
    kw = dict(lo=lo, hi=hi, n_bins=nb, d_min_mpc=synth.D_MIN_MPC, d_max_mpc=synth.D_MAX_MPC, n_per_round=50_000,
              n_eff_target=10.0, max_rounds=40, seed=452, cuda_stream=stream)
    first = ac_loop.integrate(h, s, 0, adapt=ac_loop.SKY_ONLY, **kw)
    assert first["n_eff"] >= 10.0 and first["rounds"] < 40, first
    m = rift.rift_ac_get_masses(s, 6, nb)
    assert np.allclose(m[2:], 1.0 / nb, atol=1e-15)                          # psi, iota, phi, D are not adapted
    assert first["rounds"] == 1 or np.max(np.abs(m[:2] - 1.0 / nb)) > 1e-3   # the sky is
    sigma = math.hypot(first["rel_err"], ref["rel_err"][0])
    assert abs(first["lnZ"] - ref["lnZ"][0]) < 5 * sigma + 0.02, (first, ref)

    frozen = ac_loop.integrate(h, s, 0, frozen=True, offset=first["next_offset"], **kw)
    assert frozen["n_eff"] >= 10.0 and frozen["rounds"] < 40, frozen
    assert np.array_equal(rift.rift_ac_get_masses(s, 6, nb), m)              # frozen: the sampler is left alone
    sigma = math.hypot(frozen["rel_err"], ref["rel_err"][0])
    assert abs(frozen["lnZ"] - ref["lnZ"][0]) < 5 * sigma + 0.02, (frozen, ref)
    # equal cost under the prior gives n_eff = ref n_eff * n_evals / n_ref
    assert frozen["n_eff"] > 1.5 * ref["n_eff"][0] * frozen["n_evals"] / n_ref, (frozen, ref)
    with pytest.raises(ValueError):
        rift.rift_ac_update_dims(s, m, 0.1, 1.0, [1, 0])
    rift.rift_ac_destroy(s)
    rift.rift_ile_destroy(h)
