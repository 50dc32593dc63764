"""Gaussian-mixture adaptive integration of one intrinsic point in the configuration PAPER.md recommends for loud signals
(:807): "GMM sampling, using sky- and phase-rotated coordinates, with distance marginalization" -- here the GMM sampler of
section IV.C.1 / Appendix A (rift_gmm.h), the rotated network-frame sky of :248 (rift_sky.h) and the distance-marginalised
evaluation of section IV.C.3 (rift_ile_eval_batch_dmarg).  The phase-rotated coordinates are not built.

The five extrinsic parameters left after the distance marginal are sampled by independent groups (factors of p_s): the sky pair
(lambda, beta) of the network frame by a two-dimensional mixture (the pair whose correlation the frame is chosen to remove, and
what remains of it), and iota, psi, phi_ref by one-dimensional mixtures.  Orchestration only: every round is
    rift_gmm_draw (per group) -> rift_gmm_add (ln p_s) -> rift_ac_ile_ln_weight (ln prior - ln p_s, the prior of (lambda, beta)
    being cos(beta) / 4 pi as for (RA, dec)) -> rift_sky_network_to_radec -> rift_ile_eval_batch_dmarg -> rift_ile_reduce
    (pooled over rounds, Eq. (20)-(21)) -> rift_gmm_add (ln omega) -> rift_gmm_fit_tempered (per adapted group, on weights
    tempered to an effective sample size of at least `ess_min`, reading G7; merged online from the second round, Eq. (A8)-(A11)),
all kernels of librift_ile.so on the given stream; the host sees four scalars per round and the mixtures' parameters.
"""
from __future__ import annotations

import math

from . import binding as rift

TWO_PI = 2.0 * math.pi
# (name, rows of the parameter array, lo, hi): rows index (lambda, beta, psi, iota, phi_ref)
GROUPS = (("sky", (0, 1), (0.0, -0.5 * math.pi), (TWO_PI, 0.5 * math.pi)),
          ("psi", (2,), (0.0,), (math.pi,)),
          ("iota", (3,), (0.0,), (math.pi,)),
          ("phi_ref", (4,), (0.0,), (TWO_PI,)))


def create_samplers(n_comp_sky: int = 2, n_comp_1d: int = 1) -> dict:
    """One mixture per group, in its wide initial state (close to the uniform density on the group's domain)."""
    return {name: rift.rift_gmm_create(len(rows), n_comp_sky if name == "sky" else n_comp_1d, lo, hi)
            for name, rows, lo, hi in GROUPS}


def destroy_samplers(samplers: dict) -> None:
    for g in samplers.values():
        rift.rift_gmm_destroy(g)


def integrate(h_ile, samplers: dict, point_id: int, R, gmst_rad: float, d_min_mpc: float, d_max_mpc: float, n_dist: int,
              n_per_round: int, n_eff_target: float = 10.0, max_rounds: int = 20, adapt=("sky", "iota"), em_iters: int = 20,
              em_tol: float = 1e-8, reg: float = 1e-6, ess_min: float = 300.0, seed: int = 0, offset: int = 0, cuda_stream: int = 0) -> dict:
    """Returns dict(lnZ, rel_err, n_eff, n_ess, rounds, n_evals, next_offset) of the pooled rounds; lnZ is the evidence of
    the point marginalised over all six extrinsic parameters.  `samplers` (create_samplers) are refitted in place for the
    groups named in `adapt`; R is rift_sky_network_frame of the two detectors that define the pole."""
    import torch

    n = int(n_per_round)
    x = torch.empty((6, n), dtype=torch.float64, device="cuda")          # lambda, beta, psi, iota, phi_ref, (distance)
    d_const = 0.5 * (d_min_mpc + d_max_mpc)
    x[5].fill_(d_const)                                                   # a constant: its prior density is taken out below
    sky = torch.empty((2, n), dtype=torch.float64, device="cuda")        # RA, dec of (lambda, beta)
    ln_ps_g = torch.empty((len(GROUPS), n), dtype=torch.float64, device="cuda")
    ln_ps = torch.empty(n, dtype=torch.float64, device="cuda")
    ln_w = torch.empty(n, dtype=torch.float64, device="cuda")
    ln_om = torch.empty(n, dtype=torch.float64, device="cuda")
    lnL = torch.empty(n, dtype=torch.float64, device="cuda")
    # rift_ac_ile_ln_weight includes ln p(D) of the constant distance row; the marginal already holds the distance prior
    ln_p_dist = math.log(3.0 * d_const ** 2 / (d_max_mpc ** 3 - d_min_mpc ** 3))
    out, rounds, n_refit_failures = None, 0, 0
    while rounds < max_rounds:
        for gi, (name, rows, _lo, _hi) in enumerate(GROUPS):
            # every group has its own random-number stream: seed + group index
            rift.rift_gmm_draw(samplers[name], n, seed + gi, offset + rounds * n, [x[r] for r in rows], ln_ps_g[gi],
                               cuda_stream=cuda_stream)
        rift.rift_gmm_add(n, [ln_ps_g[gi] for gi in range(len(GROUPS))], ln_ps, cuda_stream)
        rift.rift_ac_ile_ln_weight(n, x, d_min_mpc, d_max_mpc, ln_ps, ln_w, cuda_stream)
        rift.rift_sky_network_to_radec(n, R, gmst_rad, x[0], x[1], sky[0], sky[1], cuda_stream)
        rift.rift_ile_eval_batch_dmarg(h_ile, [point_id], n, [sky[0], sky[1], x[2], x[3], x[4]], d_min_mpc, d_max_mpc, n_dist,
                                       lnL, None, cuda_stream)
        out = rift.rift_ile_reduce(h_ile, 1, n, lnL, ln_w, merge=1 if rounds else 0, cuda_stream=cuda_stream)
        rounds += 1
        if float(out["n_eff"][0]) >= n_eff_target:
            break
        rift.rift_gmm_add(n, [lnL, ln_w], ln_om, cuda_stream)
        for name, rows, _lo, _hi in GROUPS:
            if name in adapt:
                try:
                    rift.rift_gmm_fit_tempered(samplers[name], n, [x[r] for r in rows], ln_om, ess_min, em_iters, em_tol, reg,
                                               merge=1 if rounds > 1 else 0, cuda_stream=cuda_stream)
                except rift.RiftError as err:        # an emptied component or a singular covariance: the library left the
                    if err.code != rift.RIFT_ESTATE:  # group's model unchanged; keep sampling from it
                        raise
                    n_refit_failures += 1
    return dict(lnZ=float(out["lnZ"][0]) - ln_p_dist, rel_err=float(out["rel_err"][0]), n_eff=float(out["n_eff"][0]),
                n_ess=float(out["n_ess"][0]), rounds=rounds, n_evals=rounds * n, next_offset=offset + rounds * n,
                refit_failures=n_refit_failures)
