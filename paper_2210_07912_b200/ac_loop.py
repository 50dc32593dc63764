"""Adaptive-cartesian integration of one intrinsic point: the loop of PAPER.md section IV.C.2 (:336-358) with the production
settings of :452 -- iterate rounds of `n_per_round` draws until the pooled n_eff (Eq. (B1), :637) reaches the target (10 in
production), adapting only the dimensions flagged in `adapt` (production: the sky, `SKY_ONLY`), optionally with the sampler
frozen (a worker that assesses a batch of points freezes the skymap after the first point).

Orchestration only: every round is rift_ac_draw -> rift_ac_ile_ln_weight -> rift_ile_eval_batch -> rift_ile_reduce (pooled
state, Eq. (20)-(21) :326-328, and the round's weighted histograms) -> rift_ac_update_dims, all kernels of librift_ile.so on
the given stream; the host sees four scalars and, while adapting, the n_dim x n_bins histograms per round (:352).
"""
from __future__ import annotations

from . import binding as rift

SKY_ONLY = (1, 1, 0, 0, 0, 0)       # RA, dec adapted; psi, iota, phi_ref, distance drawn from their (uniform) initial histograms
ALL_DIMS = (1, 1, 1, 1, 1, 1)


def integrate(h_ile, sampler, point_id: int, lo, hi, n_bins: int, d_min_mpc: float, d_max_mpc: float, n_per_round: int,
              n_eff_target: float = 10.0, max_rounds: int = 100, adapt=SKY_ONLY, frozen: bool = False, floor_mix: float = 0.1,
              temper: float = 0.75, seed: int = 0, offset: int = 0, cuda_stream: int = 0) -> dict:
    """Returns dict(lnZ, rel_err, n_eff, n_ess, rounds, n_evals, next_offset) of the pooled rounds.  `sampler` (rift_ac_create
    over the six extrinsic parameters) is refreshed in place unless `frozen`; `offset` is the first random-number index, so
    that successive calls draw fresh samples (`next_offset` of the previous call)."""
    import torch

    n = int(n_per_round)
    x = torch.empty((6, n), dtype=torch.float64, device="cuda")
    ln_ps = torch.empty(n, dtype=torch.float64, device="cuda")
    ln_w = torch.empty(n, dtype=torch.float64, device="cuda")
    lnL = torch.empty(n, dtype=torch.float64, device="cuda")
    want_hist = not frozen
    out, rounds = None, 0
    while rounds < max_rounds:
        rift.rift_ac_draw(sampler, n, seed, offset + rounds * n, x, ln_ps, cuda_stream)
        rift.rift_ac_ile_ln_weight(n, x, d_min_mpc, d_max_mpc, ln_ps, ln_w, cuda_stream)
        rift.rift_ile_eval_batch(h_ile, [point_id], n, x, lnL, None, cuda_stream)
        # the stored state pools the rounds; its histograms are the pooled ones, which is what the sampler adapts to
        out = rift.rift_ile_reduce(h_ile, 1, n, lnL, ln_w, x if want_hist else None, lo if want_hist else None,
                                   hi if want_hist else None, n_bins if want_hist else 0, merge=1 if rounds else 0,
                                   want_hist=want_hist, cuda_stream=cuda_stream)
        rounds += 1
        if float(out["n_eff"][0]) >= n_eff_target:
            break
        if not frozen:
            rift.rift_ac_update_dims(sampler, out["hist"][0], floor_mix, temper, adapt)
    return dict(lnZ=float(out["lnZ"][0]), rel_err=float(out["rel_err"][0]), n_eff=float(out["n_eff"][0]),
                n_ess=float(out["n_ess"][0]), rounds=rounds, n_evals=rounds * n, next_offset=offset + rounds * n)
