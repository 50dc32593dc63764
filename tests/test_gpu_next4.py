"""GPU parity of the small NEXT-4 pieces against oracle/sky_oracle.py on the same seeded inputs:
the rotated network-frame sky transforms (include/rift_sky.h) and rho_guess (rift_ile_rho_guess, Eq. (D7))."""
import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from paper_2210_07912_b200 import synth
from oracle import sky_oracle as so

from helpers import build, create

pytestmark = pytest.mark.gpu

TOL_ANGLE = 1e-12            # fp64 sincos / atan2 / asin away from the poles of asin (checked separately on the unit vector)


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def _unit(lon, lat):
    return np.stack([np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)], axis=-1)


@pytest.mark.parametrize("pair,gmst,n", [((0, 1), 0.0, 100_003), ((2, 0), 1.7, 4097), ((1, 2), 5.9, 1)])
def test_network_frame_transforms_match_oracle(torch, pair, gmst, n):
    loc, _ = synth.detector_arrays(synth.CONFIGS[1])
    R = rift.rift_sky_network_frame(loc[pair[0]], loc[pair[1]])
    assert np.max(np.abs(R - so.network_frame(loc[pair[0]], loc[pair[1]]))) < 1e-15
    rng = np.random.default_rng(11 + n)
    lam = rng.uniform(0, 2 * np.pi, n)
    beta = np.arcsin(rng.uniform(-1, 1, n))
    if n > 10:                                       # the poles and the seam
        lam[:4] = [0.0, np.pi, 2 * np.pi - 1e-13, 1.0]
        beta[:4] = [np.pi / 2, -np.pi / 2, 0.0, 0.0]
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ra_d, dec_d = torch.empty(n, dtype=torch.float64, device="cuda"), torch.empty(n, dtype=torch.float64, device="cuda")
    rift.rift_sky_network_to_radec(n, R, gmst, d(lam), d(beta), ra_d, dec_d, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    ra, dec = ra_d.cpu().numpy(), dec_d.cpu().numpy()
    ra_o, dec_o = so.network_to_radec(lam, beta, R, gmst)
    assert np.all((ra >= 0) & (ra < 2 * np.pi)) and np.all(np.abs(dec) <= np.pi / 2)
    # directions agree to rounding everywhere; angles agree to rounding away from the poles (asin' and atan2 blow up there)
    assert np.max(np.abs(_unit(ra, dec) - _unit(ra_o, dec_o))) < 1e-7
    away = np.abs(dec_o) < 1.5
    dra = np.abs(ra - ra_o)
    assert np.max(np.minimum(dra, 2 * np.pi - dra)[away]) < TOL_ANGLE and np.max(np.abs(dec - dec_o)[away]) < TOL_ANGLE
    # the inverse, from the oracle's equatorial angles, and in place
    lam_d, beta_d = d(ra_o), d(dec_o)
    rift.rift_sky_radec_to_network(n, R, gmst, lam_d, beta_d, lam_d, beta_d, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    lam2, beta2 = lam_d.cpu().numpy(), beta_d.cpu().numpy()
    lam_o, beta_o = so.radec_to_network(ra_o, dec_o, R, gmst)
    away = np.abs(beta_o) < 1.5
    dl = np.abs(lam2 - lam_o)
    assert np.max(np.minimum(dl, 2 * np.pi - dl)[away]) < TOL_ANGLE and np.max(np.abs(beta2 - beta_o)[away]) < TOL_ANGLE
    assert np.max(np.abs(_unit(lam2, beta2) - _unit(lam, beta))) < 1e-7


def test_rotated_sky_feeds_eval_batch(torch, oracle):
    """End to end: samples drawn in the network frame, turned into (RA, dec) on the device, evaluate to the oracle's lnL at the
    oracle's own transform of the same draws (fp64 mode, rel 1e-10 where the integer shifts agree)."""
    cfg = synth.with_overrides(synth.CONFIGS[0], n_points=1)
    inp = build(oracle, cfg, n_points=1)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    n = 3000
    params, _ = synth.draw_samples(cfg, 321, n)
    rng = np.random.default_rng(3)
    lam, beta = rng.uniform(0, 2 * np.pi, n), np.arcsin(rng.uniform(-1, 1, n))
    R = rift.rift_sky_network_frame(inp.det_location[0], inp.det_location[1])
    p = torch.from_numpy(np.ascontiguousarray(params)).cuda()
    p[0], p[1] = torch.from_numpy(lam).cuda(), torch.from_numpy(beta).cuda()
    s = torch.cuda.current_stream().cuda_stream
    rift.rift_sky_network_to_radec(n, R, cfg.gmst, p[0], p[1], p[0], p[1], s)
    lnL = torch.empty(n, dtype=torch.float64, device="cuda")
    sh = torch.zeros((n, cfg.n_det), dtype=torch.int32, device="cuda")
    rift.rift_ile_eval_batch(h, [0], n, p, lnL, sh, s)
    torch.cuda.synchronize()
    ra_o, dec_o = so.network_to_radec(lam, beta, so.network_frame(inp.det_location[0], inp.det_location[1]), cfg.gmst)
    po = params.copy()
    po[0], po[1] = ra_o, dec_o
    ref, sh_o = oracle.eval_batch(inp.det_location, inp.det_response, cfg.gmst, inp.mode_l, inp.mode_m, cfg.delta_t,
                                  synth.D_REF_MPC, inp.Q[0], inp.U[0], inp.V[0], po)[:2]
    same = np.all(sh.cpu().numpy() == sh_o, axis=1)          # a delay within 1e-12 samples of a half-integer may round either way
    assert same.mean() > 0.999
    g = lnL.cpu().numpy()
    assert np.max(np.abs(g - ref)[same] / np.maximum(1.0, np.abs(ref[same]))) < 1e-9
    rift.rift_ile_destroy(h)


@pytest.mark.parametrize("config,precision", [(0, "fp64"), (1, "fp64"), (1, "mixed")])
def test_rho_guess_matches_oracle(torch, oracle, config, precision):
    cfg = synth.with_overrides(synth.CONFIGS[config], n_points=min(3, synth.CONFIGS[config].n_points))
    inp = build(oracle, cfg, n_points=cfg.n_points)
    h = create(rift, inp, rift.RIFT_PREC_FP64 if precision == "fp64" else rift.RIFT_PREC_MIXED)
    got = rift.rift_ile_rho_guess(h, cfg.n_points)
    ref = np.array([so.rho_guess(inp.Q[p], inp.U[p]) for p in range(cfg.n_points)])
    tol = 1e-13 if precision == "fp64" else 2e-7          # mixed mode stores Q as complex64
    assert np.max(np.abs(got - ref) / ref) < tol, (got, ref)
    # the synthetic signal has rho = 12 by construction: the estimate lands within the paper's "corresponds closely"
    assert np.all((got > 12.0 / 2.3 * 0.5) & (got < 12.0 * 2.0))
    rift.rift_ile_destroy(h)
