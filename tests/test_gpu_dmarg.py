"""GPU parity of the distance-marginalised evaluation (rift_ile_eval_batch_dmarg) against
oracle/dmarg_oracle.c on the same seeded inputs: rule for rule (same nodes: the difference is rounding), and against the
converged definition (the difference is the quadrature error the header quotes)."""
import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from paper_2210_07912_b200 import synth

from helpers import build, create, rel_err

pytestmark = pytest.mark.gpu

D_MIN, D_MAX = synth.D_MIN_MPC, synth.D_MAX_MPC
TOL_FP64_REL = 1e-9          # polynomial exp2 (1e-12) and a different summation order over n_dist * N_tau terms
TOL_MIXED = 2e-3             # BASELINE.json north_star, mixed mode


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def oracle_dm(oracle, inp, point, params, n_panels):
    cfg = inp.cfg
    return oracle.eval_batch_dmarg(inp.det_location, inp.det_response, cfg.gmst, inp.mode_l, inp.mode_m, cfg.delta_t,
                                   synth.D_REF_MPC, inp.Q[point], inp.U[point], inp.V[point], params[:5], D_MIN, D_MAX, n_panels)


def gpu_dm(torch, h, ids, n, params, n_dist, K):
    p = torch.from_numpy(np.ascontiguousarray(params[:5])).cuda()
    lnL = torch.full((p.shape[1],), float("nan"), dtype=torch.float64, device="cuda")
    sh = torch.zeros((p.shape[1], K), dtype=torch.int32, device="cuda")
    rift.rift_ile_eval_batch_dmarg(h, ids, n, p, D_MIN, D_MAX, n_dist, lnL, sh, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return lnL.cpu().numpy(), sh.cpu().numpy()


@pytest.mark.parametrize("config,n", [(0, 777), (1, 400), (4, 96)])
def test_dmarg_matches_oracle_rule_for_rule(torch, oracle, config, n):
    """C0 (2 detectors, 2 modes), C1 shape, and C4 shape (3277-sample window: several blocks per sample, two contractions);
    two segments with repeated intrinsic ids and a ragged sample count."""
    cfg = synth.with_overrides(synth.CONFIGS[config], n_points=2 if config else 1)
    inp = build(oracle, cfg, n_points=cfg.n_points)
    ids = [cfg.n_points - 1, 0]
    params = np.concatenate([synth.draw_samples(cfg, 30 + s, n)[0] for s in range(2)], axis=1)
    ref = np.concatenate([oracle_dm(oracle, inp, ids[s], params[:, s * n:(s + 1) * n], 8)[0] for s in range(2)])
    sref = np.concatenate([oracle_dm(oracle, inp, ids[s], params[:, s * n:(s + 1) * n][:, :4], 1)[1] for s in range(2)])
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        got, sh = gpu_dm(torch, h, ids, n, params, 64, cfg.n_det)
        assert "dmarg" in rift.rift_ile_kernel_name(h)
        assert np.array_equal(np.concatenate([sh[:4], sh[n:n + 4]]), sref)
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL, np.max(rel_err(got, ref))
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED, np.max(np.abs(got - ref))
        rift.rift_ile_destroy(h)


def test_dmarg_against_the_converged_definition_and_evidence(torch, oracle):
    """128 nodes against the converged oracle (512 panels) at rho = 5 and rho = 12 (quadrature error < 1e-5), the 5-D
    evidence from rift_ile_reduce, a NaN sample, and argument validation."""
    for rho in (5.0, 12.0):
        cfg = synth.with_overrides(synth.CONFIGS[0], rho=rho)
        inp = build(oracle, cfg)
        n = 1500
        params = synth.draw_samples(cfg, 3, n)[0]
        params[2, 17] = np.nan
        ref = oracle_dm(oracle, inp, 0, params, 512)[0]
        assert np.isnan(ref[17]) and np.isnan(ref).sum() == 1
        ok = ~np.isnan(ref)
        zr = oracle.reduce(ref[ok])
        h = create(rift, inp, rift.RIFT_PREC_FP64)
        got, _ = gpu_dm(torch, h, [0], n, params, 128, cfg.n_det)
        assert np.isnan(got[17]) and np.isnan(got).sum() == 1
        assert np.max(rel_err(got[ok], ref[ok])) < 1e-5
        lnL = torch.from_numpy(got[ok]).cuda()
        red = rift.rift_ile_reduce(h, 1, int(ok.sum()), lnL)
        assert abs(red["lnZ"][0] - zr["lnZ"]) < 1e-5 * max(1.0, abs(zr["lnZ"])) and abs(red["n_ess"][0] - zr["n_ess"]) < 1e-4 * zr["n_ess"]
        p = torch.from_numpy(params[:5]).cuda()
        out = torch.empty(n, dtype=torch.float64, device="cuda")
        for bad in (dict(n_dist=60), dict(n_dist=1024), dict(d_min=0.0), dict(d_max=10.0)):
            kw = dict(d_min=D_MIN, d_max=D_MAX, n_dist=64)
            kw.update(bad)
            with pytest.raises(rift.RiftError) as e:
                rift.rift_ile_eval_batch_dmarg(h, [0], n, p, kw["d_min"], kw["d_max"], kw["n_dist"], out)
            assert e.value.code == rift.RIFT_EINVAL
        rift.rift_ile_destroy(h)
