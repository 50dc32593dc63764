"""GPU parity of rift_ile_precompute (Eq. (D4a-c)) against oracle/precompute_oracle.py."""
import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from oracle import precompute_oracle as po
from paper_2210_07912_b200 import synth

from helpers import oracle_geometry_fn, oracle_eval, create

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()
    return t


def device_quv(torch, h, d, w, f, n_t, dt):
    P, K, M, NF = h.shape
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()   # noqa: E731
    hd, dd, wd, fd = dev(h.view(np.float64)), dev(d.view(np.float64)), dev(w), dev(f)
    Q = torch.zeros((P, K, M, n_t, 2), dtype=torch.float64, device="cuda")
    U = torch.zeros((P, K, M, M, 2), dtype=torch.float64, device="cuda")
    V = torch.zeros((P, K, M, M, 2), dtype=torch.float64, device="cuda")
    rift.rift_ile_precompute(P, K, M, hd, dd, wd, f, fd, n_t, dt, Q, U, V, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    c = lambda t: t.cpu().numpy().view(np.complex128)[..., 0]          # noqa: E731
    return c(Q), c(U), c(V), (Q, U, V)


@pytest.mark.parametrize("config,n_points", [(0, 1), (1, 3), (4, 2)])
def test_precompute_matches_oracle_and_feeds_create(torch, oracle, config, n_points):
    """Spectra of the timing configs (C0: 2 x 2 columns, fewer than a column group; C1; C4: 3277 window times): Q, U, V to
    1e-12 of their scale; then a handle created from the DEVICE arrays evaluates lnL like one created from the oracle's."""
    cfg = synth.with_overrides(synth.CONFIGS[config], n_points=n_points)
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    gfn = oracle_geometry_fn(oracle, cfg, loc, resp, ml, mm)
    sps = []
    for p in range(n_points):
        th = synth.true_point(cfg, p)
        F, Y, shift = gfn(th)
        sps.append(synth.make_spectra(cfg, p, np.asarray(F).reshape(-1, 1) * np.asarray(Y).reshape(1, -1), shift,
                                      synth.D_REF_MPC / th[5]))
    h = np.stack([s.h for s in sps])
    d = np.stack([s.d for s in sps])
    w, f = sps[0].w, sps[0].f
    Qg, Ug, Vg, dev_arrays = device_quv(torch, h, d, w, f, cfg.n_t, cfg.delta_t)
    for p in range(n_points):
        Qo, Uo, Vo = po.quv(h[p], d[p], w, f, cfg.n_t, cfg.delta_t)
        assert np.max(np.abs(Qg[p] - Qo)) < 1e-12 * np.max(np.abs(Qo))
        assert np.max(np.abs(Ug[p] - Uo)) < 1e-12 * np.max(np.abs(Uo))
        assert np.max(np.abs(Vg[p] - Vo)) < 1e-12 * np.max(np.abs(Vo))
    # a handle from the device arrays
    Qd, Ud, Vd = dev_arrays
    hnd = rift.rift_ile_create(loc, resp, cfg.gmst, ml, mm, n_points, cfg.n_t, cfg.delta_t, cfg.n_t, synth.D_REF_MPC, Qd, Ud, Vd,
                               input_mem=rift.RIFT_MEM_DEVICE, precision=rift.RIFT_PREC_FP64)
    n = 200
    params = synth.prior_draw(np.random.default_rng(7), n)
    pdev = torch.from_numpy(params).cuda()
    lnL = torch.empty(n, dtype=torch.float64, device="cuda")
    rift.rift_ile_eval_batch(hnd, [n_points - 1], n, pdev, lnL)
    torch.cuda.synchronize()
    ref = oracle.eval_batch(loc, resp, cfg.gmst, ml, mm, cfg.delta_t, synth.D_REF_MPC, Qg[n_points - 1], Ug[n_points - 1],
                            Vg[n_points - 1], params)[0]
    got = lnL.cpu().numpy()
    assert np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))) < 1e-10
    rift.rift_ile_destroy(hnd)


def test_precompute_unequal_bins_and_two_sided_weights(torch):
    """An unequally spaced list with negative frequencies (the two-sided form of Eq. (D4a)): every phase is evaluated exactly."""
    rng = np.random.default_rng(5)
    P, K, M, NF, n_t, dt = 2, 2, 3, 301, 65, 1.0 / 2048.0
    f = np.sort(np.concatenate([rng.uniform(-900.0, -20.0, NF // 2), rng.uniform(20.0, 900.0, NF - NF // 2)]))
    h = rng.standard_normal((P, K, M, NF)) + 1j * rng.standard_normal((P, K, M, NF))
    d = rng.standard_normal((P, K, NF)) + 1j * rng.standard_normal((P, K, NF))
    w = rng.uniform(0.5, 2.0, (K, NF))
    Qg, Ug, Vg, _ = device_quv(torch, h, d, w, f, n_t, dt)
    for p in range(P):
        Qo, Uo, Vo = po.quv(h[p], d[p], w, f, n_t, dt)
        assert np.max(np.abs(Qg[p] - Qo)) < 1e-12 * np.max(np.abs(Qo))
        assert np.max(np.abs(Ug[p] - Uo)) < 1e-12 * np.max(np.abs(Uo)) and np.max(np.abs(Vg[p] - Vo)) < 1e-12 * np.max(np.abs(Vo))
