"""GPU parity: the CUDA path (through the C ABI binding) against the CPU oracle, element by element on the same
seeded inputs.  Tolerances (BASELINE.json north_star): shifts bit-exact; fp64 mode lnL relative 1e-10 (relative to
max(1,|lnL|)); mixed mode |dlnL| <= 2e-3 and |dlnZ| <= 1e-3."""
import math

import numpy as np
import pytest

import paper_2210_07912_b200 as rift
from paper_2210_07912_b200 import synth

from helpers import build, create, oracle_eval, rel_err

pytestmark = pytest.mark.gpu

TOL_FP64_REL = 1e-10
TOL_MIXED_LNL = 2e-3
TOL_MIXED_LNZ = 1e-3


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    rift.lib()                       # fail loudly if the extension is missing
    return t


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_eval(torch, h, ids, n_per_seg, params, want_shifts=True, K=None, kernel=None):
    if kernel is not None:
        rift.rift_ile_set_kernel(h, kernel)
    p = dev(torch, params)
    n = p.shape[1]
    lnL = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    sh = torch.zeros((n, K), dtype=torch.int32, device="cuda") if want_shifts else None
    rift.rift_ile_eval_batch(h, ids, n_per_seg, p, lnL, sh, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return lnL, sh, p


# ------------------------------------------------------------------------------------------------ geometry
def test_geometry_kernel_matches_oracle(torch, oracle):
    cfg = synth.with_overrides(synth.CONFIGS[2], n_points=1)          # 21 modes, l = 2..4
    inp = build(oracle, cfg, n_points=1)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    n = 3001
    params = synth.prior_draw(np.random.default_rng(5), n)
    p = dev(torch, params)
    K, M = cfg.n_det, cfg.n_modes
    F = torch.zeros((n, K, 2), dtype=torch.float64, device="cuda")
    Y = torch.zeros((n, M, 2), dtype=torch.float64, device="cuda")
    sh = torch.zeros((n, K), dtype=torch.int32, device="cuda")
    quad = torch.zeros(n, dtype=torch.float64, device="cuda")
    rift.rift_ile_geometry(h, 0, n, p, F, Y, sh, quad, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    F = F.cpu().numpy().view(np.complex128)[..., 0]
    Y = Y.cpu().numpy().view(np.complex128)[..., 0]
    Fo = oracle.antenna(params[0], params[1], params[2], cfg.gmst, inp.det_response)
    Yo = oracle.harmonics(params[3], params[4], inp.mode_l, inp.mode_m)
    _dt, so, fr = oracle.delays(params[0], params[1], cfg.gmst, inp.det_location, cfg.delta_t)
    assert np.max(np.abs(F - Fo)) < 1e-14
    assert np.max(np.abs(Y - Yo)) < 1e-14
    ok = fr.sum(axis=1) == 0
    assert np.array_equal(sh.cpu().numpy()[ok], so[ok])
    for i in range(0, n, 97):
        c = synth.D_REF_MPC / params[5, i]
        q = oracle.lnl_core(Fo[i], Yo[i], c, so[i], inp.Q[0], inp.U[0], inp.V[0])[2]
        assert abs(quad[i].item() - q) < 1e-12 * max(1.0, abs(q))
    rift.rift_ile_destroy(h)


def test_higher_l_harmonics(torch, oracle):
    modes = tuple((l, m) for l in (5, 6, 7, 8) for m in (-l, -3, 0, 2, l))
    cfg = synth.with_overrides(synth.CONFIGS[0], modes=modes, f_s=512.0, t_window=0.02)
    inp = build(oracle, cfg)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    n = 500
    params = synth.prior_draw(np.random.default_rng(6), n)
    Y = torch.zeros((n, len(modes), 2), dtype=torch.float64, device="cuda")
    rift.rift_ile_geometry(h, 0, n, dev(torch, params), None, Y, None, None)
    torch.cuda.synchronize()
    Yo = oracle.harmonics(params[3], params[4], inp.mode_l, inp.mode_m)
    assert np.max(np.abs(Y.cpu().numpy().view(np.complex128)[..., 0] - Yo)) < 2e-14
    rift.rift_ile_destroy(h)


# ------------------------------------------------------------------------------------------------ C0, whole config
KERNELS = [rift.RIFT_KERNEL_AUTO, rift.RIFT_KERNEL_DIRECT, rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS, rift.RIFT_KERNEL_MMA,
           rift.RIFT_KERNEL_SKY]
TC_FAMILY = (rift.RIFT_KERNEL_AUTO, rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS, rift.RIFT_KERNEL_MMA)   # MMA: fp64 only, AUTO in mixed
MMA_FAMILY = (rift.RIFT_KERNEL_AUTO, rift.RIFT_KERNEL_MMA, rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS)  # TC/TCS: mixed only, AUTO in fp64


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("rho", [12.0, 30.0])
def test_c0_all_samples_both_precisions(torch, oracle, rho, kernel):
    cfg = synth.with_overrides(synth.CONFIGS[0], rho=rho)
    inp = build(oracle, cfg)
    params, ln_w = synth.draw_samples(cfg, 0)
    ref, sh_ref, fr = oracle_eval(oracle, inp, 0, params)
    red_ref = oracle.reduce(ref, ln_w, params, synth.HIST_LO, synth.HIST_HI, 100)
    for prec, name in ((rift.RIFT_PREC_FP64, "fp64"), (rift.RIFT_PREC_MIXED, "mixed")):
        h = create(rift, inp, prec)
        lnL, sh, p = gpu_eval(torch, h, [0], cfg.n_samples, params, K=cfg.n_det, kernel=kernel)
        got = lnL.cpu().numpy()
        assert np.array_equal(sh.cpu().numpy()[fr == 0], sh_ref[fr == 0])
        # the tcgen05 kernel is the default of the mixed mode (and never runs in fp64 mode)
        assert ("lnl_tc" in rift.rift_ile_kernel_name(h)) == (
            prec == rift.RIFT_PREC_MIXED and kernel in TC_FAMILY)
        assert ("lnl_sky" in rift.rift_ile_kernel_name(h)) == (kernel == rift.RIFT_KERNEL_SKY)   # both precision modes
        # the shift-sorted variant: on request, or by default when the segments are long enough to fill its buckets
        if prec == rift.RIFT_PREC_MIXED and kernel == rift.RIFT_KERNEL_TCS:
            assert "lnl_tcs" in rift.rift_ile_kernel_name(h)
        # the FP64 tensor-core kernel is the default of the fp64 mode (and never runs in mixed mode)
        assert ("lnl_mma" in rift.rift_ile_kernel_name(h)) == (prec == rift.RIFT_PREC_FP64 and kernel in MMA_FAMILY)
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL, name
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL, name
        red = rift.rift_ile_reduce(h, 1, cfg.n_samples, lnL, dev(torch, ln_w), p, synth.HIST_LO, synth.HIST_HI, 100,
                                   merge=0, want_hist=True)
        tol = 1e-10 * max(1.0, abs(red_ref["lnZ"])) if prec == rift.RIFT_PREC_FP64 else TOL_MIXED_LNZ
        assert abs(red["lnZ"][0] - red_ref["lnZ"]) < tol
        rtol = 1e-9 if prec == rift.RIFT_PREC_FP64 else 5e-3
        assert abs(red["n_eff"][0] - red_ref["n_eff"]) < rtol * red_ref["n_eff"]
        assert abs(red["n_ess"][0] - red_ref["n_ess"]) < rtol * red_ref["n_ess"]
        assert abs(red["rel_err"][0] - red_ref["rel_err"]) < rtol
        assert np.max(np.abs(red["hist"][0] - red_ref["hist"])) < rtol
        assert "lnl_" in rift.rift_ile_kernel_name(h)
        assert rift.rift_ile_launch_count(h) >= 4
        rift.rift_ile_destroy(h)


# ------------------------------------------------------------------------------------------------ C1 reduced + ragged
@pytest.mark.parametrize("kernel", KERNELS)
def test_c1_multi_point_ragged_segments(torch, oracle, kernel):
    cfg = synth.CONFIGS[1]
    inp = build(oracle, cfg, n_points=3)
    n_per = 2 * 256 + 37                                    # several warps' worth and a ragged tail
    ids = [2, 0, 1, 0]                                      # repeated and permuted intrinsic ids
    params = np.concatenate([synth.draw_samples(cfg, 10 + s, n_per)[0] for s in range(len(ids))], axis=1)
    ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n_per:(s + 1) * n_per])[0]
                          for s in range(len(ids))])
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        lnL, _sh, _p = gpu_eval(torch, h, ids, n_per, params, K=cfg.n_det, kernel=kernel)
        got = lnL.cpu().numpy()
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL
        rift.rift_ile_destroy(h)


def test_edge_sizes_and_invalid_samples(torch, oracle):
    cfg = synth.CONFIGS[0]
    inp = build(oracle, cfg)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    # empty batches are a no-op
    lnL = torch.zeros(4, dtype=torch.float64, device="cuda")
    p4 = dev(torch, synth.prior_draw(np.random.default_rng(1), 4))
    rift.rift_ile_eval_batch(h, [], 0, p4, lnL)
    rift.rift_ile_eval_batch(h, [0], 0, p4, lnL)
    for n in (1, 7, 33):
        params = synth.prior_draw(np.random.default_rng(n), n)
        got, _, _ = gpu_eval(torch, h, [0], n, params, K=cfg.n_det)
        ref = oracle_eval(oracle, inp, 0, params)[0]
        assert np.max(rel_err(got.cpu().numpy(), ref)) < TOL_FP64_REL
    # dist <= 0 and NaN parameters: NaN for that sample only
    params = synth.prior_draw(np.random.default_rng(9), 64)
    params[5, 3] = -10.0
    params[5, 4] = 0.0
    params[0, 5] = np.nan
    params[3, 40] = np.nan
    got = gpu_eval(torch, h, [0], 64, params, K=cfg.n_det)[0].cpu().numpy()
    ref = oracle_eval(oracle, inp, 0, params)[0]
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.isnan(got).sum() == 4
    ok = ~np.isnan(ref)
    assert np.max(rel_err(got[ok], ref[ok])) < TOL_FP64_REL
    # error codes
    with pytest.raises(rift.RiftError) as e:
        rift.rift_ile_eval_batch(h, [1], 4, p4, lnL)
    assert e.value.code == rift.RIFT_ERANGE
    with pytest.raises(rift.RiftError) as e:
        rift.rift_ile_eval_batch(h, [0], 4, p4, None)
    assert e.value.code == rift.RIFT_EINVAL
    rift.rift_ile_destroy(h)


@pytest.mark.parametrize("kernel", [rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS])
def test_tc_edge_sizes_ragged_batches_and_invalid_samples(torch, oracle, kernel):
    """Tensor-core kernel (mixed mode): sample counts around the 16-sample batch, several short segments in one call,
    NaN / non-positive distance samples (NaN for that sample only)."""
    cfg = synth.CONFIGS[1]
    inp = build(oracle, cfg, n_points=2)
    h = create(rift, inp, rift.RIFT_PREC_MIXED)
    for n in (1, 7, 16, 17, 33):
        ids = [1, 0, 1]
        params = synth.prior_draw(np.random.default_rng(100 + n), n * len(ids))
        got = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=kernel)[0].cpu().numpy()
        assert ("lnl_tcs" if kernel == rift.RIFT_KERNEL_TCS else "lnl_tc<") in rift.rift_ile_kernel_name(h)
        ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(len(ids))])
        assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL, n
    params = synth.prior_draw(np.random.default_rng(9), 64)
    params[5, 3] = -10.0
    params[5, 4] = 0.0
    params[0, 5] = np.nan
    params[3, 40] = np.nan
    got = gpu_eval(torch, h, [0], 64, params, K=cfg.n_det, kernel=kernel)[0].cpu().numpy()
    ref = oracle_eval(oracle, inp, 0, params)[0]
    assert np.array_equal(np.isnan(got), np.isnan(ref)) and np.isnan(got).sum() == 4
    ok = ~np.isnan(ref)
    assert np.max(np.abs(got[ok] - ref[ok])) < TOL_MIXED_LNL
    rift.rift_ile_destroy(h)


_L2 = tuple((2, m) for m in range(-2, 3))
_L3 = tuple((3, m) for m in range(-3, 4))
TC_SHAPES = [
    # detectors, modes, f_s, window -> (row tiles, passes) of the tensor-core kernel
    (("H1",), _L2[:3], 1024.0, 0.04),                                # K=1, 3 modes, N_t=83: one row tile, no exchange
    (("H1", "L1"), _L2 + _L3, 4096.0, 0.05),                         # K=2, 12 modes: two passes of 6
    (("H1", "L1", "V1"), _L2 + _L3[1:5], 2048.0, 0.05),              # K=3, 9 modes, N_t=205: two row tiles, two passes
    (("H1", "L1", "V1", "S0"), _L2[1:4], 2048.0, 0.08),              # K=4, 3 modes, N_t=329: three row tiles
    (("H1", "L1", "V1", "S0", "S1"), ((2, 2), (2, -2)), 512.0, 0.2),    # K=5, 2 modes, N_t=205 at 512 Hz (small halo)
]


@pytest.mark.parametrize("kernel", [rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS])
@pytest.mark.parametrize("shape", range(len(TC_SHAPES)))
def test_tc_kernel_shapes(torch, oracle, shape, kernel):
    """Detector counts, mode counts (one or several mode-subset passes) and window lengths other than C0-C3's: every
    (row tiles, pitch, pass) instantiation the plan can pick is compared with the oracle.  The shift-sorted variant exists
    for two or more detectors (K = 2: no exchange left; K = 4, 5: two and three exchanged detectors), single- and multi-pass."""
    dets, modes, f_s, t_w = TC_SHAPES[shape]
    cfg = synth.with_overrides(synth.CONFIGS[1], detectors=dets, modes=modes, f_s=f_s, t_window=t_w, n_points=2)
    inp = build(oracle, cfg, n_points=2)
    n = 333
    ids = [1, 0]
    params = np.concatenate([synth.draw_samples(cfg, 40 + s, n)[0] for s in range(len(ids))], axis=1)
    ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(len(ids))])
    h = create(rift, inp, rift.RIFT_PREC_MIXED)
    got, sh, _ = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=kernel)
    name = rift.rift_ile_kernel_name(h)
    assert "lnl_tc" in name, name
    assert ("passes" in name) == (len(modes) > 8)
    assert ("lnl_tcs" in name) == (kernel == rift.RIFT_KERNEL_TCS and len(dets) >= 2), name
    assert np.max(np.abs(got.cpu().numpy() - ref)) < TOL_MIXED_LNL
    rift.rift_ile_destroy(h)


@pytest.mark.parametrize("shape", ["c4", "c1", "c2", "m12", "k1", "k2_512hz"])
def test_sky_kernel_shapes(torch, oracle, shape):
    """Sky-sorted, time-tiled kernel (mixed mode) on request: the C4 shape (5 detectors, 9 modes, 3277-sample window = 15 time
    blocks), the C1 shape (two blocks), 21 and 12 modes (operand rows cut into two K pieces), one detector (no shifts at
    all), two detectors at 512 Hz (a handful of sky cells);
    three segments with repeated intrinsic ids, sample counts far below a cell's batch (mostly padding slots), a NaN sample."""
    cfg = {"c4": synth.with_overrides(synth.CONFIGS[4], n_points=2),
           "c1": synth.with_overrides(synth.CONFIGS[1], n_points=2),
           "c2": synth.with_overrides(synth.CONFIGS[2], n_points=2),                      # 21 modes: two K pieces per chunk
           "m12": synth.with_overrides(synth.CONFIGS[1], modes=_L2 + _L3, n_points=2),    # 12 modes: two pieces of 6 planes
           "k1": synth.with_overrides(synth.CONFIGS[1], detectors=("V1",), n_points=2),
           "k2_512hz": synth.with_overrides(synth.CONFIGS[0], f_s=512.0, t_window=0.5, n_points=2)}[shape]
    inp = build(oracle, cfg, n_points=2)
    n, ids = (257 if shape == "c4" else 1111), [1, 0, 1]
    params = np.concatenate([synth.draw_samples(cfg, 50 + s, n)[0] for s in range(len(ids))], axis=1)
    params[3, 5] = np.nan
    ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(len(ids))])
    sref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[1] for s in range(len(ids))])
    ok = ~np.isnan(ref)
    for prec in (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64):
        if prec == rift.RIFT_PREC_FP64 and shape in ("c2", "m12"):
            continue                                          # fp64 sibling: mode sets whose 256-row chunks fit the ring (M <~ 10)
        h = create(rift, inp, prec)
        got, sh, _ = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=rift.RIFT_KERNEL_SKY)
        assert rift.rift_ile_kernel_name(h) == ("lnl_sky<f16x3>" if prec == rift.RIFT_PREC_MIXED else "lnl_sky<f64>")
        got = got.cpu().numpy()
        assert np.isnan(got[5]) and np.isnan(ref[5]) and np.isnan(got).sum() == 1
        if prec == rift.RIFT_PREC_MIXED:
            assert np.max(np.abs(got[ok] - ref[ok])) < TOL_MIXED_LNL, np.max(np.abs(got[ok] - ref[ok]))
        else:
            assert np.max(rel_err(got[ok], ref[ok])) < TOL_FP64_REL, np.max(rel_err(got[ok], ref[ok]))
        assert np.array_equal(sh.cpu().numpy()[ok], sref[ok])
        rift.rift_ile_destroy(h)


def test_tcs_chunks_across_segments(torch, oracle):
    """Shift-sorted variant with a small chunk workspace: chunks that start and end inside segments, several segments
    per chunk, a ragged last batch in every segment; and the default kernel choice."""
    cfg = synth.CONFIGS[1]
    inp = build(oracle, cfg, n_points=3)
    n, ids = 3533, [2, 0, 1, 1, 0, 2, 0, 1, 2, 0, 1, 2]
    params = np.concatenate([synth.draw_samples(cfg, 70 + s, n)[0] for s in range(len(ids))], axis=1)
    h = create(rift, inp, rift.RIFT_PREC_MIXED)
    rift.rift_ile_set_option(h, rift.RIFT_OPT_TC_CHUNK_MIB, 1)   # raised to 8 batches per SM = 1184 batches = 5.4 segments
    got, sh, _ = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=rift.RIFT_KERNEL_TCS)
    rift.rift_ile_set_option(h, rift.RIFT_OPT_TC_CHUNK_MIB, 4096)
    assert "lnl_tcs" in rift.rift_ile_kernel_name(h)
    one, _, _ = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=rift.RIFT_KERNEL_TC)
    assert "lnl_tc<" in rift.rift_ile_kernel_name(h)
    # the default choice: the sorted variant for calls of >= 32768 samples in segments of >= 100 samples per shift bucket
    gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=rift.RIFT_KERNEL_AUTO)
    assert "lnl_tc<" in rift.rift_ile_kernel_name(h)         # 3533 < 100 * 85
    big = np.tile(params[:, :n], (1, 12))[:, :4 * 9000]
    gpu_eval(torch, h, [0, 1, 2, 0], 9000, big, K=cfg.n_det)
    assert "lnl_tcs" in rift.rift_ile_kernel_name(h)
    rift.rift_ile_set_option(h, rift.RIFT_OPT_TC_SORT, 0)     # the automatic choice can be switched off
    gpu_eval(torch, h, [0, 1, 2, 0], 9000, big, K=cfg.n_det)
    assert "lnl_tc<" in rift.rift_ile_kernel_name(h)
    with pytest.raises(rift.RiftError) as e:
        rift.rift_ile_set_option(h, 99, 1)
    assert e.value.code == rift.RIFT_EINVAL
    got, one = got.cpu().numpy(), one.cpu().numpy()
    assert not np.isnan(got).any()
    assert np.max(np.abs(got - one)) < TOL_MIXED_LNL          # against the unsorted tensor-core kernel, every sample
    for s in (0, 5, 11):                                      # against the oracle, a subsample of three segments
        sel = np.arange(0, n, 7)
        ref = oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n][:, sel])[0]
        assert np.max(np.abs(got[s * n:(s + 1) * n][sel] - ref)) < TOL_MIXED_LNL, s
    rift.rift_ile_destroy(h)


@pytest.mark.parametrize("kernel", KERNELS)
def test_guard_band_window(torch, oracle, kernel):
    """n_tau < n_t (reading A4): the physical mode in which the circular wrap never triggers."""
    cfg = synth.CONFIGS[1]
    inp = build(oracle, cfg, n_points=1)
    n_tau = cfg.n_t - 2 * 88 - 2                              # S_max = 88 at 4096 Hz
    params = synth.draw_samples(cfg, 0, 1500)[0]
    ref = oracle_eval(oracle, inp, 0, params, n_tau=n_tau)[0]
    for prec, tol in ((rift.RIFT_PREC_FP64, None), (rift.RIFT_PREC_MIXED, TOL_MIXED_LNL)):
        h = create(rift, inp, prec, n_tau=n_tau)
        got = gpu_eval(torch, h, [0], 1500, params, K=cfg.n_det, kernel=kernel)[0].cpu().numpy()
        assert ("lnl_tc" in rift.rift_ile_kernel_name(h)) == (
            prec == rift.RIFT_PREC_MIXED and kernel in TC_FAMILY)
        if tol is None:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(got - ref)) < tol
        rift.rift_ile_destroy(h)
    with pytest.raises(rift.RiftError) as e:
        create(rift, inp, rift.RIFT_PREC_FP64, n_tau=cfg.n_t - 100)
    assert e.value.code == rift.RIFT_EWINDOW


# ------------------------------------------------------------------------------------------------ C2 / C4 shapes, reduced
def test_c2_shape_21_modes(torch, oracle):
    cfg = synth.CONFIGS[2]
    inp = build(oracle, cfg, n_points=2)
    n = 1200
    params, ln_w = synth.draw_samples(cfg, 1, n, theta_true=inp.theta_true[1])
    ref = oracle_eval(oracle, inp, 1, params)[0]
    zref = oracle.reduce(ref, ln_w)
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        lnL, _, _ = gpu_eval(torch, h, [1], n, params, K=cfg.n_det)
        got = lnL.cpu().numpy()
        red = rift.rift_ile_reduce(h, 1, n, lnL, dev(torch, ln_w))
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL
            assert abs(red["lnZ"][0] - zref["lnZ"]) < 1e-10 * max(1.0, abs(zref["lnZ"]))
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL
            assert abs(red["lnZ"][0] - zref["lnZ"]) < TOL_MIXED_LNZ
        rift.rift_ile_destroy(h)


def test_quadratic_term_pair_program(torch, oracle):
    """More than 8 modes: the quadratic term a4 (Eq. (D3)) runs the pair program of rift_internal.h (mode pairs grouped by
    their common phase exponent).  With the same contraction, lnL from the program and from the plain double sum over
    mode pairs (RIFT_OPT_QUAD_PROG = 0) differ by the rounding of q only; both match the oracle.  Mode lists in scrambled order
    with gaps in m, two segments whose boundary falls inside a thread block (program image of another point)."""
    modes = ((3, -3), (2, 2), (4, 0), (2, -2), (3, 2), (4, 4), (2, 1), (4, -3), (3, 3), (2, 0), (4, -4))
    cfg = synth.with_overrides(synth.CONFIGS[1], modes=modes, n_points=2)
    inp = build(oracle, cfg, n_points=2)
    n = 333
    ids = [1, 0]
    params = np.concatenate([synth.draw_samples(cfg, 70 + s, n)[0] for s in range(len(ids))], axis=1)
    ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(len(ids))])
    for prec in (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64):
        out = []
        h = create(rift, inp, prec)
        for no_prog in (False, True, False):
            rift.rift_ile_set_option(h, rift.RIFT_OPT_QUAD_PROG, 0 if no_prog else 1)
            got, _, _ = gpu_eval(torch, h, ids, n, params, K=cfg.n_det)
            out.append(got.cpu().numpy())
        rift.rift_ile_destroy(h)
        assert np.array_equal(out[0], out[2])                 # switching the option back restores the program
        assert np.max(rel_err(out[0], out[1])) < 1e-12
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(out[0], ref)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(out[0] - ref)) < TOL_MIXED_LNL


def test_eval_batch_under_cuda_graph(torch, oracle):
    """A steady-state eval_batch (workspace grown, id list already on the device) is kernel launches only, so it can be
    captured into a CUDA graph (bench.py times C0 this way); replays with new sample values in the
    same buffers match the oracle."""
    cfg = synth.CONFIGS[0]
    inp = build(oracle, cfg, n_points=1)
    n = 1000
    p1, _ = synth.draw_samples(cfg, 11, n)
    p2, _ = synth.draw_samples(cfg, 12, n)
    ref2 = oracle_eval(oracle, inp, 0, p2)[0]
    for prec, tol in ((rift.RIFT_PREC_FP64, None), (rift.RIFT_PREC_MIXED, TOL_MIXED_LNL)):
        h = create(rift, inp, prec)
        params_d = dev(torch, p1)
        lnL = torch.empty(n, dtype=torch.float64, device="cuda")
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            rift.rift_ile_eval_batch(h, [0], n, params_d, lnL, None, side.cuda_stream)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            rift.rift_ile_eval_batch(h, [0], n, params_d, lnL, None, torch.cuda.current_stream().cuda_stream)
        params_d.copy_(dev(torch, p2))
        lnL.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        got = lnL.cpu().numpy()
        if tol is None:
            assert np.max(rel_err(got, ref2)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(got - ref2)) < tol
        del g
        rift.rift_ile_destroy(h)


def test_c4_shape_long_window(torch, oracle):
    cfg = synth.CONFIGS[4]
    inp = build(oracle, cfg, n_points=1)
    n = 600
    params, _ = synth.draw_samples(cfg, 0, n)
    ref, sh_ref, fr = oracle_eval(oracle, inp, 0, params)
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        lnL, sh, _ = gpu_eval(torch, h, [0], n, params, K=cfg.n_det)
        got = lnL.cpu().numpy()
        assert np.array_equal(sh.cpu().numpy()[fr == 0], sh_ref[fr == 0])
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL
        rift.rift_ile_destroy(h)


# ------------------------------------------------------------------------------------------------ reduce
def test_reduce_merge_and_degenerate(torch, oracle):
    cfg = synth.CONFIGS[0]
    inp = build(oracle, cfg)
    h = create(rift, inp, rift.RIFT_PREC_FP64)
    rng = np.random.default_rng(3)
    n_seg, n = 3, 40_000
    lnL = 6.0 * rng.standard_normal(n_seg * n)
    lw = 0.4 * rng.standard_normal(n_seg * n)
    params = synth.prior_draw(rng, n_seg * n)
    one = rift.rift_ile_reduce(h, n_seg, n, dev(torch, lnL), dev(torch, lw), dev(torch, params), synth.HIST_LO,
                               synth.HIST_HI, 50, merge=0, want_hist=True)
    for s in range(n_seg):
        sl = slice(s * n, (s + 1) * n)
        ref = oracle.reduce(lnL[sl], lw[sl], params[:, sl], synth.HIST_LO, synth.HIST_HI, 50)
        for key in ("lnZ", "rel_err", "n_eff", "n_ess"):
            assert abs(one[key][s] - ref[key]) < 1e-10 * max(1.0, abs(ref[key])), (s, key)
        assert np.max(np.abs(one["hist"][s] - ref["hist"])) < 1e-12
    # two halves merged == one pass (Eq. (20)-(21)); segments are interleaved halves of the same data
    half = n // 2
    a = np.concatenate([lnL[s * n:s * n + half] for s in range(n_seg)])
    b = np.concatenate([lnL[s * n + half:(s + 1) * n] for s in range(n_seg)])
    wa = np.concatenate([lw[s * n:s * n + half] for s in range(n_seg)])
    wb = np.concatenate([lw[s * n + half:(s + 1) * n] for s in range(n_seg)])
    pa = np.concatenate([params[:, s * n:s * n + half] for s in range(n_seg)], axis=1)
    pb = np.concatenate([params[:, s * n + half:(s + 1) * n] for s in range(n_seg)], axis=1)
    rift.rift_ile_reduce(h, n_seg, half, dev(torch, a), dev(torch, wa), dev(torch, pa), synth.HIST_LO, synth.HIST_HI, 50,
                         merge=0, want_hist=True)
    two = rift.rift_ile_reduce(h, n_seg, half, dev(torch, b), dev(torch, wb), dev(torch, pb), synth.HIST_LO,
                               synth.HIST_HI, 50, merge=1, want_hist=True)
    for key in ("lnZ", "rel_err", "n_eff", "n_ess"):
        assert np.max(np.abs(one[key] - two[key])) < 1e-10 * max(1.0, np.max(np.abs(one[key]))), key
    assert np.max(np.abs(one["hist"] - two["hist"])) < 1e-12
    with pytest.raises(rift.RiftError) as e:
        rift.rift_ile_reduce(h, n_seg + 1, half, dev(torch, np.zeros((n_seg + 1) * half)), merge=1)
    assert e.value.code == rift.RIFT_ESTATE
    # degenerate inputs
    r = rift.rift_ile_reduce(h, 1, 1, dev(torch, np.array([2.5])), dev(torch, np.array([-0.5])))
    assert abs(r["lnZ"][0] - 2.0) < 1e-15 and r["n_eff"][0] == 1.0 and r["rel_err"][0] == 0.0
    r = rift.rift_ile_reduce(h, 1, 4, dev(torch, np.full(4, -np.inf)))
    assert r["lnZ"][0] == -np.inf and r["n_eff"][0] == 0.0
    r = rift.rift_ile_reduce(h, 1, 4, dev(torch, np.array([0.0, np.nan, 1.0, 2.0])))
    assert math.isnan(r["lnZ"][0])
    x = np.array([800.0, 799.0, -800.0, -np.inf])
    r = rift.rift_ile_reduce(h, 1, 4, dev(torch, x))
    assert abs(r["lnZ"][0] - oracle.reduce(x)["lnZ"]) < 1e-12
    rift.rift_ile_destroy(h)


# ------------------------------------------------------------------------------------------------ broad weights, determinism
@pytest.mark.parametrize("config", [0, 1])
def test_reduce_parity_with_broad_weights(torch, oracle, config):
    """At rho = 12 under prior sampling a single sample dominates the evidence (n_eff ~ 1-2), so lnZ parity there is nearly a
    one-sample check.  At rho = 4 (C0; C1 with noise-free data, whose noisy likelihood is spiky at any amplitude) the weights
    are broad (n_eff 50-130, n_ess in the thousands): lnZ, n_eff, n_ess, rel_err and the six weighted histograms of the whole
    path are compared with the oracle's."""
    cfg = synth.with_overrides(synth.CONFIGS[config], rho=4.0, n_points=1, n_samples=200_000)
    inp = build(oracle, cfg, n_points=1, noise=config == 0)
    params, ln_w = synth.draw_samples(cfg, 0)
    ref = oracle_eval(oracle, inp, 0, params)[0]
    rr = oracle.reduce(ref, ln_w, params, synth.HIST_LO, synth.HIST_HI, 100)
    assert rr["n_eff"] > 30.0 and rr["n_ess"] > 500.0, (rr["n_eff"], rr["n_ess"])
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        lnL, _sh, p = gpu_eval(torch, h, [0], cfg.n_samples, params, K=cfg.n_det)
        red = rift.rift_ile_reduce(h, 1, cfg.n_samples, lnL, dev(torch, ln_w), p, synth.HIST_LO, synth.HIST_HI, 100,
                                   merge=0, want_hist=True)
        if prec == rift.RIFT_PREC_FP64:
            assert abs(red["lnZ"][0] - rr["lnZ"]) < 1e-10 * max(1.0, abs(rr["lnZ"]))
            rtol, htol = 1e-8, 1e-10
        else:
            assert abs(red["lnZ"][0] - rr["lnZ"]) < TOL_MIXED_LNZ
            rtol, htol = 2e-3, 2e-4
        for key in ("n_eff", "n_ess", "rel_err"):
            assert abs(red[key][0] - rr[key]) < rtol * abs(rr[key]), (key, red[key][0], rr[key])
        assert np.max(np.abs(red["hist"][0] - rr["hist"])) < htol
        rift.rift_ile_destroy(h)


@pytest.mark.parametrize("case", ["tc", "tcs", "tcs_passes", "mma_resident", "mma_resident_two_groups", "mma_stream", "mma_stream_one_group", "sky",
                                  "sky64"])
def test_repeated_calls_are_bit_identical(torch, oracle, case):
    """The warp-specialised kernels hand data between warps through mbarriers, named barriers, tensor memory and shared
    memory; compute-sanitizer is closed on this pool, so the cheap race detector is determinism: 20 calls on the same inputs
    must return bit-identical lnL (the sorted variant assigns bucket positions by atomics, but no result depends on them)."""
    l234 = tuple((l, m) for l in (2, 3, 4) for m in range(-l, l + 1))
    modes = {"tcs_passes": _L2 + _L3, "mma_stream": l234, "mma_stream_one_group": l234}.get(case, _L2)
    cfg = synth.with_overrides(synth.CONFIGS[1], modes=modes, n_points=2)
    if case == "mma_resident_two_groups":          # a window of 477 samples: three windows no longer fit beside the Q block
        cfg = synth.with_overrides(cfg, t_window=0.058)
    if case == "mma_stream_one_group":             # 465 samples = 472 rows > 448: the streamed shape with one group of 15 warps
        cfg = synth.with_overrides(cfg, t_window=0.0567)
    inp = build(oracle, cfg, n_points=2)
    n, ids = 4099, [1, 0, 1]
    params = np.concatenate([synth.draw_samples(cfg, 90 + s, n)[0] for s in range(len(ids))], axis=1)
    mixed = case in ("tc", "tcs", "tcs_passes", "sky")
    h = create(rift, inp, rift.RIFT_PREC_MIXED if mixed else rift.RIFT_PREC_FP64)
    kernel = {"tc": rift.RIFT_KERNEL_TC, "tcs": rift.RIFT_KERNEL_TCS, "tcs_passes": rift.RIFT_KERNEL_TCS,
              "sky": rift.RIFT_KERNEL_SKY, "sky64": rift.RIFT_KERNEL_SKY}.get(case, rift.RIFT_KERNEL_MMA)
    first = None
    for _ in range(20):
        lnL, _sh, _p = gpu_eval(torch, h, ids, n, params, want_shifts=False, kernel=kernel)
        g = lnL.cpu().numpy()
        if first is None:
            first = g
            name = rift.rift_ile_kernel_name(h)
            want = {"tc": "lnl_tc<f16x3>", "tcs": "lnl_tcs<f16x3>", "tcs_passes": "lnl_tcs<f16x3,passes>",
                    "mma_resident": "lnl_mma<f64,resident>", "mma_resident_two_groups": "lnl_mma<f64,resident>",
                    "mma_stream": "lnl_mma<f64,stream>", "mma_stream_one_group": "lnl_mma<f64,stream>", "sky": "lnl_sky<f16x3>",
                    "sky64": "lnl_sky<f64>"}[case]
            assert name == want, name
            ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(len(ids))])
            if mixed:
                assert np.max(np.abs(g - ref)) < TOL_MIXED_LNL
            else:
                assert np.max(rel_err(g, ref)) < TOL_FP64_REL
        else:
            assert np.array_equal(first.view(np.int64), g.view(np.int64))
    rift.rift_ile_destroy(h)


def test_reserve_presizes_the_workspaces(torch, oracle):
    """rift_ile_reserve: after it, a first eval_batch / reduce of that shape allocates nothing, so it can even be the first
    call inside a CUDA-graph capture once the id list is on the device (a cudaMalloc during capture would fail)."""
    cfg = synth.CONFIGS[1]
    inp = build(oracle, cfg, n_points=2)
    n, ids = 3000, [0, 1]
    params = np.concatenate([synth.draw_samples(cfg, 20 + s, n)[0] for s in range(2)], axis=1)
    ref = np.concatenate([oracle_eval(oracle, inp, ids[s], params[:, s * n:(s + 1) * n])[0] for s in range(2)])
    for prec in (rift.RIFT_PREC_FP64, rift.RIFT_PREC_MIXED):
        h = create(rift, inp, prec)
        rift.rift_ile_reserve(h, 2, n, 100)
        p = dev(torch, params)
        lnL = torch.full((2 * n,), float("nan"), dtype=torch.float64, device="cuda")
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            rift.rift_ile_eval_batch(h, ids, 1, p[:, :2].contiguous(), lnL[:2], None, side.cuda_stream)   # uploads the ids only
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            rift.rift_ile_eval_batch(h, ids, n, p, lnL, None, torch.cuda.current_stream().cuda_stream)
        g.replay()
        torch.cuda.synchronize()
        got = lnL.cpu().numpy()
        if prec == rift.RIFT_PREC_FP64:
            assert np.max(rel_err(got, ref)) < TOL_FP64_REL
        else:
            assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL
        red = rift.rift_ile_reduce(h, 2, n, lnL, None, p, synth.HIST_LO, synth.HIST_HI, 100, merge=0, want_hist=True)
        assert np.all(np.isfinite(red["lnZ"]))
        del g
        with pytest.raises(rift.RiftError):
            rift.rift_ile_reserve(h, 2, n, 5000)
        rift.rift_ile_destroy(h)


# ------------------------------------------------------------------------------------------------ full sizes, sampled
def _full_size_sampled(torch, oracle, cfg, precisions, n_check_points, stride, lnz_points=0, kernel=None,
                       expect_kernel=None):
    """Run a whole config on the GPU (the launch configuration bench.py times: all segments in one eval_batch
    where memory allows) in every precision mode, then compare with the oracle (computed ONCE per checked point): a strided
    subsample of per-sample lnL and shifts on `n_check_points` points, every sample plus lnZ / n_eff / n_ess of the whole
    point on the first `lnz_points` of them ("Parity coverage").  Returns the number of compared
    samples per precision."""
    P = cfg.n_points
    inp = build(oracle, cfg)
    n = cfg.n_samples
    pts = sorted(set(np.linspace(0, P - 1, n_check_points).astype(int).tolist()))
    seg_per_call = max(1, min(P, int(2.5e7 // n)))
    got, red_of, shg, prm, lnw = {}, {}, {}, {}, {}
    for prec in precisions:
        h = create(rift, inp, prec)
        for p0 in range(0, P, seg_per_call):
            ids = list(range(p0, min(P, p0 + seg_per_call)))
            ps, ws = zip(*[synth.draw_samples(cfg, p, theta_true=inp.theta_true[p]) for p in ids])
            params = np.concatenate(ps, axis=1)
            lnL, sh, pdev = gpu_eval(torch, h, ids, n, params, K=cfg.n_det, kernel=kernel)
            if expect_kernel is not None:
                assert expect_kernel[prec] in rift.rift_ile_kernel_name(h), rift.rift_ile_kernel_name(h)
            red = rift.rift_ile_reduce(h, len(ids), n, lnL, dev(torch, np.concatenate(ws)))
            g = lnL.cpu().numpy()
            assert not np.isnan(g).any()
            s_all = sh.cpu().numpy()
            for p in ids:
                if p in pts:
                    o = (p - p0) * n
                    got[prec, p] = g[o:o + n].copy()
                    red_of[prec, p] = {k: red[k][p - p0] for k in ("lnZ", "n_eff", "n_ess", "rel_err")}
                    shg[prec, p] = s_all[o:o + n].copy()
                    prm[p], lnw[p] = ps[p - p0], ws[p - p0]
            del lnL, sh, pdev
        rift.rift_ile_destroy(h)
    compared, fragile = 0, 0
    for p in pts:
        full = p in pts[:lnz_points]
        sel = np.arange(n) if full else np.arange(0, n, stride)
        ref, sh_ref, fr = oracle_eval(oracle, inp, p, prm[p][:, sel])
        ok = fr.sum(axis=1) == 0 if fr.ndim == 2 else fr == 0
        fragile += int((~ok).sum())
        compared += len(sel)
        zr = oracle.reduce(ref, lnw[p]) if full else None
        for prec in precisions:
            assert np.array_equal(shg[prec, p][sel][ok], sh_ref[ok]), (cfg.name, p)
            if prec == rift.RIFT_PREC_FP64:
                assert np.max(rel_err(got[prec, p][sel], ref)) < TOL_FP64_REL, (cfg.name, p)
            else:
                assert np.max(np.abs(got[prec, p][sel] - ref)) < TOL_MIXED_LNL, (cfg.name, p)
            if full:
                r = red_of[prec, p]
                if prec == rift.RIFT_PREC_FP64:
                    assert abs(r["lnZ"] - zr["lnZ"]) < 1e-10 * max(1.0, abs(zr["lnZ"])), (cfg.name, p)
                    assert abs(r["n_eff"] - zr["n_eff"]) < 1e-8 * zr["n_eff"], (cfg.name, p)
                    assert abs(r["n_ess"] - zr["n_ess"]) < 1e-8 * zr["n_ess"], (cfg.name, p)
                else:
                    assert abs(r["lnZ"] - zr["lnZ"]) < TOL_MIXED_LNZ, (cfg.name, p)
                    assert abs(r["n_eff"] - zr["n_eff"]) < 5e-3 * zr["n_eff"], (cfg.name, p)
    # samples whose x + 1/2 lies within 1e-9 of an integer are excluded from the bit-exact shift comparison: SURVEY.md H6
    # expects < 1e-4 such events per config, so more than a couple would mean the exclusion hides a shift bug
    assert fragile <= 2, fragile
    return compared


def test_c1_full_size(torch, oracle):
    # 16 points x 1e5 samples in ONE eval_batch (bench.py's launch); two whole points and a 1/50 subsample elsewhere
    n = _full_size_sampled(torch, oracle, synth.CONFIGS[1], (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64), 4, 50, lnz_points=2,
                           expect_kernel={rift.RIFT_PREC_MIXED: "lnl_tcs", rift.RIFT_PREC_FP64: "lnl_mma<f64,resident>"})
    assert n >= 100_000


@pytest.mark.slow
def test_c2_full_size(torch, oracle):
    # 64 points x 1e6 samples; two whole points (lnZ) and a 1/40 subsample of two more: 2.05e6 compared samples per mode
    n = _full_size_sampled(torch, oracle, synth.CONFIGS[2], (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64), 4, 40, lnz_points=2,
                           expect_kernel={rift.RIFT_PREC_MIXED: "lnl_tcs<f16x3,passes>", rift.RIFT_PREC_FP64: "lnl_mma<f64,stream>"})
    assert n >= 100_000


@pytest.mark.slow
def test_c3_full_size(torch, oracle):
    # 1024 points x 1e5 samples, complex64 (mixed) and complex128 (fp64 mode) storage of Q; two whole points and a 1/10
    # subsample of four more
    n = _full_size_sampled(torch, oracle, synth.CONFIGS[3], (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64), 6, 10, lnz_points=2,
                           expect_kernel={rift.RIFT_PREC_MIXED: "lnl_tcs", rift.RIFT_PREC_FP64: "lnl_mma<f64,resident>"})
    assert n >= 100_000


@pytest.mark.slow
def test_c4_full_size(torch, oracle):
    # 8 points x 4e6 samples, mixed and fp64; a 1/60 subsample of four points (2.7e5 samples) ...
    n = _full_size_sampled(torch, oracle, synth.CONFIGS[4], (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64), 4, 60, lnz_points=0,
                           expect_kernel={rift.RIFT_PREC_MIXED: "lnl_sky<f16x3>", rift.RIFT_PREC_FP64: "lnl_sky<f64>"})
    assert n >= 100_000


@pytest.mark.slow
def test_c4_full_size_lnz(torch, oracle):
    # ... and every sample of two whole points with lnZ / n_eff / n_ess (2.4e12 flop per point on the host: minutes)
    _full_size_sampled(torch, oracle, synth.CONFIGS[4], (rift.RIFT_PREC_MIXED, rift.RIFT_PREC_FP64), 2, 1, lnz_points=2)


# ------------------------------------------------------------------------------------------------ seeded random shapes
@pytest.mark.parametrize("precision", ["fp64", "mixed"])
def test_random_shapes_every_kernel_family(torch, oracle, precision):
    """24 seeded random shapes (1-5 detectors, 1-8 modes, windows of 33-499 samples at 1-4 kHz, circular and guard-band, 1-300
    samples in two segments of different points) through every kernel family that takes them: the row-block counts, wrap
    thresholds, halo sizes and ragged tails that the fixed configs never visit.  fp64: relative 1e-10; mixed: |dlnL| <= 2e-3."""
    rng = np.random.default_rng(20221007 + (0 if precision == "fp64" else 1))
    dets = ("H1", "L1", "V1", "S0", "S1")
    modes = ((2, 2), (2, -2), (2, 1), (2, -1), (2, 0), (3, 3), (3, -3), (3, 2))
    prec = rift.RIFT_PREC_FP64 if precision == "fp64" else rift.RIFT_PREC_MIXED
    kernels = (rift.RIFT_KERNEL_MMA, rift.RIFT_KERNEL_SKY) if precision == "fp64" else (
        rift.RIFT_KERNEL_AUTO, rift.RIFT_KERNEL_TC, rift.RIFT_KERNEL_TCS, rift.RIFT_KERNEL_SKY)
    seen = set()
    for trial in range(24):
        K, M = int(rng.integers(1, 6)), int(rng.integers(1, 9))
        f_s = float(rng.choice([1024.0, 2048.0, 4096.0]))
        cfg = synth.with_overrides(synth.CONFIGS[1], detectors=dets[:K], modes=modes[:M], f_s=f_s,
                                   t_window=int(rng.integers(16, 250)) / f_s, n_points=2)
        inp = build(oracle, cfg, n_points=2)
        n = int(rng.integers(1, 300))
        params = np.concatenate([synth.draw_samples(cfg, 1000 + 2 * trial + s, n)[0] for s in range(2)], axis=1)
        n_tau = None
        if rng.random() < 0.3:
            n_tau = cfg.n_t - 2 * (int(np.ceil(2 * 6.4e6 / 299792458.0 * f_s)) + 2) - 2
            n_tau = n_tau if n_tau >= 8 else None
        h = create(rift, inp, prec, n_tau=n_tau)
        ref = np.concatenate([oracle_eval(oracle, inp, p, params[:, s * n:(s + 1) * n], n_tau=n_tau)[0]
                              for s, p in enumerate((1, 0))])
        for kernel in kernels:
            got = gpu_eval(torch, h, [1, 0], n, params, want_shifts=False, kernel=kernel)[0].cpu().numpy()
            name = rift.rift_ile_kernel_name(h)
            seen.add(name)
            if precision == "fp64":
                assert np.max(rel_err(got, ref)) < TOL_FP64_REL, (trial, K, M, cfg.n_t, n_tau, n, name)
            else:
                assert np.max(np.abs(got - ref)) < TOL_MIXED_LNL, (trial, K, M, cfg.n_t, n_tau, n, name)
        rift.rift_ile_destroy(h)
    want = {"lnl_mma<f64,resident>", "lnl_mma<f64,stream>", "lnl_sky<f64>"} if precision == "fp64" else {
        "lnl_tc<f16x3>", "lnl_tcs<f16x3>", "lnl_sky<f16x3>"}
    assert want <= seen, seen
