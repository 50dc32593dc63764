#!/usr/bin/env python
"""bench.py -- time-marginalised lnL evaluations / second of the ILE factored-likelihood hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config k] [--precision mixed|fp64]

A "step" is one pass of the whole hot path (geometry a1-a5, fused lnL a6-a7, reduce a8) over one batch of synthetic
input.  Without --config the run covers ALL FIVE configs of BASELINE.json in BOTH precision modes (ten rows, `per_config`)
and prints ONE JSON line (rank 0) whose headline `value` / `roofline` / `e2e` / `config.workload` are those of the largest
single-GPU config, C4 (5 detectors, 9 modes, N_t = 3277, 8 intrinsic points x 4e6 samples) in mixed precision, timed over
exactly K steps after W warm-ups; the other rows are timed over fewer steps (stated per row) so that the run ends within
minutes.  N > 1: one process per GPU, every rank runs the same per-GPU workload on its own intrinsic points (no data-path
collective; intrinsic points are independent) -> "scaling": "weak".

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the headline
workload; it is a deliberately slow program, see DESIGN.md section 7.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2210_07912_b200 import synth  # noqa: E402

METRIC = "time-marginalized lnL evals/sec"
UNIT = "evals/s"
HEADLINE = (4, "mixed")                            # the largest single-GPU config of BASELINE.json
N_SM, FP32_LANES, FP64_LANES = 148, 128, 64        # B200: guide unit counts (B200_PROFILING.md, B300_MICROARCH.md)
EVIDENCE = os.path.join(ROOT, "profiles", "r2_roofline_evidence.json")
KERNEL_OVERRIDE = None                             # --kernel (A/B runs of one row): a RIFT_KERNEL_* value


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def roofline_evidence() -> dict:
    """ncu evidence per row, written from the committed `ncu --set full` captures under profiles/ (see profiles/README.md):
    {"C1/mixed": {"kernel": ..., "dram_bytes_per_eval": ..., "binding": ..., "profile": ...}, ...}."""
    try:
        return json.load(open(EVIDENCE))
    except Exception:
        return {}


def pipe_peak_tflops(fp64: bool, sm_mhz: float) -> float:
    """FMA-pipe peak DESIGN.md section 6 derives: SMs x lanes x 2 flop x clock."""
    return N_SM * (FP64_LANES if fp64 else FP32_LANES) * 2 * sm_mhz * 1e6 / 1e12


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.lines, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(index), "-lms", "50"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def window(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.1] or [l for (_t, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
                for nme, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()


def cpu_oracle_rate(cfg, n_points: int, n_per_point: int, repeats: int = 1):
    """Time the oracle as it stands on the host cores: (evals/s, cores, seconds, evals)."""
    import oracle
    oracle.build()
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    inp = synth.build_inputs(cfg, lambda th: oracle.geometry_at(th, loc, resp, cfg.gmst, ml, mm, cfg.delta_t),
                             n_points=n_points)
    samples = [synth.draw_samples(cfg, p, n_per_point, theta_true=inp.theta_true[p]) for p in range(n_points)]
    t0 = time.perf_counter()
    for _ in range(repeats):
        for p in range(n_points):
            lnL, _sh, _fr = oracle.eval_batch(loc, resp, cfg.gmst, ml, mm, cfg.delta_t, synth.D_REF_MPC, inp.Q[p],
                                              inp.U[p], inp.V[p], samples[p][0], want_shifts=False)
            oracle.reduce(lnL, samples[p][1], samples[p][0], synth.HIST_LO, synth.HIST_HI, 100)
    dt = time.perf_counter() - t0
    n = repeats * n_points * n_per_point
    return n / dt, oracle.num_threads(), dt, n


def cpu_baseline(cfg, seconds: float) -> dict:
    """The oracle on a bounded sample of `cfg` sized for about `seconds` of host work (whole path a1-a8)."""
    c1 = synth.with_overrides(cfg, n_points=1)
    r0, cores, _dt0, _n0 = cpu_oracle_rate(c1, 1, max(64, int(2.0e9 / cfg.flop_per_eval())))
    n_big = int(min(max(256, r0 * seconds), 20_000_000))
    r1, cores, dt1, n1 = cpu_oracle_rate(c1, 1, n_big)
    return {"value": r1, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"1 intrinsic point x {n1} samples of {cfg.name}, {dt1:.1f} s (a1-a8)"}


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = synth.CONFIGS[HEADLINE[0] if args.config is None else args.config]
    # bounded sample: every step evaluates n_pts points x n_per samples of the same workload
    n_pts = min(cfg.n_points, 4)
    per_eval_flop = cfg.flop_per_eval()
    n_per = max(256, int(2.0e9 / per_eval_flop / n_pts))       # ~2 GFLOP of oracle work per step
    cpu_oracle_rate(cfg, 1, 64)                                   # build + touch
    times = []
    for i in range(args.warmup + args.steps):
        rate, cores, dt, n = cpu_oracle_rate(cfg, n_pts, n_per)
        if i >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = n_pts * n_per / (ms * 1e-3)
    sample = f"{n_pts} intrinsic points x {n_per} extrinsic samples of {cfg.name} per step (whole path a1-a8)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg.name} (BASELINE.json configs[{cfg.index}]), bounded sample", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def cuda_geometry_fn(rift, torch, cfg, loc, resp, ml, mm):
    """(F, Y, shift) of an extrinsic point from the CUDA geometry kernel (no oracle on the product path)."""
    K, M = cfg.n_det, cfg.n_modes
    z = np.zeros
    h = rift.rift_ile_create(loc, resp, cfg.gmst, ml, mm, 1, 1, cfg.delta_t, 1, synth.D_REF_MPC,
                             z((1, K, M, 1), complex), z((1, K, M, M), complex), z((1, K, M, M), complex))

    def fn(theta):
        p = torch.from_numpy(np.ascontiguousarray(theta, dtype=np.float64).reshape(6, 1)).cuda()
        F = torch.zeros((1, K, 2), dtype=torch.float64, device="cuda")
        Y = torch.zeros((1, M, 2), dtype=torch.float64, device="cuda")
        sh = torch.zeros((1, K), dtype=torch.int32, device="cuda")
        rift.rift_ile_geometry(h, 0, 1, p, F, Y, sh, None, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return (F.cpu().numpy().view(np.complex128)[0, :, 0], Y.cpu().numpy().view(np.complex128)[0, :, 0],
                sh.cpu().numpy()[0])

    return fn, h


class ConfigData:
    """Synthetic inputs of one config on this rank: Q/U/V on the host, samples in pinned host memory and on the device."""

    def __init__(self, rift, torch, cfg, gids, pool):
        self.cfg = cfg
        P, N, K, M = len(gids), cfg.n_samples, cfg.n_det, cfg.n_modes
        self.P, self.N = P, N
        loc, resp = synth.detector_arrays(cfg)
        ml, mm = synth.mode_arrays(cfg)
        self.loc, self.resp, self.ml, self.mm = loc, resp, ml, mm
        # injected points: coefficients F_k Y_lm and integer delays from the CUDA geometry kernel (serial: one small handle)
        gfn, hboot = cuda_geometry_fn(rift, torch, cfg, loc, resp, ml, mm)
        th = [synth.true_point(cfg, pid) for pid in gids]
        geo = [gfn(t) for t in th]
        rift.rift_ile_destroy(hboot)
        # frequency series of every point on the host (seeded recipe), Q / U / V on the device (rift_ile_precompute, NEXT-3)
        hs = np.empty((P, K, M, synth.N_FREQ), dtype=np.complex128)
        ds = np.empty((P, K, synth.N_FREQ), dtype=np.complex128)
        sp0 = [None]
        self.params_h = torch.empty((6, P * N), dtype=torch.float64).pin_memory()
        self.has_w = cfg.proposal != "prior"
        self.lnw_h = torch.empty(P * N, dtype=torch.float64).pin_memory() if self.has_w else None
        pn = self.params_h.numpy()
        wn = self.lnw_h.numpy() if self.has_w else None

        def one(p):                                          # numpy releases the GIL in the heavy parts
            F, Y, shift = geo[p]
            coeff = np.asarray(F).reshape(K, 1) * np.asarray(Y).reshape(1, M)
            sp = synth.make_spectra(cfg, gids[p], coeff, shift, synth.D_REF_MPC / th[p][5])
            hs[p], ds[p] = sp.h, sp.d
            if p == 0:
                sp0[0] = sp
            ps, ws = synth.draw_samples(cfg, gids[p], theta_true=th[p])
            pn[:, p * N:(p + 1) * N] = ps
            if wn is not None:
                wn[p * N:(p + 1) * N] = ws

        list(pool.map(one, range(P)))
        sp = sp0[0]
        h_d, d_d = torch.from_numpy(hs.view(np.float64)).cuda(), torch.from_numpy(ds.view(np.float64)).cuda()
        w_d, f_d = torch.from_numpy(sp.w).cuda(), torch.from_numpy(sp.f).cuda()
        self.Q = torch.empty((P, K, M, cfg.n_t, 2), dtype=torch.float64, device="cuda")
        self.U = torch.empty((P, K, M, M, 2), dtype=torch.float64, device="cuda")
        self.V = torch.empty((P, K, M, M, 2), dtype=torch.float64, device="cuda")
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev[0].record()
        rift.rift_ile_precompute(P, K, M, h_d, d_d, w_d, sp.f, f_d, cfg.n_t, cfg.delta_t, self.Q, self.U, self.V,
                                 torch.cuda.current_stream().cuda_stream)
        ev[1].record()
        torch.cuda.synchronize()
        self.precompute_ms = ev[0].elapsed_time(ev[1])
        del h_d, d_d, hs, ds
        self.params_d = self.params_h.cuda()
        self.lnw_d = self.lnw_h.cuda() if self.has_w else None
        self.lnL_d = torch.empty(P * N, dtype=torch.float64, device="cuda")
        self.lnL_h = torch.empty(P * N, dtype=torch.float64).pin_memory()


def bench_row(rift, torch, dist_util, data: ConfigData, precision: str, steps, warmup, flush, sampler, evidence,
              peaks, world):
    """One (config, precision) row: device-resident steps, the fused kernel's roofline, the host-buffer (e2e) steps.
    steps = None: chosen from a probe step so that the row takes about 3 s."""
    cfg, P, N, K, M = data.cfg, data.P, data.N, data.cfg.n_det, data.cfg.n_modes
    fp64 = precision == "fp64"
    h = rift.rift_ile_create(data.loc, data.resp, cfg.gmst, data.ml, data.mm, P, cfg.n_t, cfg.delta_t, cfg.n_t,
                             synth.D_REF_MPC, data.Q, data.U, data.V, input_mem=rift.RIFT_MEM_DEVICE,
                             precision=rift.RIFT_PREC_FP64 if fp64 else rift.RIFT_PREC_MIXED)
    ids = list(range(P))
    stream = torch.cuda.current_stream().cuda_stream
    n_bins = 100
    if KERNEL_OVERRIDE is not None:
        rift.rift_ile_set_kernel(h, KERNEL_OVERRIDE)
    rift.rift_ile_reserve(h, P, N, n_bins)

    def step_resident():
        rift.rift_ile_eval_batch(h, ids, N, data.params_d, data.lnL_d, None, stream)
        return rift.rift_ile_reduce(h, P, N, data.lnL_d, data.lnw_d, data.params_d, synth.HIST_LO, synth.HIST_HI, n_bins,
                                    merge=0, want_hist=True, cuda_stream=stream)

    def step_e2e():
        # the library's host-buffer call: sliced H2D / evaluate / D2H pipeline, then the reduce on the staged device copies
        rift.rift_ile_eval_batch_host(h, ids, N, data.params_h, data.lnw_h, data.lnL_h, 0, stream)
        st = rift.rift_ile_staged(h)
        return rift.rift_ile_reduce(h, P, N, st["lnL"], st["ln_weight"], st["params"], synth.HIST_LO, synth.HIST_HI, n_bins,
                                    merge=0, want_hist=True, cuda_stream=stream)

    def barrier():
        dist_util.barrier()
        torch.cuda.synchronize()

    def timed(fn, n_steps, n_warm, profile=False):
        for _ in range(n_warm):
            flush.zero_()
            fn()
        barrier()
        if profile:
            rift.rift_ile_profile(h, True)
            rift.rift_ile_profile_read(h)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        l0 = rift.rift_ile_launch_count(h)
        t0 = time.time()
        out = None
        for a, b in ev:
            flush.zero_()                     # L2 flush between timed iterations, outside the event bracket
            a.record()
            out = fn()
            b.record()
        barrier()
        t1 = time.time()
        prof = rift.rift_ile_profile_read(h) if profile else None
        if profile:
            rift.rift_ile_profile(h, False)
        per = sorted(a.elapsed_time(b) for a, b in ev)
        ms = dist_util.max_over_ranks(float(sum(per)), device="cuda") / n_steps
        return dict(ms=ms, best=per[0], median=per[len(per) // 2], launches=rift.rift_ile_launch_count(h) - l0,
                    window=(t0, t1), prof=prof, out=out)

    if steps is None:                         # probe: one untimed step sizes the row
        step_resident()
        torch.cuda.synchronize()
        t = time.time()
        step_resident()
        torch.cuda.synchronize()
        probe_ms = 1e3 * (time.time() - t)
        steps = int(max(2, min(20, 3000.0 / max(probe_ms, 1e-3))))
        warmup = 3 if probe_ms < 1500.0 else 1
    r = timed(step_resident, steps, warmup, profile=True)
    e2e_steps = int(max(2, min(steps, 2500.0 / max(r["ms"], 1e-3))))
    e = timed(step_e2e, e2e_steps, 1 if r["ms"] > 300.0 else 3)
    evals = P * N
    name = rift.rift_ile_kernel_name(h)
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    peak = pipe_peak_tflops(fp64, sm_max)
    prof = r["prof"]
    n_lnl = max(1, prof["launches"][1])
    flop_eval = 4 * K * M * cfg.n_t           # n_tau = n_t in every config (circular window)
    flop_launch = float(flop_eval) * evals * steps / n_lnl
    lnl_ms = prof["ms"][1] / n_lnl
    achieved = flop_launch / (lnl_ms * 1e-3) / 1e12
    micro = rift.rift_ile_fma_peak(1 if fp64 else 0, 8192, stream)
    key = f"C{cfg.index}/{precision}"
    ev = evidence.get(key, {})
    ev_ok = ev.get("kernel") == name          # evidence of another kernel is never attached
    traffic = ev["dram_bytes_per_eval"] * evals * steps / n_lnl if ev_ok and "dram_bytes_per_eval" in ev else None
    tensor = "lnl_tc" in name or "lnl_mma" in name
    row = {
        "evals_per_s": world * evals / (r["ms"] * 1e-3), "ms_per_step": r["ms"], "ms_per_step_best": r["best"],
        "ms_per_step_median": r["median"], "steps": steps, "warmup": warmup, "kernel": name,
        "workload": f"{cfg.name} (BASELINE.json configs[{cfg.index}]): {K} detectors, {M} modes, N_t={cfg.n_t}, "
                    f"{P} intrinsic points x {N} extrinsic samples per GPU",
        "dtype": "f64" if fp64 else "f32 contraction+exp / f64 geometry, quadratic term, reductions",
        "kernel_ms_per_step": {"geometry": prof["ms"][0] / steps, "lnl": prof["ms"][1] / steps, "reduce": prof["ms"][2] / steps},
        "gpu_launches": int(r["launches"]),
        "roofline": {"bound": "alu", "kernel": name, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": traffic, "fma_microbench_tflops": micro,
                     "frac_of_microbench": achieved / micro, "kernel_ms_per_launch": lnl_ms, "flop_per_launch": flop_launch,
                     "flop_per_eval": flop_eval,
                     "binding": ev.get("binding") if ev_ok else None, "profile": ev.get("profile") if ev_ok else None,
                     "peak_source": f"derived: {N_SM} SM x {FP64_LANES if fp64 else FP32_LANES} lanes x 2 x {sm_max:.0f} MHz "
                                    "(MEASURED_PEAKS.json sm_max_mhz); the in-process FMA microbenchmark is beside it",
                     "note": ("algorithmic flop (4 K M N_tau per evaluation) over the fused kernel's time, against the "
                              + ("FP64" if fp64 else "FP32") + " FMA-pipe peak"
                              + ("; the contraction runs on the tensor cores (" + ("DMMA, which shares the FP64 pipe's rate"
                                 if fp64 else "tcgen05, fp16 hi/lo pieces with fp32 accumulation")
                                 + "), so this is an FMA-pipe-equivalent fraction" if tensor else ""))},
        "e2e": {"value": world * evals / (e["ms"] * 1e-3), "unit": UNIT, "ms_per_step": e["ms"], "steps": e2e_steps,
                "h2d_bytes_per_step": int(data.params_h.numel() * 8 + (data.lnw_h.numel() * 8 if data.has_w else 0)),
                "d2h_bytes_per_step": int(data.lnL_h.numel() * 8 + P * (4 + 6 * n_bins) * 8),
                "h2d_gb_per_s": (data.params_h.numel() * 8 + (data.lnw_h.numel() * 8 if data.has_w else 0)) / (e["ms"] * 1e-3) / 1e9,
                "path": "rift_ile_eval_batch_host (4 slices: upload / evaluate / read back overlapped) + rift_ile_reduce"},
        "clocks": sampler.window(*r["window"]) if sampler else None,
        "precompute_ms": data.precompute_ms,      # Q, U, V of all points from their frequency series on the device (NEXT-3)
        "lnZ_point0": float(r["out"]["lnZ"][0]), "n_eff_point0": float(r["out"]["n_eff"][0]),
    }
    if evals <= 65536:
        row["launch_rate"] = launch_rate(rift, torch, h, ids, N, data)
    if cfg.index == 1:                        # NEXT-2: the distance-marginalised evaluation on the same samples (5 parameters)
        row["dmarg"] = dmarg_row(rift, torch, h, ids, N, data, flush, row)
        row["gmm"] = gmm_row(rift, torch, h, data, cfg, row["dmarg"])
    rift.rift_ile_destroy(h)
    return row


def dmarg_row(rift, torch, h, ids, N, data, flush, row, n_dist=128):
    """rift_ile_eval_batch_dmarg: evaluations/s, and the sampling efficiency n_ess per
    evaluation of the 5-D integral against that of the 6-D one on the same intrinsic points."""
    stream = torch.cuda.current_stream().cuda_stream
    P = len(ids)
    lnL = torch.empty_like(data.lnL_d)

    def step():
        rift.rift_ile_eval_batch_dmarg(h, ids, N, data.params_d, synth.D_MIN_MPC, synth.D_MAX_MPC, n_dist, lnL, None, stream)
        return rift.rift_ile_reduce(h, P, N, lnL, data.lnw_d, cuda_stream=stream)

    step()
    torch.cuda.synchronize()
    ms = []
    for _ in range(3):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        red5 = step()
        b.record()
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    red6 = rift.rift_ile_reduce(h, P, N, data.lnL_d, data.lnw_d, cuda_stream=stream)
    t5, t6 = float(np.mean(ms)), row["ms_per_step"]
    e5, e6 = float(np.median(red5["n_ess"])), float(np.median(red6["n_ess"]))
    return {"kernel": rift.rift_ile_kernel_name(h), "n_dist": n_dist, "evals_per_s": P * N / (t5 * 1e-3), "ms_per_step": t5,
            "steps": 3, "cost_ratio_vs_plain": t5 / t6, "median_n_ess_5d": e5, "median_n_ess_6d": e6,
            "n_ess_gain_at_equal_cost": (e5 / t5) / (e6 / t6) if e6 > 0 else None,
            "median_lnZ_5d_minus_6d": float(np.median(red5["lnZ"] - red6["lnZ"]))}


def gmm_row(rift, torch, h, data, cfg, dm, n_per_round=200_000, rounds=8, n_dist=128):
    """the configuration PAPER.md:807 recommends for loud signals on intrinsic point 0 -- GMM
    sampling (rift_gmm.h) in the rotated network-frame sky (rift_sky.h) with distance marginalisation (gmm_loop.integrate) --
    timed as a whole (draws, weights, evaluation, reduce, EM refits), with its effective samples per evaluation next to the
    prior-sampling ones of the dmarg row; plus the sampler kernels alone on 4e6 samples."""
    from paper_2210_07912_b200 import gmm_loop
    stream = torch.cuda.current_stream().cuda_stream
    R = rift.rift_sky_network_frame(data.loc[0], data.loc[1])
    res = None
    ms = []
    for rep in range(2):                      # the first repetition warms up (workspace growth, lazy module load)
        samplers = gmm_loop.create_samplers(n_comp_sky=3, n_comp_1d=1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        res = gmm_loop.integrate(h, samplers, 0, R, cfg.gmst, synth.D_MIN_MPC, synth.D_MAX_MPC, n_dist, n_per_round,
                                 n_eff_target=float("inf"), max_rounds=rounds, seed=11, cuda_stream=stream)
        b.record()
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
        gmm_loop.destroy_samplers(samplers)
    n = 4_000_000
    g = rift.rift_gmm_create(2, 4, [-3.0, -3.0], [3.0, 3.0])
    xs = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(2)]
    lnp = torch.empty(n, dtype=torch.float64, device="cuda")
    rift.rift_gmm_draw(g, n, 1, 0, xs, lnp, cuda_stream=stream)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    ev[0].record()
    for _ in range(10):
        rift.rift_gmm_draw(g, n, 1, 0, xs, lnp, cuda_stream=stream)
    ev[1].record()
    lw = torch.zeros(n, dtype=torch.float64, device="cuda")
    rift.rift_gmm_fit(g, n, xs, lw, 1, cuda_stream=stream)
    ev[2].record()
    it, _ll = rift.rift_gmm_fit(g, n, xs, lw, 10, cuda_stream=stream)
    ev[3].record()
    torch.cuda.synchronize()
    rift.rift_gmm_destroy(g)
    t_draw, t_em = ev[0].elapsed_time(ev[1]) / 10, ev[2].elapsed_time(ev[3]) / max(it, 1)
    return {"loop": "gmm_loop.integrate: GMM (sky pair 3 components, iota 1) + network-frame sky + dmarg, point 0",
            "rounds": res["rounds"], "n_evals": res["n_evals"], "ms_total": ms[-1], "evals_per_s": res["n_evals"] / (ms[-1] * 1e-3),
            "lnZ": res["lnZ"], "rel_err": res["rel_err"], "n_ess": res["n_ess"], "n_ess_per_eval": res["n_ess"] / res["n_evals"],
            "n_ess_per_eval_prior_sampling_5d": dm["median_n_ess_5d"] / (data.N),
            "note": ("n_ess of prior sampling is at its floor of 1 (one sample carries the weight of a point's 1e5 draws), so its "
                     "per-evaluation figure is an upper bound; tests/test_gpu_gmm.py compares at 4e6-1.6e7 prior draws"),
            "draw_samples_per_s": n / (t_draw * 1e-3), "em_iteration_samples_per_s": n / (t_em * 1e-3),
            "draw_ms_4e6": t_draw, "em_iteration_ms_4e6": t_em}


def launch_rate(rift, torch, h, ids, N, data, n_calls=200):
    """a latency-bound workload (C0) is also timed as n_calls eval_batch calls issued back to
    back with no host synchronisation in between, and as replays of one CUDA graph that captured the call."""
    out = {"calls": n_calls}
    stream = torch.cuda.current_stream().cuda_stream
    evals = len(ids) * N
    for _ in range(5):
        rift.rift_ile_eval_batch(h, ids, N, data.params_d, data.lnL_d, None, stream)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n_calls):
        rift.rift_ile_eval_batch(h, ids, N, data.params_d, data.lnL_d, None, stream)
    b.record()
    torch.cuda.synchronize()
    out["back_to_back_us_per_call"] = a.elapsed_time(b) * 1e3 / n_calls
    out["back_to_back_evals_per_s"] = evals / (a.elapsed_time(b) * 1e-3 / n_calls)
    try:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):                     # the id list is cached per stream: upload it before the capture
            rift.rift_ile_eval_batch(h, ids, N, data.params_d, data.lnL_d, None, side.cuda_stream)
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            rift.rift_ile_eval_batch(h, ids, N, data.params_d, data.lnL_d, None, torch.cuda.current_stream().cuda_stream)
        for _ in range(5):
            g.replay()
        torch.cuda.synchronize()
        a.record()
        for _ in range(n_calls):
            g.replay()
        b.record()
        torch.cuda.synchronize()
        out["graph_us_per_call"] = a.elapsed_time(b) * 1e3 / n_calls
        out["graph_evals_per_s"] = evals / (a.elapsed_time(b) * 1e-3 / n_calls)
    except Exception as e:                                # reported, not hidden: the graph leg is optional
        out["graph_error"] = str(e)[:200]
    return out


def run_ours(args) -> None:
    import torch
    import paper_2210_07912_b200 as rift
    from paper_2210_07912_b200 import build as build_mod
    from paper_2210_07912_b200 import dist_util

    rank, world, local = dist_util.env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist_util.init("nccl", torch.device("cuda", local))
    if rank == 0:
        build_mod.build()
    dist_util.barrier()
    rift.lib()

    single = args.config is not None
    rows_wanted = ([(args.config, args.precision or "mixed")] if single else
                   [(c, p) for c in (0, 1, 2, 3, 4) for p in ("mixed", "fp64")])
    headline = rows_wanted[0] if single else HEADLINE
    peaks = measured_peaks()
    evidence = roofline_evidence()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    sampler = ClockSampler(local) if rank == 0 else None
    pool = ThreadPoolExecutor(max_workers=max(2, min(16, (os.cpu_count() or 8))))
    per_config, t_prep = {}, {}
    for ci in sorted({c for c, _ in rows_wanted}):
        cfg = synth.CONFIGS[ci]
        if args.points:
            cfg = synth.with_overrides(cfg, n_points=args.points)
        if args.samples:
            cfg = synth.with_overrides(cfg, n_samples=args.samples)
        gids = dist_util.shard_points(cfg.n_points, rank, world)     # every rank owns its own intrinsic points
        t = time.time()
        data = ConfigData(rift, torch, cfg, gids, pool)
        t_prep[f"C{ci}"] = round(time.time() - t, 2)
        for (c, prec) in rows_wanted:
            if c != ci:
                continue
            is_head = (c, prec) == headline
            row = bench_row(rift, torch, dist_util, data, prec, args.steps if is_head else None,
                            args.warmup if is_head else 3, flush, sampler, evidence, peaks, world)
            per_config[f"C{c}/{prec}"] = row
        del data
        torch.cuda.empty_cache()

    if rank == 0:
        head = per_config[f"C{headline[0]}/{headline[1]}"]
        line = {
            "metric": METRIC, "value": head["evals_per_s"], "unit": UNIT, "n_gpus": world, "steps": head["steps"],
            "warmup": head["warmup"], "ms_per_step": head["ms_per_step"], "ms_per_step_best": head["ms_per_step_best"],
            "ms_per_step_median": head["ms_per_step_median"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": head["dtype"], "data": "synthetic",
            "config": {"workload": head["workload"], "precision": headline[1], "kernel": head["kernel"],
                       "l2": "flushed between timed iterations (256 MiB memset)", "parallelism": f"replicas x{world}",
                       "step": "eval_batch (geometry + fused lnL) + reduce with 6x100-bin histograms",
                       "rows": "per_config holds all five configs x both precision modes; rows other than the headline are "
                               "timed over the `steps` they state"},
            "clocks": head["clocks"], "e2e": head["e2e"], "gpu_launches": head["gpu_launches"],
            "roofline": head["roofline"], "kernel_ms_per_step": head["kernel_ms_per_step"],
            "lnZ_point0": head["lnZ_point0"], "n_eff_point0": head["n_eff_point0"],
            "per_config": per_config, "input_generation_s": t_prep,
        }
        if "launch_rate" in head:
            line["launch_rate"] = head["launch_rate"]
        if world == 1 and not args.no_cpu:
            cfgs = sorted({c for c, _ in rows_wanted})
            base = {c: cpu_baseline(synth.CONFIGS[c], 12.0 if c == headline[0] else 4.0) for c in cfgs}
            line["cpu_baseline"] = base[headline[0]]
            for key, row in per_config.items():
                row["cpu_baseline"] = base[int(key[1])]
        print(json.dumps(line))
    if sampler:
        sampler.stop()
    pool.shutdown()
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=None, help="one config only (default: all five, headline C4 mixed)")
    ap.add_argument("--precision", default=None, choices=[None, "mixed", "fp64"], help="with --config: the precision mode")
    ap.add_argument("--points", type=int, default=0, help="override the number of intrinsic points (debug)")
    ap.add_argument("--samples", type=int, default=0, help="override samples per point (debug)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--kernel", default=None, choices=[None, "auto", "direct", "tc", "tcs", "mma", "sky"],
                    help="force a fused-kernel variant (A/B runs with --config)")
    args = ap.parse_args()
    if args.kernel:
        global KERNEL_OVERRIDE
        KERNEL_OVERRIDE = {"auto": 0, "direct": 1, "tc": 2, "tcs": 3, "mma": 4, "sky": 5}[args.kernel]
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
