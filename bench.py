#!/usr/bin/env python
"""bench.py -- time-marginalised lnL evaluations / second of the ILE factored-likelihood hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--precision mixed|fp64]

A "step" is one pass of the whole hot path (geometry a1-a5, fused lnL a6-a7, reduce a8) over one batch of
synthetic input: BASELINE.json configs[1] (3 detectors, 5 modes, 16 intrinsic points x 1e5 extrinsic samples).
Prints ONE JSON line (rank 0).  N > 1: one process per GPU, every rank runs the same per-GPU workload on its own
intrinsic points (no data-path collective; intrinsic points are independent) -> "scaling": "weak".

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the same
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2210_07912_b200 import synth  # noqa: E402

METRIC = "time-marginalized lnL evals/sec"
UNIT = "evals/s"
N_SM, FP32_LANES, FP64_LANES = 148, 128, 64        # B200: guide unit counts (B200_PROFILING.md, B300_MICROARCH.md)
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the fused kernel from the committed `ncu --set full` captures
# (profiles/), keyed by (kernel, config index); a launch of lnl_tc on C1 = the whole step (1.6e6 evaluations).
NCU_TRAFFIC_BYTES = {("lnl_tcs<f16x3>", 1): 396.7e6, ("lnl_tc<f16x3>", 1): 379.7e6, ("lnl_direct_ext<f32>", 1): 58.5e6}


def measured_peaks() -> dict:
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
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

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
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


def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = synth.CONFIGS[args.config]
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

    cfg = synth.CONFIGS[args.config]
    if args.points:
        cfg = synth.with_overrides(cfg, n_points=args.points)
    if args.samples:
        cfg = synth.with_overrides(cfg, n_samples=args.samples)
    fp64 = args.precision == "fp64"
    prec = rift.RIFT_PREC_FP64 if fp64 else rift.RIFT_PREC_MIXED
    loc, resp = synth.detector_arrays(cfg)
    ml, mm = synth.mode_arrays(cfg)
    gfn, hboot = cuda_geometry_fn(rift, torch, cfg, loc, resp, ml, mm)
    gids = dist_util.shard_points(cfg.n_points, rank, world)     # every rank owns its own intrinsic points
    inp = synth.build_inputs(cfg, gfn, point_ids=gids)
    rift.rift_ile_destroy(hboot)
    P, N, K, M = cfg.n_points, cfg.n_samples, cfg.n_det, cfg.n_modes
    h = rift.rift_ile_create(loc, resp, cfg.gmst, ml, mm, P, cfg.n_t, cfg.delta_t, cfg.n_t, synth.D_REF_MPC,
                             inp.Q, inp.U, inp.V, precision=prec)
    if args.kernel:
        rift.rift_ile_set_kernel(h, {"auto": 0, "direct": 1, "tc": 2, "tcs": 3, "mma": 4}[args.kernel])
    ids = list(range(P))
    ps, ws = zip(*[synth.draw_samples(cfg, gids[p], theta_true=inp.theta_true[p]) for p in ids])
    params_np = np.concatenate(ps, axis=1)
    if args.same_sky:                       # debug: one shift tuple for every sample (upper bound of grouping)
        params_np[0, :] = params_np[0, 0]
        params_np[1, :] = params_np[1, 0]
    params_h = torch.from_numpy(params_np).pin_memory()
    has_w = cfg.proposal != "prior"
    lnw_h = torch.from_numpy(np.concatenate(ws)).pin_memory() if has_w else None
    params_d = params_h.cuda()
    lnw_d = lnw_h.cuda() if has_w else None
    lnL_d = torch.empty(P * N, dtype=torch.float64, device="cuda")
    lnL_h = torch.empty(P * N, dtype=torch.float64).pin_memory()
    stream = torch.cuda.current_stream().cuda_stream
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    n_bins = 100

    def step_resident():
        rift.rift_ile_eval_batch(h, ids, N, params_d, lnL_d, None, stream)
        return rift.rift_ile_reduce(h, P, N, lnL_d, lnw_d, params_d, synth.HIST_LO, synth.HIST_HI, n_bins, merge=0,
                                    want_hist=True, cuda_stream=stream)

    # End to end through the same public calls, host buffers in and out.  The step is pipelined over groups of
    # intrinsic points: a copy stream moves group g+1's samples host->device and a second one group g-1's lnL device->host
    # (the link is full duplex; on one stream the read-backs would queue behind all the uploads) while the compute stream
    # evaluates group g; the reduce runs once over all groups at the end.
    copy_stream = torch.cuda.Stream()
    d2h_stream = torch.cuda.Stream()
    import ctypes
    cudart = ctypes.CDLL("libcudart.so.12")
    n_groups = min(P, int(os.environ.get("RIFT_BENCH_GROUPS", "4")))    # measured on C1: 2 / 4 / 8 / 16 groups -> 7.1 / 7.7 / 7.3 / 6.2e8
    bounds = [(P * i) // n_groups for i in range(n_groups + 1)]

    def step_e2e(pd, wd):
        cur = torch.cuda.current_stream()
        copy_stream.wait_stream(cur)
        h2d = []
        with torch.cuda.stream(copy_stream):
            for gi in range(n_groups):
                a, b = bounds[gi] * N, bounds[gi + 1] * N
                # six rows of the [6][total] arrays in ONE strided DMA (a 2-D slice copy_ would stage through pageable memory)
                rc = cudart.cudaMemcpy2DAsync(ctypes.c_void_p(pd.data_ptr() + 8 * a), ctypes.c_size_t(8 * pd.shape[1]),
                                              ctypes.c_void_p(params_h.data_ptr() + 8 * a), ctypes.c_size_t(8 * params_h.shape[1]),
                                              ctypes.c_size_t(8 * (b - a)), ctypes.c_size_t(6), 1,
                                              ctypes.c_void_p(copy_stream.cuda_stream))
                assert rc == 0, rc
                if has_w:
                    wd[a:b].copy_(lnw_h[a:b], non_blocking=True)
                ev = torch.cuda.Event()
                ev.record(copy_stream)
                h2d.append(ev)
        for gi in range(n_groups):
            a, b = bounds[gi] * N, bounds[gi + 1] * N
            cur.wait_event(h2d[gi])
            rift.rift_ile_eval_batch(h, ids[bounds[gi]:bounds[gi + 1]], N, [pd[d, a:b] for d in range(6)], lnL_d[a:b],
                                     None, stream)
            done = torch.cuda.Event()
            done.record(cur)
            with torch.cuda.stream(d2h_stream):
                d2h_stream.wait_event(done)
                lnL_h[a:b].copy_(lnL_d[a:b], non_blocking=True)
        red = rift.rift_ile_reduce(h, P, N, lnL_d, wd, pd, synth.HIST_LO, synth.HIST_HI, n_bins, merge=0,
                                   want_hist=True, cuda_stream=stream)
        cur.wait_stream(copy_stream)
        cur.wait_stream(d2h_stream)
        return red

    def barrier():
        dist_util.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup, profile=False):
        for _ in range(warmup):
            flush.zero_()
            fn()
        barrier()
        if profile:
            rift.rift_ile_profile(h, True)
            rift.rift_ile_profile_read(h)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        l0 = rift.rift_ile_launch_count(h)
        t0 = time.time()
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
        timed.last = {"best": per[0], "median": per[len(per) // 2]}       # this rank's per-step spread
        ms = dist_util.max_over_ranks(float(sum(per)), device="cuda")
        return ms / steps, rift.rift_ile_launch_count(h) - l0, (t0, t1), prof, out

    def launch_rate(n_calls=200):
        """a latency-bound workload (C0) is also timed as n_calls eval_batch calls issued back to
        back with no host synchronisation in between, and as replays of one CUDA graph that captured the call."""
        out = {"calls": n_calls}
        for _ in range(5):
            rift.rift_ile_eval_batch(h, ids, N, params_d, lnL_d, None, stream)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n_calls):
            rift.rift_ile_eval_batch(h, ids, N, params_d, lnL_d, None, stream)
        b.record()
        torch.cuda.synchronize()
        out["back_to_back_us_per_call"] = a.elapsed_time(b) * 1e3 / n_calls
        out["back_to_back_evals_per_s"] = P * N / (a.elapsed_time(b) * 1e-3 / n_calls)
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):                     # the id list is cached per stream: upload it before the capture
                rift.rift_ile_eval_batch(h, ids, N, params_d, lnL_d, None, side.cuda_stream)
            side.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                rift.rift_ile_eval_batch(h, ids, N, params_d, lnL_d, None, torch.cuda.current_stream().cuda_stream)
            for _ in range(5):
                g.replay()
            torch.cuda.synchronize()
            a.record()
            for _ in range(n_calls):
                g.replay()
            b.record()
            torch.cuda.synchronize()
            out["graph_us_per_call"] = a.elapsed_time(b) * 1e3 / n_calls
            out["graph_evals_per_s"] = P * N / (a.elapsed_time(b) * 1e-3 / n_calls)
        except Exception as e:                                # reported, not hidden: the graph leg is optional
            out["graph_error"] = str(e)[:200]
        return out

    sampler = ClockSampler(local) if rank == 0 else None
    ms_step, launches, (t0, t1), prof, red = timed(step_resident, args.steps, args.warmup, profile=True)
    spread = dict(timed.last)
    clocks = sampler.stop(t0, t1) if sampler else None
    pd, wd = torch.empty_like(params_d), (torch.empty_like(lnw_d) if has_w else None)
    ms_e2e, _l, _t, _p, _r = timed(lambda: step_e2e(pd, wd), args.steps, args.warmup)
    evals = P * N
    latency = launch_rate() if evals <= 65536 else None        # after every timed leg: it does not touch their numbers
    value = world * evals / (ms_step * 1e-3)
    e2e_value = world * evals / (ms_e2e * 1e-3)

    if rank == 0:
        peaks = measured_peaks()
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        peak = pipe_peak_tflops(fp64, sm_max)
        flop_launch = 4.0 * K * M * cfg.n_t * evals / max(1, prof["launches"][1] // args.steps)
        lnl_ms = prof["ms"][1] / max(1, prof["launches"][1])
        achieved = flop_launch / (lnl_ms * 1e-3) / 1e12
        micro = rift.rift_ile_fma_peak(fp64, 8192, stream)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "ms_per_step_best": spread["best"],
            "ms_per_step_median": spread["median"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if fp64 else "f32 contraction+exp / f64 geometry, quadratic term, reductions",
            "data": "synthetic",
            "config": {"workload": f"{cfg.name} (BASELINE.json configs[{cfg.index}]): {K} detectors, {M} modes, "
                                   f"N_t={cfg.n_t}, {P} intrinsic points x {N} extrinsic samples per GPU",
                       "precision": args.precision, "kernel": rift.rift_ile_kernel_name(h),
                       "l2": "flushed between timed iterations (256 MiB memset)", "parallelism": f"replicas x{world}",
                       "step": "eval_batch (geometry + fused lnL) + reduce with 6x100-bin histograms"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": ms_e2e,
                    "h2d_bytes_per_step": int(params_h.numel() * 8 + (lnw_h.numel() * 8 if has_w else 0)),
                    "d2h_bytes_per_step": int(lnL_h.numel() * 8 + P * (4 + 6 * n_bins) * 8)},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "kernel": rift.rift_ile_kernel_name(h), "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC_BYTES.get((rift.rift_ile_kernel_name(h), cfg.index)),
                         "note": ("algorithmic FP32 flop (4 K M N_tau per evaluation) over the fused kernel's time, against the "
                                  "FP32 FMA-pipe peak; lnl_tc runs the contraction on the tensor pipe (fp16 hi/lo pieces, fp32 "
                                  "accumulate), so this is an FMA-pipe-equivalent fraction"
                                  if "lnl_tc" in rift.rift_ile_kernel_name(h) else
                                  "algorithmic flop (4 K M N_tau per evaluation) over the fused kernel's time"),
                         "peak_source": f"derived: {N_SM} SM x {FP64_LANES if fp64 else FP32_LANES} lanes x 2 x "
                                        f"{sm_max:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz)",
                         "fma_microbench_tflops": micro, "frac_of_microbench": achieved / micro,
                         "kernel_ms_per_launch": lnl_ms, "flop_per_launch": flop_launch,
                         "flop_per_eval": 4 * K * M * cfg.n_t},
            "kernel_ms_per_step": {"geometry": prof["ms"][0] / args.steps, "lnl": prof["ms"][1] / args.steps,
                                   "reduce": prof["ms"][2] / args.steps, "group_sort": prof["ms"][3] / args.steps},
            "lnZ_point0": float(red["lnZ"][0]), "n_eff_point0": float(red["n_eff"][0]),
        }
        if latency is not None:
            line["launch_rate"] = latency
        if world == 1 and not args.no_cpu:
            c1 = synth.with_overrides(cfg, n_points=1)
            r0, cores, dt0, n0 = cpu_oracle_rate(c1, 1, 4000)
            n_big = int(min(max(4000, r0 * 12.0), 20_000_000))
            r1, cores, dt1, n1 = cpu_oracle_rate(c1, 1, n_big)
            if dt1 < 8.0:                                   # the cold first estimate was low: one refinement
                r1, cores, dt1, n1 = cpu_oracle_rate(c1, 1, int(min(r1 * 12.0, 20_000_000)))
            line["cpu_baseline"] = {"value": r1, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"1 intrinsic point x {n1} samples of {cfg.name}, {dt1:.1f} s (a1-a8)"}
        print(json.dumps(line))
    rift.rift_ile_destroy(h)
    if world > 1:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--precision", default="mixed", choices=["mixed", "fp64"])
    ap.add_argument("--kernel", default=None, choices=[None, "auto", "direct", "tc", "tcs", "mma"])
    ap.add_argument("--points", type=int, default=0, help="override the number of intrinsic points (debug)")
    ap.add_argument("--samples", type=int, default=0, help="override samples per point (debug)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--same-sky", action="store_true", help="debug: every sample at one sky position")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
