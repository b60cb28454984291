#!/usr/bin/env python
"""bench.py -- frames/s of the 1D azimuthal-integration hot path on B200 (BASELINE.json metric, configs[1]).

A step is one pass of the whole per-frame hot path (cast + corrections + SpMV + ratio)
through the C ABI (`ai_integrate1d`) on one synthetic 2048x2048 float32 gold-ring frame, 1000 bins in r (mm).
Everything is resident in HBM when the timed region starts.  Matrix + frame (70 MB) would stay in the 126 MB L2
from one step to the next, so the timed steps cycle through REPLICAS contexts (each owns its own copy of the matrix)
and POOL frames: ~700 MB of inputs, five times the L2, touched round-robin -- every step reads its matrix and its
frame from HBM.  The K steps are enqueued back to back on one stream and timed as a whole with one pair of CUDA
events (a pair of events around a single 20 us step costs ~6 us by itself on this box; `extras` reports that
protocol, with an explicit L2 flush before every step, next to the headline).  With N > 1 every rank runs an
independent replica (frames are independent) and the job time is the max over ranks.

    python bench.py [--gpus N] [--steps K] [--warmup W]                 our arm
    python bench.py --impl reference [--steps K] [--warmup W]          the CPU oracle, timed on the host cores

Prints ONE JSON line (rank 0).  See DESIGN.md section 7 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1412_6367_b200 import dist, workloads as W  # noqa: E402

METRIC = "frames_per_s_2048x2048_1d_integration"
WORKLOAD = "cfg2: 2048x2048 float32 gold-ring frame, pixel 1e-4 m, D 0.1 m, centre (1024,1024), r (mm), 1000 bins, bbox-split CSR"
L2_FLUSH_BYTES = 256 << 20
POOL = 16                      # distinct frames rotated through the steps
REPLICAS = 6                   # contexts (matrix copies) rotated through the steps: working set >> L2
# dram__bytes_read.sum + dram__bytes_write.sum of one stage-1 launch on this workload, from the committed capture
NCU_TRAFFIC_BYTES = 72323328
NCU_TRAFFIC_SOURCE = "profiles/r01_v9_ncu_full_stream_cfg2.txt (ncu --set full, one launch: 71.27 MB read + 1.05 MB written)"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def algorithmic_bytes(cfg, nnz, corrections=False):
    """north_star's byte count per frame: image + mask/correction arrays + CSR coef/index/indptr + output."""
    esz = 2 if cfg.dtype in ("uint16", "int16") else 4
    b = cfg.npix * esz + nnz * 8 + (cfg.npt + 1) * 4 + 3 * cfg.npt * 4
    if corrections:
        b += 4 * cfg.npix * 4 + cfg.npix
    return b


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed regions (B200_PROFILING.md clocks line)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            text, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            text, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in text.splitlines():
            p = [x.strip() for x in line.split(",")]
            if len(p) < 8:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1]))
            except ValueError:
                continue
            for n, v in zip(names, p[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm),
                       sm_mhz_max_seen=max(sm))
        return out


# ----------------------------------------------------------------------------------------------------------------------
# CPU oracle legs
# ----------------------------------------------------------------------------------------------------------------------
def time_oracle(cfg, image, budget_s=12.0, rows=None):
    """Per-frame integrate of the oracle (O4-O7 forward scatter over precomputed bounds) on the host cores.
    Returns dict(value frames/s, cores, single_thread, ms_per_frame, sample)."""
    from oracle import oracle as O
    umin, umax = O.pixel_bounds(cfg)
    u0, u1 = O.auto_range(umin, umax)
    img = np.ascontiguousarray(image, dtype=np.float64).ravel()
    if rows is not None:
        n = rows * cfg.width
        umin, umax, img = umin[:n].copy(), umax[:n].copy(), img[:n].copy()
    frac = 1.0 if rows is None else rows / cfg.height
    ncores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else O.num_threads_available()
    res = {}
    for nt in sorted({1, ncores}):
        O.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, nthreads=nt)       # warm-up
        ts, t_end = [], time.perf_counter() + budget_s / 2
        while len(ts) < 5 or (time.perf_counter() < t_end and len(ts) < 40):
            t0 = time.perf_counter()
            O.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, nthreads=nt)
            ts.append(time.perf_counter() - t0)
        res[nt] = statistics.median(ts)
    best = min(res, key=res.get)
    return {"value": frac / res[best], "unit": "frames/s", "cores": best, "kind": "oracle",
            "sample": (f"median of >=5 per-frame integrate calls (O4-O7 over precomputed bounds) on "
                       f"{'the whole frame' if rows is None else f'{rows} of {cfg.height} image rows'} of {cfg.name}; "
                       f"threads tried: {sorted(res)}"),
            "ms_per_frame": {str(k): v * 1e3 / frac for k, v in res.items()}, "host_cores": ncores}


def run_reference(args):
    rank, _, world = dist.env_world()
    if rank != 0:
        return 0
    cfg = W.CONFIGS["cfg2"]
    from oracle import oracle as O
    fr = W.make_frame(cfg)
    umin, umax = O.pixel_bounds(cfg)
    u0, u1 = O.auto_range(umin, umax)
    img = np.ascontiguousarray(fr.image, dtype=np.float64).ravel()
    ncores = len(os.sched_getaffinity(0))
    # choose the faster thread count on one whole frame, then size the per-step sample so the run ends in minutes
    t = {}
    for nt in sorted({1, ncores}):
        O.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, nthreads=nt)
        t0 = time.perf_counter()
        O.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, nthreads=nt)
        t[nt] = time.perf_counter() - t0
    nt = min(t, key=t.get)
    total = args.steps + args.warmup
    rows = int(min(cfg.height, max(8, cfg.height * 120.0 / max(total * t[nt], 1e-9))))
    n = rows * cfg.width
    a, b, c = umin[:n].copy(), umax[:n].copy(), img[:n].copy()
    for _ in range(args.warmup):
        O.integrate1d_bounds(a, b, cfg.npt, u0, u1, c, nthreads=nt)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.integrate1d_bounds(a, b, cfg.npt, u0, u1, c, nthreads=nt)
    dt = time.perf_counter() - t0
    fps = args.steps * (rows / cfg.height) / dt
    sample = f"each step = the first {rows} of {cfg.height} image rows of one cfg2 frame (O4-O7 over precomputed bounds), {nt} thread(s)"
    line = {"impl": "reference", "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": sample}, "mpix_per_s": fps * cfg.npix / 1e6,
            "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": nt, "kind": "oracle", "sample": sample},
            "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------------------------
class Flusher:
    def __init__(self, torch):
        self.torch = torch
        n = L2_FLUSH_BYTES // 4
        self.w = torch.empty(n, dtype=torch.float32, device="cuda")
        self.r = torch.ones(n, dtype=torch.float32, device="cuda")
        self.sink = torch.zeros(1, dtype=torch.float32, device="cuda")

    def __call__(self):
        self.w.zero_()                       # write a buffer larger than L2 ...
        self.sink += self.r.sum()            # ... then read another one: L2 now holds clean unrelated lines


def timed_steps(torch, B, integ, frames_dev, corr, steps, warmup, flush, profile=True):
    """Returns (total_ms, kernel_ms list, launches).  One ai_integrate1d per step, events around each step."""
    out = integ.outputs()
    if profile:
        B.ai_profile_enable(integ.ctx, True)
    for k in range(warmup):
        if flush:
            flush()
        integ.integrate1d(frames_dev[k % len(frames_dev)], *corr, out=out)
    torch.cuda.synchronize()
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    stops = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    kernel_ms, launches = [], 0
    for k in range(steps):
        if flush:
            flush()
        starts[k].record()
        integ.integrate1d(frames_dev[k % len(frames_dev)], *corr, out=out)
        stops[k].record()
        launches += B.ai_last_launch_count(integ.ctx)
        if profile:
            kernel_ms.append(B.ai_profile_last(integ.ctx))
    torch.cuda.synchronize()
    total = sum(s.elapsed_time(e) for s, e in zip(starts, stops))
    if profile:
        B.ai_profile_enable(integ.ctx, False)
    return total, kernel_ms, launches


def timed_train(torch, B, integs, frames_dev, corr, steps, warmup, stage1_only=False):
    """K steps enqueued back to back, step k on context k % len(integs) and frame k % len(frames_dev); one event pair
    around the whole train.  Returns (total_ms, launches).  stage1_only: only the dominant kernel of every step."""
    outs = [it.outputs() for it in integs]
    for it in integs:
        B.ai_profile_enable(it.ctx, 2 if stage1_only else 0)
    launches = 0
    # every context runs at least twice before the timed region (its first call allocates its scratch buffers)
    warmup = max(warmup, 2 * len(integs))
    for k in range(warmup):
        integs[k % len(integs)].integrate1d(frames_dev[k % len(frames_dev)], *corr, out=outs[k % len(integs)])
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(steps):
        j = (k + warmup) % len(integs)
        integs[j].integrate1d(frames_dev[(k + warmup) % len(frames_dev)], *corr, out=outs[j])
        launches += B.ai_last_launch_count(integs[j].ctx)
    e1.record()
    torch.cuda.synchronize()
    for it in integs:
        B.ai_profile_enable(it.ctx, 0)
    return e0.elapsed_time(e1), launches


def back_to_back(torch, integ, frames_dev, corr, calls, warmup=20):
    """Steady-state streaming: no flush, one event pair around `calls` back-to-back calls on rotating frames."""
    out = integ.outputs()
    for k in range(warmup):
        integ.integrate1d(frames_dev[k % len(frames_dev)], *corr, out=out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(calls):
        integ.integrate1d(frames_dev[k % len(frames_dev)], *corr, out=out)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def run_ours(args):
    import torch
    from paper_1412_6367_b200 import binding as B

    rank, local_rank, world = dist.init()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    if rank == 0:
        from paper_1412_6367_b200 import build as cuda_build
        cuda_build.build()                       # no-op when libazint.so is newer than its sources
    dist.barrier()
    B.lib()
    peak_gbs, peak_src = measured_peaks()
    cfg = W.CONFIGS["cfg2"]

    # ---- inputs: POOL distinct seeded frames per rank, generated on the host, resident in HBM before timing -----------
    host_frames = [W.make_frame(cfg, frame_index=(0 if (rank == 0 and k == 0) else 100 * rank + k)).image
                   for k in range(POOL)]
    frames_dev = [torch.from_numpy(f).cuda() for f in host_frames]
    none5 = (None, None, None, None, None)
    integs = [B.Integrator(cfg) for _ in range(REPLICAS)]
    integ = integs[0]
    nnz = B.ai_get_csr(integ.ctx)[3]
    alg_bytes = algorithmic_bytes(cfg, nnz)
    flush = Flusher(torch)

    sampler = ClockSampler(torch.cuda.current_device()) if rank == 0 else None
    dist.barrier()
    torch.cuda.synchronize()
    # headline: a train of K whole steps (stage 1 + stage 2), every step on inputs that are not in L2
    total_ms, launches = timed_train(torch, B, integs, frames_dev, none5, args.steps, args.warmup)
    torch.cuda.synchronize()
    dist.barrier()
    fps, job_ms = dist.aggregate_throughput(args.steps, total_ms)
    ms_per_step = job_ms / args.steps
    # roofline: the same train with only the dominant kernel (stage 1, the SpMV) launched
    k_total_ms, _ = timed_train(torch, B, integs, frames_dev, none5, args.steps, args.warmup, stage1_only=True)
    kernel_ms = [k_total_ms / args.steps]
    k_steps = args.steps
    # ---- end to end through the host entry point for a stream of frames: every frame is copied from pinned host
    # memory inside the timed region (the upload of frame k+1 overlaps the kernel of frame k) and its three profiles
    # are copied back to the host
    E2E_BLOCK = 8
    pinned = torch.from_numpy(np.stack(host_frames[:E2E_BLOCK])).pin_memory()
    outs = [torch.empty((E2E_BLOCK, cfg.npt), dtype=torch.float32).pin_memory() for _ in range(3)]
    e2e_calls = max(2, min(args.steps, 200) // E2E_BLOCK)
    e2e_steps = e2e_calls * E2E_BLOCK

    def e2e_call():
        B.ai_integrate1d_host_frames(integ.ctx, pinned.numpy(), E2E_BLOCK, cfg.npix, *none5, *[o.numpy() for o in outs])

    e2e_call()
    torch.cuda.synchronize()
    dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(e2e_calls):
        e2e_call()
    e1.record()
    torch.cuda.synchronize()
    e2e_fps, _ = dist.aggregate_throughput(e2e_steps, e0.elapsed_time(e1))
    # the one-frame synchronous call, for reference
    one = [torch.empty(cfg.npt, dtype=torch.float32).pin_memory() for _ in range(3)]
    t0 = time.perf_counter()
    for k in range(20):
        B.ai_integrate1d_host(integ.ctx, pinned[k % E2E_BLOCK].numpy(), *none5, *[o.numpy() for o in one], dtype=B.AI_F32)
    torch.cuda.synchronize()
    e2e_single_fps = 20 / (time.perf_counter() - t0)

    extras = {}
    if world == 1 and not args.no_extras:
        extras = run_extras(torch, B, integ, cfg, frames_dev, flush, peak_gbs, args)
    clocks = sampler.stop() if sampler else None

    if rank != 0:
        dist.finalize()
        return 0

    k_ms = statistics.mean(kernel_ms)
    achieved = alg_bytes / (k_ms * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": fps, "unit": "frames/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD, "layout": "tiled", "accum": "f32_kahan", "frames_in_rotation": POOL,
                   "matrix_replicas_in_rotation": REPLICAS,
                   "warmup_steps_run": max(args.warmup, 2 * REPLICAS),
                   "l2": f"inputs larger than L2: {REPLICAS} copies of the matrix and {POOL} frames "
                         f"({(REPLICAS * 53.6 + POOL * 16.8):.0f} MB) touched round-robin, no flush kernels; steps "
                         "enqueued back to back, one event pair around the K steps",
                   "parallelism": f"{world} independent replica(s)"},
        "mpix_per_s": fps * cfg.npix / 1e6,
        "clocks": clocks,
        "e2e": {"value": e2e_fps, "unit": "frames/s", "h2d_bytes_per_step": cfg.npix * 4,
                "d2h_bytes_per_step": 3 * cfg.npt * 4, "steps": e2e_steps,
                "api": f"ai_integrate1d_host_frames, {E2E_BLOCK} pinned host frames per call (double-buffered upload), "
                       "3 pinned host profiles per frame out",
                "single_frame_synchronous_call_fps": e2e_single_fps},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak_gbs, "unit": "GB/s",
                     "frac": achieved / peak_gbs, "traffic": NCU_TRAFFIC_BYTES,
                     "traffic_GBps": NCU_TRAFFIC_BYTES / (k_ms * 1e-3) / 1e9, "kernel": "tiled_stream_kernel",
                     "kernel_time_steps": k_steps, "traffic_source": NCU_TRAFFIC_SOURCE,
                     "kernel_ms": k_ms, "kernel_timing": "one event pair around a train of stage-1-only launches "
                     "(ai_profile_enable(ctx, 2)) on the same rotation of inputs", "algorithmic_bytes": alg_bytes,
                     "peak_source": peak_src, "frac_of_8TBs_nominal": achieved / 8000.0,
                     "whole_step_achieved": alg_bytes / (ms_per_step * 1e-3) / 1e9},
    }
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = time_oracle(cfg, host_frames[0], budget_s=args.cpu_budget)
    else:
        line["cpu_baseline"] = None
    if extras:
        line["extras"] = extras
    print(json.dumps(line))
    dist.finalize()
    return 0


def run_extras(torch, B, integ, cfg, frames_dev, flush, peak_gbs, args):
    """Context numbers beside the headline (N = 1 only): steady-state streaming, latency, the paper's own layouts, the
    accumulator choices, the corrected and the batched paths.  Each is small; none feeds `value`."""
    none5 = (None, None, None, None, None)
    ex = {}
    nnz = B.ai_get_csr(integ.ctx)[3]
    ab = algorithmic_bytes(cfg, nnz)
    n = max(50, min(args.steps, 500))
    # steady state: matrix stays in L2, frames rotate
    ms = back_to_back(torch, integ, frames_dev, none5, 2000)
    ex["warm_back_to_back"] = {"frames_per_s": 2000 / (ms * 1e-3), "algorithmic_GBps": ab * 2000 / (ms * 1e-3) / 1e9,
                               "note": "no L2 flush, 16 frames rotating, matrix L2-resident"}
    # the other protocol: L2 flushed before every step, one event pair per step (and the library's events around
    # stage 1); the cost of an event pair around a trivial kernel after the same flush is reported beside it
    tot, _, _ = timed_steps(torch, B, integ, frames_dev, none5, n, 3, flush, profile=False)
    x = torch.zeros(32, device="cuda")
    ov = []
    for _ in range(30):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); x.add_(1); e1.record()
        torch.cuda.synchronize()
        ov.append(e0.elapsed_time(e1))
    ex["flushed_per_step_events"] = {"frames_per_s": n / (tot * 1e-3), "ms_per_step": tot / n,
                                     "event_pair_around_trivial_kernel_ms": statistics.median(ov),
                                     "note": "256 MiB written + 256 MiB read before every step; events around each step"}
    # the paper's own layouts and the other accumulators, cold (same flushed protocol, library events around the kernel)
    for lname, layout in (("tiled", B.AI_LAYOUT_TILED), ("csr", B.AI_LAYOUT_CSR), ("lut", B.AI_LAYOUT_LUT)):
        for aname, acc in (("kahan", B.AI_ACC_F32_KAHAN), ("f64", B.AI_ACC_F64), ("plain", B.AI_ACC_F32_PLAIN)):
            if lname != "tiled" and aname != "kahan":
                continue
            integ.set_options(layout, acc)
            steps = n if lname != "lut" else 20
            tot, kms, _ = timed_steps(torch, B, integ, frames_dev, none5, steps, 3, flush)
            k = statistics.mean(kms)
            ex[f"cold_{lname}_{aname}"] = {"frames_per_s": steps / (tot * 1e-3), "kernel_ms": k,
                                           "algorithmic_GBps": ab / (k * 1e-3) / 1e9,
                                           "frac_of_peak": ab / (k * 1e-3) / 1e9 / peak_gbs}
    integ.set_options()
    # configs[2] (full preprocessing, q, 3000 bins) and configs[4] (4096^2, 5000 bins): the same train protocol as the
    # headline -- 3 contexts and 4 frames in rotation (> L2), one event pair around the train, whole steps
    for name in ("cfg3", "cfg5"):
        c = W.CONFIGS[name]
        fr = W.make_frame(c)
        its = [B.Integrator(c) for _ in range(3)]
        fdev = [torch.from_numpy(fr.image).cuda() for _ in range(4)]
        corr = tuple(None if a is None else torch.from_numpy(a).cuda()
                     for a in (fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask))
        ab_c = algorithmic_bytes(c, B.ai_get_csr(its[0].ctx)[3], corrections=c.corrections)
        steps = max(20, n // 2)
        tot, launches = timed_train(torch, B, its, fdev, corr, steps, 6)
        ms = tot / steps
        ex[f"train_{name}_tiled_kahan"] = {"frames_per_s": 1e3 / ms, "ms_per_step": ms, "launches_per_step": launches / steps,
                                           "algorithmic_bytes": ab_c, "algorithmic_GBps": ab_c / (ms * 1e-3) / 1e9,
                                           "frac_of_peak": ab_c / (ms * 1e-3) / 1e9 / peak_gbs,
                                           "layout": B.ai_get_layout_info(its[0].ctx)}
        for it in its:
            it.close()
        del corr, fdev
    # context (SURVEY.md section 8(d) "T3"): the frame shape of the paper's Table 3 (Pilatus 1M, 981 x 1043 int32,
    # PAPER.md:257) -- geometry is a reading (centre of the image, 172 um pixels, 0.1 m, 1000 bins in 2theta)
    cp = W.tiny_config(981, 1043, center_x=521.5, center_y=490.5, unit=W.TTH_DEG, npt=1000, pixel_m=172e-6,
                       distance_m=0.1, name="pilatus1m")
    rngp = np.random.default_rng(14126367 + 9)
    fp = [torch.from_numpy(rngp.poisson(30.0, size=(cp.height, cp.width)).astype(np.int32)).cuda() for _ in range(4)]
    its = [B.Integrator(cp) for _ in range(6)]
    tot, launches = timed_train(torch, B, its, fp, none5, 200, 10)
    ex["pilatus1m_int32_table3_shape"] = {"frames_per_s": 200 / (tot * 1e-3), "ms_per_step": tot / 200,
                                          "launches_per_step": launches / 200,
                                          "paper_table3": "integrate kernel 0.384 ms, OpenCL total 1.445 ms, Python call "
                                                          "2.030 ms on a GeForce Titan (PAPER.md:244-257): context, "
                                                          "other hardware",
                                          "note": "width 1043 is not a multiple of 4 (rows off 16-byte boundaries): the "
                                                  "pre-pass casts and re-pitches the frame, then the single-frame kernel"}
    for it in its:
        it.close()
    # the headline workload through the batched entry point: 64 frames of cfg2 (1.07 GB > L2) in one call, the
    # matrix read once per chunk of frames (north_star: "batched path reported the same way")
    nb = 64
    fb = torch.stack([frames_dev[k % len(frames_dev)] for k in range(nb)])
    outb = integ.outputs(nb)
    for _ in range(2):
        integ.integrate1d_batch(fb, out=outb)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(5):
        integ.integrate1d_batch(fb, out=outb)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 5
    abb = nb * cfg.npix * 4 + nnz * 8 + (cfg.npt + 1) * 4 + nb * 3 * cfg.npt * 4
    ex["batch_cfg2_64_frames"] = {"frames_per_s": nb / (ms * 1e-3), "ms_per_batch": ms, "us_per_frame": ms * 1e3 / nb,
                                  "mpix_per_s": nb * cfg.npix / (ms * 1e-3) / 1e6,
                                  "algorithmic_bytes": abb, "algorithmic_GBps": abb / (ms * 1e-3) / 1e9,
                                  "frac_of_peak": abb / (ms * 1e-3) / 1e9 / peak_gbs,
                                  "kernel": "tiled_bstream_kernel (two frames per pass) + tiled_stage2_kernel",
                                  "note": "ai_integrate1d_batch on 64 device-resident cfg2 frames; results are bit-identical "
                                          "to the single-frame kernel's"}
    del fb, outb
    # configs[3]: 1024 int32 frames of 1024x1024 in one batched call
    c4 = W.CONFIGS["cfg4"]
    pool = torch.from_numpy(W.make_frames(c4, 8)).cuda()
    frames = pool.repeat(c4.nframes // 8, 1, 1)
    it = B.Integrator(c4)
    out = it.outputs(c4.nframes)
    for _ in range(2):
        it.integrate1d_batch(frames, out=out)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        it.integrate1d_batch(frames, out=out)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    nnz4 = B.ai_get_csr(it.ctx)[3]
    ab4 = c4.nframes * c4.npix * 4 + nnz4 * 8 + (c4.npt + 1) * 4 + c4.nframes * 3 * c4.npt * 4
    ex["batch_cfg4_1024_frames"] = {"frames_per_s": c4.nframes / (ms * 1e-3), "ms_per_batch": ms,
                                    "algorithmic_bytes": ab4, "algorithmic_GBps": ab4 / (ms * 1e-3) / 1e9,
                                    "frac_of_peak": ab4 / (ms * 1e-3) / 1e9 / peak_gbs,
                                    "vs_3000_fps_detector": c4.nframes / (ms * 1e-3) / 3000.0,
                                    "kernel": "tiled_bstream_kernel (two frames per pass) + tiled_stage2_kernel",
                                    "note": "4.3 GB of frames > L2; 8 distinct frames repeated"}
    it.close()
    return ex


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of CPU work for the cpu_baseline leg")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        if args.steps > 200:
            args.steps = args.steps          # the per-step sample shrinks instead (run_reference)
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
