"""Context numbers printed beside bench.py's headline (N = 1 only); none of them feeds `value`.

Steady-state streaming and the flushed per-step protocol on cfg2, the other accumulators, configs[2] (full
preprocessing), configs[4] (4096^2: tiled vs canonical CSR vs LUT x plain / Kahan / fp64, each with its time, its
fraction of the HBM roofline on its own algorithmic bytes and its largest per-bin error against the fp64 oracle --
BASELINE.json configs[4]), the frame shape of the paper's Table 3, the batched entry point on cfg2 and cfg4
(configs[3]), and the one-time build next to the oracle's matrix build.
"""
from __future__ import annotations

import statistics
import time

import numpy as np

from paper_1412_6367_b200 import workloads as W


def _rel_err_max(got, want, count):
    ok = count > 0
    return float(np.max(np.abs(got[ok] - want[ok]) / np.abs(want[ok]))) if ok.any() else 0.0


def run(torch, B, integ, cfg, frames_dev, flush, peak_gbs, args, device):
    import bench as BM
    none5 = (None, None, None, None, None)
    ex = {}
    nnz = B.ai_get_csr(integ.ctx)[3]
    ab = BM.algorithmic_bytes(cfg, nnz)
    n = max(50, min(args.steps, 500))
    # steady state: matrix stays in L2, frames rotate
    ms = BM.back_to_back(torch, integ, frames_dev, none5, 2000, warmup=400)
    ex["warm_back_to_back"] = {"frames_per_s": 2000 / (ms * 1e-3), "algorithmic_GBps": ab * 2000 / (ms * 1e-3) / 1e9,
                               "note": "no L2 flush, 16 frames rotating, matrix L2-resident"}
    # the other protocol: L2 flushed before every step, one event pair per step (isolated launches: no overlap between
    # consecutive kernels); the cost of an event pair around a trivial kernel after the same flush is reported beside it
    tot, _, _ = BM.timed_steps(torch, B, integ, frames_dev, none5, n, 3, flush, profile=False)
    x = torch.zeros(32, device=device)
    ov = []
    for _ in range(30):
        flush()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); x.add_(1); e1.record()
        torch.cuda.synchronize()
        ov.append(e0.elapsed_time(e1))
    ex["flushed_per_step_events"] = {"frames_per_s": n / (tot * 1e-3), "ms_per_step": tot / n,
                                     "event_pair_around_trivial_kernel_ms": statistics.median(ov),
                                     "note": "single-call latency: 256 MiB written + 256 MiB read before every step, events "
                                             "around each step (stream kernel + finish kernel, nothing to overlap with)"}
    # the other accumulators on the headline workload: same train protocol, 3 contexts in rotation
    its = [B.Integrator(cfg, device=device) for _ in range(3)]
    for aname, acc in (("kahan", B.AI_ACC_F32_KAHAN), ("f64", B.AI_ACC_F64), ("plain", B.AI_ACC_F32_PLAIN)):
        for it in its:
            it.set_options(B.AI_LAYOUT_TILED, acc)
        tr = BM.Train(torch, B, its, frames_dev, none5)
        tr.warm_up(50, 100, max_trains=12)
        med, _, _ = tr.measure(100, 5)
        ex[f"train_cfg2_tiled_{aname}"] = {"ms_per_step": med / 100, "frames_per_s": 100 / (med * 1e-3),
                                           "frac_of_peak": ab / (med / 100 * 1e-3) / 1e9 / peak_gbs}
    for it in its:
        it.close()
    # configs[2] (full preprocessing, q, 3000 bins) and configs[4] (4096^2, 5000 bins): the same train protocol as the
    # headline -- 3 contexts and 4 frames in rotation (> L2), one event pair around the train, whole steps
    for name in ("cfg3", "cfg5"):
        c = W.CONFIGS[name]
        fr = W.make_frame(c)
        its = [B.Integrator(c, device=device) for _ in range(3)]
        fdev = [torch.from_numpy(fr.image).to(device) for _ in range(4)]
        corr = tuple(None if a is None else torch.from_numpy(a).to(device)
                     for a in (fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask))
        ab_c = BM.algorithmic_bytes(c, B.ai_get_csr(its[0].ctx)[3], corrections=c.corrections)
        steps = max(20, n // 2)
        tr = BM.Train(torch, B, its, fdev, corr)
        tr.warm_up(steps, 3 * steps, max_trains=12)
        med, allms, launches = tr.measure(steps, 5)
        ms = med / steps
        info = B.ai_get_layout_info(its[0].ctx)
        ex[f"train_{name}_tiled_kahan"] = {"frames_per_s": 1e3 / ms, "ms_per_step": ms, "launches_per_step": launches / steps,
                                           "algorithmic_bytes": ab_c, "algorithmic_GBps": ab_c / (ms * 1e-3) / 1e9,
                                           "frac_of_peak": ab_c / (ms * 1e-3) / 1e9 / peak_gbs,
                                           "extra_bytes_not_in_the_algorithmic_count": (
                                               {"corrected_frame_written_and_read_back": 2 * 4 * c.npix,
                                                "partial_records_written_and_read_back": 2 * 16 * info["nslot"]}
                                               if c.corrections else
                                               {"partial_records_written_and_read_back": 2 * 16 * info["nslot"]}),
                                           "layout": info}
        if name == "cfg3":
            # the same frames against HELD corrections (ai_hold_corrections): the division and the mask are folded into a
            # copy of the matrix once, the single-frame kernel loads the dark tile beside the frame tile -- no pre-pass
            for it in its:
                it.hold_corrections(*corr)
            trh = BM.Train(torch, B, its, fdev, (None,) * 5)
            trh.warm_up(steps, 3 * steps, max_trains=12)
            medh, _, launches_h = trh.measure(steps, 5)
            msh = medh / steps
            ab_h = c.npix * 4 + c.npix * 4 + B.ai_get_csr(its[0].ctx)[3] * 8 + (c.npt + 1) * 4 + 3 * c.npt * 4
            ex["train_cfg3_held_corrections"] = {
                "frames_per_s": 1e3 / msh, "ms_per_step": msh, "launches_per_step": launches_h / steps,
                "algorithmic_bytes_of_the_per_call_path": ab_c, "frac_of_peak_on_those": ab_c / (msh * 1e-3) / 1e9 / peak_gbs,
                "bytes_this_path_needs": ab_h, "frac_of_peak_on_its_own_bytes": ab_h / (msh * 1e-3) / 1e9 / peak_gbs,
                "note": "frame + held dark current (4 B per pixel each) + matrix + outputs; flat, solid angle, polarisation "
                        "and mask are not read per frame"}
            for it in its:
                it.hold_corrections()
        if name == "cfg5":
            ex["cfg5_layouts_and_accumulators"] = cfg5_table(torch, B, BM, c, fr, its[0], fdev, flush, peak_gbs)
        for it in its:
            it.close()
        del corr, fdev
    # context (SURVEY.md section 8(d) "T3"): the frame shape of the paper's Table 3 (Pilatus 1M, 981 x 1043 int32,
    # PAPER.md:257) -- geometry is a reading (centre of the image, 172 um pixels, 0.1 m, 1000 bins in 2theta)
    cp = W.CONFIGS["t3"]
    rngp = np.random.default_rng(14126367 + 9)
    fp = [torch.from_numpy(rngp.poisson(30.0, size=(cp.height, cp.width)).astype(np.int32)).to(device) for _ in range(4)]
    its = [B.Integrator(cp, device=device) for _ in range(6)]
    tr = BM.Train(torch, B, its, fp, none5)
    tr.warm_up(100, 300, max_trains=12)
    med, _, launches = tr.measure(200, 5)
    ex["pilatus1m_int32_table3_shape"] = {"frames_per_s": 200 / (med * 1e-3), "ms_per_step": med / 200,
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
    import os

    def time_batch64(it):
        for _ in range(2):
            it.integrate1d_batch(fb, out=outb)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            it.integrate1d_batch(fb, out=outb)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / 5

    ms = time_batch64(integ)                  # one full group of 64 frames: the frame-lane kernel
    fl_info = B.ai_get_batch_layout_info(integ.ctx)
    it_nofl = B.Integrator(cfg, device=device, path={"no_fl": 1})
    ms_nofl = time_batch64(it_nofl)           # the slice-per-lane batch kernel on the same call
    it_nofl.close()
    abb = nb * cfg.npix * 4 + nnz * 8 + (cfg.npt + 1) * 4 + nb * 3 * cfg.npt * 4
    info = B.ai_get_layout_info(integ.ctx)
    ex["batch_cfg2_64_frames"] = {"frames_per_s": nb / (ms * 1e-3), "ms_per_batch": ms, "us_per_frame": ms * 1e3 / nb,
                                  "mpix_per_s": nb * cfg.npix / (ms * 1e-3) / 1e6,
                                  "algorithmic_bytes": abb, "algorithmic_GBps": abb / (ms * 1e-3) / 1e9,
                                  "frac_of_peak": abb / (ms * 1e-3) / 1e9 / peak_gbs,
                                  "kernel": "fl_batch_kernel (one full group of 64 frames)" if fl_info.get("built") else
                                            "tiled_bstream_kernel",
                                  "slice_per_lane_kernel_no_fl": {
                                      "ms_per_batch": ms_nofl, "us_per_frame": ms_nofl * 1e3 / nb,
                                      "frac_of_peak": abb / (ms_nofl * 1e-3) / 1e9 / peak_gbs,
                                      "partial_records_written_and_read_back": 2 * 16 * info["nslot"] * nb,
                                      "note": "bit-identical to the single-frame kernel's results"},
                                  "note": "ai_integrate1d_batch on 64 device-resident cfg2 frames"}
    del fb, outb
    # configs[3]: 1024 int32 frames of 1024x1024 in one batched call
    c4 = W.CONFIGS["cfg4"]
    pool = torch.from_numpy(W.make_frames(c4, 8)).to(device)
    frames = pool.repeat(c4.nframes // 8, 1, 1)

    def time_cfg4(path):
        """ms per 1024-frame call (5 calls back to back after 2 warm-up calls) and the context, still open"""
        it4 = B.Integrator(c4, device=device, path=path)
        out4 = it4.outputs(c4.nframes)
        for _ in range(2):
            it4.integrate1d_batch(frames, out=out4)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 5
        e0.record()
        for _ in range(reps):
            it4.integrate1d_batch(frames, out=out4)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps, it4, out4

    ms, it, out = time_cfg4({})
    nnz4 = B.ai_get_csr(it.ctx)[3]
    ab4 = c4.nframes * c4.npix * 4 + nnz4 * 8 + (c4.npt + 1) * 4 + c4.nframes * 3 * c4.npt * 4
    fl4 = B.ai_get_batch_layout_info(it.ctx)
    res_fl = [o.clone() for o in out]
    it.close()
    # the same call through the slice-per-lane batched kernel (ai_path_options.no_fl): what the frame-lane kernel replaced here
    ms_sl, it, out = time_cfg4({"no_fl": 1})
    info4 = B.ai_get_layout_info(it.ctx)
    dmax = max(float(((a - b).abs() / b.abs().clamp_min(1e-30)).max()) for a, b in zip(res_fl[:2], out[:2]))
    it.close()
    ex["batch_cfg4_1024_frames"] = {"frames_per_s": c4.nframes / (ms * 1e-3), "ms_per_batch": ms,
                                    "kernel": "fl_batch_kernel (frame-lane: lane = two frames, DESIGN.md 5.4)" if fl4["built"]
                                              else "tiled_bstream_kernel",
                                    "algorithmic_bytes": ab4, "algorithmic_GBps": ab4 / (ms * 1e-3) / 1e9,
                                    "frac_of_peak": ab4 / (ms * 1e-3) / 1e9 / peak_gbs,
                                    "extra_bytes_not_in_the_algorithmic_count":
                                        {"partial_sums_written_and_read_back": 2 * 8 * fl4["nslot"] * c4.nframes,
                                         "matrix_blobs_read_once_per_group_of_64_frames_mostly_from_L2":
                                             fl4["blob_bytes"] * (c4.nframes // 64)} if fl4["built"] else
                                        {"partial_records_written_and_read_back": 2 * 16 * info4["nslot"] * c4.nframes},
                                    "layout": fl4,
                                    "vs_3000_fps_detector": c4.nframes / (ms * 1e-3) / 3000.0,
                                    "slice_per_lane_kernel_no_fl": {
                                        "ms_per_batch": ms_sl, "frac_of_peak": ab4 / (ms_sl * 1e-3) / 1e9 / peak_gbs,
                                        "partial_records_written_and_read_back": 2 * 16 * info4["nslot"] * c4.nframes,
                                        "max_rel_diff_of_the_two_kernels_profiles": dmax},
                                    "note": "4.3 GB of frames > L2; 8 distinct frames repeated"}
    # configs[2] as a stream: 256 frames with every correction array and the mask in ONE batched call (PAPER.md:240-254:
    # the corrections are per-detector constants, only the image changes from frame to frame)
    c3 = W.CONFIGS["cfg3"]
    fr3 = W.make_frame(c3)
    b3 = torch.from_numpy(fr3.image).to(device)
    fb3 = torch.stack([b3, b3 * 0.5]).repeat(128, 1, 1)
    cor3 = tuple(None if a is None else torch.from_numpy(a).to(device)
                 for a in (fr3.dark, fr3.flat, fr3.solidangle, fr3.polarization, fr3.mask))
    it = B.Integrator(c3, device=device)
    out3 = it.outputs(256)
    for _ in range(2):
        it.integrate1d_batch(fb3, *cor3, out=out3)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        it.integrate1d_batch(fb3, *cor3, out=out3)
    e1.record()
    torch.cuda.synchronize()
    ms3 = e0.elapsed_time(e1) / 3
    ab3 = 256 * c3.npix * 4 + 17 * c3.npix + B.ai_get_csr(it.ctx)[3] * 8 + (c3.npt + 1) * 4 + 256 * 3 * c3.npt * 4
    ex["batch_cfg3_256_frames_all_corrections"] = {
        "frames_per_s": 256 / (ms3 * 1e-3), "ms_per_batch": ms3, "us_per_frame": ms3 * 1e3 / 256,
        "launches_per_call": B.ai_last_launch_count(it.ctx), "algorithmic_bytes": ab3,
        "frac_of_peak": ab3 / (ms3 * 1e-3) / 1e9 / peak_gbs,
        "kernel": "fl_batch_kernel, corrected variant (per call: validity, scale and dark per pixel, the blobs with the "
                  "coefficients scaled, the static count; the loaders subtract the dark current as they stage a tile)",
        "note": "the same frames one by one (extras.train_cfg3_tiled_kahan) take 45 us each"}
    it.hold_corrections(*cor3)
    for _ in range(2):
        it.integrate1d_batch(fb3, out=out3)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(3):
        it.integrate1d_batch(fb3, out=out3)
    e1.record()
    torch.cuda.synchronize()
    ms3h = e0.elapsed_time(e1) / 3
    ex["batch_cfg3_256_frames_held_corrections"] = {
        "frames_per_s": 256 / (ms3h * 1e-3), "ms_per_batch": ms3h, "us_per_frame": ms3h * 1e3 / 256,
        "launches_per_call": B.ai_last_launch_count(it.ctx),
        "note": "ai_hold_corrections: the scaled blobs and the static count are kept from call to call"}
    it.close()
    del fb3, out3, cor3
    # bidimensional integration of the headline frame: 360 azimuthal x 500 radial bins
    ck = W.CONFIGS["cake2"]
    its = [B.Integrator(ck, device=device) for _ in range(3)]
    outs = [tuple(torch.empty((ck.npt_azim, ck.npt), dtype=torch.float32, device=device) for _ in range(3)) for _ in its]
    nnz2 = B.ai_get_csr(its[0].ctx)[3]

    def cake_train(k):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(k):
            its[i % 3].integrate2d(frames_dev[i % len(frames_dev)], out=outs[i % 3])
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / k

    for _ in range(6):
        cake_train(50)
    ms = statistics.median(cake_train(100) for _ in range(5))
    ab2 = ck.npix * 4 + nnz2 * 8 + (ck.npt * ck.npt_azim + 1) * 4 + 3 * ck.npt * ck.npt_azim * 4
    ex["train_cake2_360x500_bins"] = {"frames_per_s": 1e3 / ms, "ms_per_step": ms, "nnz": nnz2, "algorithmic_bytes": ab2,
                                      "frac_of_peak": ab2 / (ms * 1e-3) / 1e9 / peak_gbs,
                                      "layout": B.ai_get_layout_info(its[0].ctx)}
    # the same with the correction arrays of cfg3 (same detector size): per call, and held by the contexts
    fr3c = W.make_frame(W.CONFIGS["cfg3"])
    corc = tuple(torch.from_numpy(a).to(device) for a in (fr3c.dark, fr3c.flat, fr3c.solidangle, fr3c.polarization, fr3c.mask))

    def cake_train_corrected(k, args):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(k):
            its[i % 3].integrate2d(frames_dev[i % len(frames_dev)], *args, out=outs[i % 3])
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / k

    for _ in range(4):
        cake_train_corrected(50, corc)
    ms_pc = statistics.median(cake_train_corrected(100, corc) for _ in range(5))
    for it in its:
        it.hold_corrections(*corc)
    for _ in range(4):
        cake_train_corrected(50, (None,) * 5)
    ms_h = statistics.median(cake_train_corrected(100, (None,) * 5) for _ in range(5))
    ex["train_cake2_all_corrections"] = {"per_call_arrays_ms_per_step": ms_pc, "held_corrections_ms_per_step": ms_h,
                                         "held_launches_per_step": B.ai_last_launch_count(its[0].ctx)}
    del corc
    for it in its:
        it.close()
    ex["build_vs_oracle"] = build_times(torch, B, device)
    return ex


def cfg5_table(torch, B, BM, c, fr, integ, fdev, flush, peak_gbs):
    """BASELINE.json configs[4]: layouts x accumulators on the 4096^2 frame.  Flushed L2, library events around the
    dominant kernel of each call (isolated launches); error = largest per-bin relative error of `intensity` against the
    fp64 oracle on the same frame."""
    from oracle import oracle as O
    want = O.integrate1d(c, fr)
    nnz = B.ai_get_csr(integ.ctx)[3]
    info = B.ai_get_layout_info(integ.ctx)
    none5 = (None,) * 5
    table = {}
    lut_w = None
    for lname, layout in (("tiled", B.AI_LAYOUT_TILED), ("csr", B.AI_LAYOUT_CSR), ("lut", B.AI_LAYOUT_LUT),
                          ("scatter", B.AI_LAYOUT_SCATTER)):
        for aname, acc in (("plain", B.AI_ACC_F32_PLAIN), ("kahan", B.AI_ACC_F32_KAHAN), ("f64", B.AI_ACC_F64)):
            if lname == "scatter" and aname != "plain":
                continue                              # fp32 atomics: there is only one arithmetic
            integ.set_options(layout, acc)
            i, s, cnt = integ.integrate1d(fdev[0])
            torch.cuda.synchronize()
            err = _rel_err_max(i.cpu().numpy().astype(np.float64), want["intensity"], want["count"])
            steps = 12
            tot, kms, _ = BM.timed_steps(torch, B, integ, fdev, none5, steps, 2, flush)
            k = statistics.median(kms)
            if lname == "scatter":
                bytes_ = c.npix * 4 + c.npix * 12 + 3 * c.npt * 4       # frame + 12 B of split geometry per pixel + outputs
            elif lname == "lut":
                if lut_w is None:                       # padded row length = the longest row of the CSR
                    indptr = np.empty(c.npt + 1, dtype=np.int32)
                    B.ai_copy_csr_to_host(integ.ctx, indptr)
                    lut_w = (int(np.diff(indptr).max()) + 3) // 4 * 4
                bytes_ = c.npix * 4 + 8 * lut_w * c.npt + 3 * c.npt * 4
            else:
                bytes_ = BM.algorithmic_bytes(c, nnz)
            table[f"{lname}_{aname}"] = {"kernel_ms": k, "algorithmic_bytes": bytes_,
                                         "frac_of_peak": bytes_ / (k * 1e-3) / 1e9 / peak_gbs,
                                         "max_rel_err_vs_oracle": err}
    integ.set_options()
    table["note"] = ("isolated launches (L2 flushed, events around the dominant kernel); LUT bytes = frame + padded table "
                     f"(8 B x {lut_w} x {c.npt}) + outputs; tiled layout really moves {info['blob_bytes']} B of matrix")
    return table


def build_times(torch, B, device):
    """One-time cost: ai_setup + ai_build_csr (B1-B6 on the GPU, including the execution layouts) next to the oracle's
    bounds + CSR build on one host core."""
    from oracle import oracle as O
    out = {}
    for name in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
        c = W.CONFIGS[name]
        ts = []
        for _ in range(2):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            it = B.Integrator(c, device=device)
            torch.cuda.synchronize()
            ts.append(time.perf_counter() - t0)
            it.close()
        t0 = time.perf_counter()
        umin, umax = O.pixel_bounds(c)
        u0, u1 = O.auto_range(umin, umax)
        O.csr(umin, umax, c.npt, u0, u1)
        t_or = time.perf_counter() - t0
        out[name] = {"gpu_build_ms": min(ts) * 1e3, "oracle_bounds_plus_csr_ms_1_core": t_or * 1e3}
    return out
