"""A few calls of one named workload, for `ncu` to capture (the commands are quoted in profiles/*.md|*.txt).

    python profile_cases.py cfg2 [--calls 12]            # BASELINE.json configs[1]: one plain 2048^2 frame per call
    python profile_cases.py cfg4_batch [--calls 3]       # configs[3]: 1024 int32 frames per call
    python profile_cases.py cfg3 [--calls 12]            # configs[2]: every correction array + mask
    python profile_cases.py cfg3_held [--calls 12]       # the same against held corrections (ai_hold_corrections)
    python profile_cases.py cfg2_batch64                 # 64 frames of configs[1] per call
    python profile_cases.py cfg2_batch16                 # 16 frames per call: the slice-per-lane batched kernel
    python profile_cases.py cake2                        # 2048^2 into 360 x 500 bins
    python profile_cases.py cfg5_csr | cfg5_lut | cfg5_scatter      # configs[4] through the paper's own layouts

    --train K [--warm W]: W untimed calls (default 600: the enqueue rate of a fresh process has settled by then), then
    cudaProfilerStart, K calls back to back, a synchronise, cudaProfilerStop -- for `ncu --replay-mode app-range`,
    which measures the range as a whole with the launches overlapping as they do without the profiler (consecutive calls
    overlap through programmatic dependent launch; a per-kernel capture serialises them).  Under the profiler the host
    needs ~65 us to enqueue a call, so the GPU idles between calls; --hold-cycles N opens the range with a kernel that
    spins N cycles while the calls queue up behind it.  Two such ranges of K1 and K2 calls differ by exactly K2 - K1 calls
    running back to back: (time2 - time1) / (K2 - K1) and (bytes2 - bytes1) / (K2 - K1) are the in-situ figures per call.

Inputs are the seeded synthetic frames of workloads.py; nothing is checked or timed here (tests/ and bench.py do that).
"""
from __future__ import annotations

import argparse

import torch

from paper_1412_6367_b200 import binding as B
from paper_1412_6367_b200 import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("case", choices=["cfg2", "cfg4_batch", "cfg3", "cfg3_held", "cfg2_batch64", "cfg2_batch16", "cake2",
                                     "cfg5_csr", "cfg5_lut", "cfg5_scatter"])
    ap.add_argument("--calls", type=int, default=0)
    ap.add_argument("--train", type=int, default=0, help="profiler range around this many back-to-back calls")
    ap.add_argument("--warm", type=int, default=600, help="untimed calls before the range (with --train)")
    ap.add_argument("--hold-cycles", type=int, default=0,
                    help="with --train: a kernel that spins this many clock cycles opens the range, so that the calls are "
                         "all enqueued (slowly, under the profiler) while the GPU is held, and then run back to back")
    args = ap.parse_args()
    B.lib()
    dev = "cuda:0"
    if args.case == "cfg4_batch":
        c = W.CONFIGS["cfg4"]
        pool = torch.from_numpy(W.make_frames(c, 8)).to(dev)
        frames = pool.repeat(c.nframes // 8, 1, 1)
        it = B.Integrator(c, device=dev)
        out = it.outputs(c.nframes)
        call, default_calls = (lambda k: it.integrate1d_batch(frames, out=out)), 3
    elif args.case in ("cfg2_batch64", "cfg2_batch16"):
        n = 64 if args.case == "cfg2_batch64" else 16
        c = W.CONFIGS["cfg2"]
        base = torch.from_numpy(W.make_frame(c).image).to(dev)
        frames = torch.stack([base * (1.0 + 0.01 * k) for k in range(n)])
        it = B.Integrator(c, device=dev)
        out = it.outputs(n)
        call, default_calls = (lambda k: it.integrate1d_batch(frames, out=out)), 3
    elif args.case in ("cfg3", "cfg3_held"):
        c = W.CONFIGS["cfg3"]
        fr = W.make_frame(c)
        fdev = [torch.from_numpy(fr.image).to(dev) for _ in range(4)]
        corr = tuple(None if a is None else torch.from_numpy(a).to(dev)
                     for a in (fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask))
        its = [B.Integrator(c, device=dev) for _ in range(3)]
        outs = [it.outputs() for it in its]
        if args.case == "cfg3_held":
            for it in its:
                it.hold_corrections(*corr)
            corr = (None,) * 5
        call, default_calls = (lambda k: its[k % 3].integrate1d(fdev[k % 4], *corr, out=outs[k % 3])), 12
    elif args.case == "cfg2":
        # the rotation bench.py uses: more matrix copies and frames than the L2 holds
        c = W.CONFIGS["cfg2"]
        fdev = [torch.from_numpy(W.make_frame(c, k).image).to(dev) for k in range(8)]
        its = [B.Integrator(c, device=dev) for _ in range(6)]
        outs = [it.outputs() for it in its]
        call, default_calls = (lambda k: its[k % 6].integrate1d(fdev[k % 8], out=outs[k % 6])), 12
    elif args.case.startswith("cfg5_"):
        c = W.CONFIGS["cfg5"]
        layout = {"cfg5_csr": B.AI_LAYOUT_CSR, "cfg5_lut": B.AI_LAYOUT_LUT, "cfg5_scatter": B.AI_LAYOUT_SCATTER}[args.case]
        img = torch.from_numpy(W.make_frame(c).image).to(dev)
        it = B.Integrator(c, device=dev, layout=layout)
        out = it.outputs()
        call, default_calls = (lambda k: it.integrate1d(img, out=out)), 3
    else:
        c = W.CONFIGS["cake2"]
        imgs = [torch.from_numpy(W.make_frame(W.CONFIGS["cfg2"], k).image).to(dev) for k in range(4)]
        its = [B.Integrator(c, device=dev) for _ in range(3)]
        outs = [tuple(torch.empty((c.npt_azim, c.npt), dtype=torch.float32, device=dev) for _ in range(3)) for _ in its]
        call, default_calls = (lambda k: its[k % 3].integrate2d(imgs[k % 4], out=outs[k % 3])), 6
    if args.train > 0:
        for k in range(args.warm):
            call(k)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.cudart().cudaProfilerStart()
        e0.record()
        if args.hold_cycles > 0:
            torch.cuda._sleep(args.hold_cycles)
        for k in range(args.train):
            call(args.warm + k)
        e1.record()
        torch.cuda.synchronize()
        torch.cuda.cudart().cudaProfilerStop()
        # the same range by CUDA events (meaningful when no profiler is attached): hold kernel + K calls
        print(f'{{"case": "{args.case}", "train": {args.train}, "hold_cycles": {args.hold_cycles}, '
              f'"range_ms_by_events": {e0.elapsed_time(e1):.4f}}}')
    else:
        for k in range(args.calls or default_calls):
            call(k)
    torch.cuda.synchronize()


if __name__ == "__main__":
    main()
