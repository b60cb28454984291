"""A few calls of one named workload, for `ncu` to capture (the commands are quoted in profiles/*.md|*.txt).

    python -m paper_1412_6367_b200.profile_cases cfg4_batch [--calls 3]      # BASELINE.json configs[3]: 1024 int32 frames per call
    python -m paper_1412_6367_b200.profile_cases cfg3 [--calls 12]           # configs[2]: every correction array + mask
    python -m paper_1412_6367_b200.profile_cases cfg3_held [--calls 12]      # the same against held corrections (ai_hold_corrections)
    python -m paper_1412_6367_b200.profile_cases cfg2_batch64                # 64 frames of configs[1] per call
    python -m paper_1412_6367_b200.profile_cases cake2                       # 2048^2 into 360 x 500 bins

Inputs are the seeded synthetic frames of workloads.py; nothing is checked or timed here (tests/ and bench.py do that).
"""
from __future__ import annotations

import argparse

import torch

from . import binding as B
from . import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("case", choices=["cfg4_batch", "cfg3", "cfg3_held", "cfg2_batch64", "cake2"])
    ap.add_argument("--calls", type=int, default=0)
    args = ap.parse_args()
    B.lib()
    dev = "cuda:0"
    if args.case == "cfg4_batch":
        c = W.CONFIGS["cfg4"]
        pool = torch.from_numpy(W.make_frames(c, 8)).to(dev)
        frames = pool.repeat(c.nframes // 8, 1, 1)
        it = B.Integrator(c, device=dev)
        out = it.outputs(c.nframes)
        for _ in range(args.calls or 3):
            it.integrate1d_batch(frames, out=out)
    elif args.case == "cfg2_batch64":
        c = W.CONFIGS["cfg2"]
        base = torch.from_numpy(W.make_frame(c).image).to(dev)
        frames = torch.stack([base * (1.0 + 0.01 * k) for k in range(64)])
        it = B.Integrator(c, device=dev)
        out = it.outputs(64)
        for _ in range(args.calls or 3):
            it.integrate1d_batch(frames, out=out)
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
        for k in range(args.calls or 12):
            its[k % 3].integrate1d(fdev[k % 4], *corr, out=outs[k % 3])
    else:
        c = W.CONFIGS["cake2"]
        img = torch.from_numpy(W.make_frame(W.CONFIGS["cfg2"]).image).to(dev)
        it = B.Integrator(c, device=dev)
        out = tuple(torch.empty((c.npt_azim, c.npt), dtype=torch.float32, device=dev) for _ in range(3))
        for _ in range(args.calls or 6):
            it.integrate2d(img, out=out)
    torch.cuda.synchronize()


if __name__ == "__main__":
    main()
