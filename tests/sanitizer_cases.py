"""Small cases through EVERY kernel of libazint, for compute-sanitizer (memcheck / racecheck / initcheck / synccheck).

    compute-sanitizer --tool memcheck python tests/sanitizer_cases.py

Not collected by pytest (the parity tests cover correctness); this script only drives the kernels on cfg1, cfg1b and a
64 x 64 toy -- plain, corrected, 16-bit, batched, and through the test switches that force the fallback kernels -- and
checks each result loosely against the oracle so that a kernel that silently did nothing is noticed.  The paper's own
race was found through wrong results; the sanitizer logs are kept under profiles/.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from oracle import oracle as O  # noqa: E402
from paper_1412_6367_b200 import binding as B, workloads as W  # noqa: E402


def check(name, got, want):
    ok = want["count"] > 0
    err = np.abs(got[ok] - want["intensity"][ok]) / np.maximum(np.abs(want["intensity"][ok]), 1e-30)
    assert err.max() < 1e-5, (name, float(err.max()))
    print(f"  {name}: max rel err {err.max():.2e}")


def dev(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def corrected_frame(cfg, seed):
    rng = np.random.default_rng(seed)
    fr = W.make_frame(cfg)
    shape = fr.image.shape
    return W.Frame(image=fr.image, dark=rng.poisson(5.0, shape).astype(np.float32),
                   flat=rng.uniform(0.9, 1.1, shape).astype(np.float32),
                   solidangle=rng.uniform(0.8, 1.0, shape).astype(np.float32),
                   polarization=rng.uniform(0.95, 1.0, shape).astype(np.float32),
                   mask=(rng.random(shape) < 0.04).astype(np.uint8))


def run_cfg(cfg, switches):
    for k in ("AZINT_NO_TMA", "AZINT_NO_STREAM", "AZINT_NO_PREPASS"):
        os.environ.pop(k, None)
    for k in switches:
        os.environ[k] = "1"
    tag = cfg.name + ("[" + ",".join(s.replace("AZINT_", "") for s in switches) + "]" if switches else "")
    print(tag)
    fr = W.make_frame(cfg)
    frc = corrected_frame(cfg, 7)
    want, wantc = O.integrate1d(cfg, fr), O.integrate1d(cfg, frc)
    layouts = [("tiled", B.AI_LAYOUT_TILED)]
    if not switches:
        layouts += [("direct", B.AI_LAYOUT_TILED_DIRECT), ("csr", B.AI_LAYOUT_CSR), ("lut", B.AI_LAYOUT_LUT)]
    for lname, layout in layouts:
        for aname, acc in (("kahan", B.AI_ACC_F32_KAHAN), ("f64", B.AI_ACC_F64), ("plain", B.AI_ACC_F32_PLAIN)):
            integ = B.Integrator(cfg, layout=layout, accum=acc)
            img = dev(fr.image)
            # a short chain of calls: consecutive launches overlap (programmatic dependent launch)
            for _ in range(3):
                i, s, c = integ.integrate1d(img)
            torch.cuda.synchronize()
            check(f"{lname}/{aname}/plain frame", i.cpu().numpy(), want)
            args = [dev(x) for x in (frc.image, frc.dark, frc.flat, frc.solidangle, frc.polarization, frc.mask)]
            for _ in range(2):
                i, s, c = integ.integrate1d(*args)
            torch.cuda.synchronize()
            check(f"{lname}/{aname}/corrected frame", i.cpu().numpy(), wantc)
            if lname == "tiled" and aname == "kahan":
                # 16-bit and int32 frames, a batch of plain frames, a batch with a mask
                u16 = np.minimum(fr.image, 60000).astype(np.uint16)
                w16 = O.integrate1d(cfg, W.Frame(image=u16))
                i, s, c = integ.outputs()
                B.ai_integrate1d(integ.ctx, dev(u16.view(np.int16)), None, None, None, None, None, None, i, s, c,
                                 dtype=B.AI_U16)
                torch.cuda.synchronize()
                check("tiled/kahan/uint16 frame", i.cpu().numpy(), w16)
                i32 = fr.image.astype(np.int32)
                i, s, c = integ.integrate1d(dev(i32))
                torch.cuda.synchronize()
                check("tiled/kahan/int32 frame", i.cpu().numpy(), O.integrate1d(cfg, W.Frame(image=i32)))
                frames = np.stack([fr.image, fr.image * 2, fr.image + 1, fr.image * 0.5, fr.image + 3]).astype(np.float32)
                i, s, c = integ.integrate1d_batch(dev(frames))
                torch.cuda.synchronize()
                check("tiled/kahan/batch of 5, frame 3", i[3].cpu().numpy(), O.integrate1d(cfg, W.Frame(image=frames[3])))
                i, s, c = integ.integrate1d_batch(dev(frames), mask=dev(frc.mask))
                torch.cuda.synchronize()
                check("tiled/kahan/masked batch, frame 4", i[4].cpu().numpy(),
                      O.integrate1d(cfg, W.Frame(image=frames[4], mask=frc.mask)))
                # the corrected frame again, against the same arrays held by the context (hold.cu): a chain of calls
                integ.hold_corrections(*args[1:])
                for _ in range(3):
                    i, s, c = integ.integrate1d(args[0])
                torch.cuda.synchronize()
                check("tiled/kahan/held corrections", i.cpu().numpy(), wantc)
                i, s, c = integ.integrate1d_batch(dev(np.stack([frc.image] * 4)))
                torch.cuda.synchronize()
                check("tiled/kahan/held corrections, batch of 4, frame 2", i[2].cpu().numpy(), wantc)
                integ.hold_corrections()
            integ.close()


def main():
    assert torch.cuda.is_available()
    toy = W.tiny_config(64, 64, center_x=20.5, center_y=-3.0, unit=W.Q_NM, npt=90, name="toy64")
    odd = W.tiny_config(70, 1028, center_x=500.0, center_y=30.0, unit=W.TTH_DEG, npt=333, name="odd70x1028")
    # 160 tiles: the single-frame kernel fills the GPU and streams ahead of the grid dependency (the launch chain)
    mid = W.tiny_config(640, 1024, center_x=300.0, center_y=700.0, unit=W.R_MM, npt=700, name="mid640x1024")
    for cfg in (W.CONFIGS["cfg1"], W.CONFIGS["cfg1b"], toy, odd, mid):
        for switches in ((), ("AZINT_NO_STREAM",), ("AZINT_NO_PREPASS",), ("AZINT_NO_TMA",)):
            if cfg is mid and switches not in ((), ("AZINT_NO_STREAM",)):
                continue
            run_cfg(cfg, switches)
    print("sanitizer cases done")


if __name__ == "__main__":
    main()
