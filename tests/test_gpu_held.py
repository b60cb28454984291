"""Held corrections (ai_hold_corrections, include/azint.h; hold.cu): a set of correction arrays held by the context serves
the calls that pass none.  PAPER.md:240 (dark current, flat field, solid angle, polarisation, mask are applied to every
frame) is what is computed; the oracle gets the arrays themselves.  Single 32-bit frames take the single-frame kernel with
the held copy of the matrix (2 launches), batches the frame-lane kernel without its per-call preparation, everything
else sees a (dark, denominator) pair.
"""
import numpy as np
import pytest

from parity import assert_profile

pytestmark = pytest.mark.gpu

LAYOUTS = {"tiled": 0, "csr": 1, "lut": 2, "direct": 3}
ACCUMS = {"kahan": 0, "plain": 1, "f64": 2}
SMALL = dict(center_x=100.3, center_y=90.1, npt=257, distance_m=0.02)      # blobs of 84 KB: one held stage only -> fallback
FITS = dict(center_x=100.3, center_y=90.1, npt=120, distance_m=0.03)


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(cuda_lib):
    from paper_1412_6367_b200 import binding
    binding.lib()
    return binding


def _arrays(shape, seed, edge=True):
    """dark, flat, solid angle, polarisation, mask with the degenerate pixels the method has"""
    rng = np.random.default_rng(seed)
    dark = rng.poisson(5.0, shape).astype(np.float32)
    flat = rng.uniform(0.9, 1.1, shape).astype(np.float32)
    solid = rng.uniform(0.7, 1.0, shape).astype(np.float32)
    pol = rng.uniform(0.95, 1.0, shape).astype(np.float32)
    mask = (rng.random(shape) < 0.04).astype(np.uint8)
    if edge:
        mask[80:100, 90:112] = 1                  # around the beam centre: the innermost bins lose every pixel
        flat[10, 10] = 0.0
        flat[150, 200] = np.inf
        dark[60, 70] = np.nan                     # invalid for every frame
        dark[61, 170] = np.inf
    return dark, flat, solid, pol, mask


def _got(i, s, c):
    return {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}


def _oracle(oracle, cfg, image, arrays, empty=0.0):
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    return oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, image, *arrays, empty=empty)


def _dev(torch, arrays):
    return [None if a is None else torch.from_numpy(a).cuda() for a in arrays]


@pytest.mark.parametrize("dtype", ["float32", "int32", "uint32"])
def test_held_single_frames(torch, B, oracle, workloads, dtype):
    """One 32-bit frame per call against a held set: the single-frame kernel with the dark tile beside the frame tile, two
    launches; float frames with NaN / Inf pixels (one of them under the mask) repeat the blocks that meet them."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="held1", **FITS)
    rng = np.random.default_rng(3)
    frames = rng.poisson(80.0, size=(3, cfg.height, cfg.width)).astype(dtype)
    arrays = _arrays((cfg.height, cfg.width), 11)
    if dtype == "float32":
        frames[1, 33, 44] = np.nan
        frames[0, 85, 95] = np.nan                # under the mask: must not touch anything
        frames[2, 120, 7] = np.inf
    integ = B.Integrator(cfg, empty_value=-1.0)
    integ.hold_corrections(*_dev(torch, arrays))
    for f in range(3):
        if dtype == "uint32":
            t, code = torch.from_numpy(frames[f].view(np.int32)).cuda(), B.AI_U32
        else:
            t, code = torch.from_numpy(frames[f]).cuda(), None
        i, s, c = integ.outputs()
        B.ai_integrate1d(integ.ctx, t, None, None, None, None, None, None, i, s, c, dtype=code)
        torch.cuda.synchronize()
        assert B.ai_last_launch_count(integ.ctx) == 2
        want = _oracle(oracle, cfg, frames[f], arrays, empty=-1.0)
        assert (want["count"] <= 0).sum() >= 3
        assert_profile(_got(i, s, c), want, what=f"held/{dtype}/frame {f}")
    integ.close()


@pytest.mark.parametrize("which", ["dark", "mask", "flat", "solid+pol"])
def test_held_subsets(torch, B, oracle, workloads, which):
    """Any subset of the five arrays can be held."""
    cfg = workloads.tiny_config(130, 200, unit=workloads.Q_NM, name="held_sub", center_x=60.2, center_y=70.7, npt=150,
                                distance_m=0.03)
    img = np.random.default_rng(5).poisson(200.0, size=(cfg.height, cfg.width)).astype(np.float32)
    dark, flat, solid, pol, mask = _arrays((cfg.height, cfg.width), 23, edge=False)
    arrays = {"dark": (dark, None, None, None, None), "mask": (None, None, None, None, mask),
              "flat": (None, flat, None, None, None), "solid+pol": (None, None, solid, pol, None)}[which]
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    i, s, c = integ.integrate1d(torch.from_numpy(img).cuda())
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 2
    assert_profile(_got(i, s, c), _oracle(oracle, cfg, img, arrays), what=f"held subset {which}")
    integ.close()


@pytest.mark.parametrize("layout", ["tiled", "direct", "csr", "lut"])
def test_held_dark_only_with_non_finite_pixels(torch, B, oracle, workloads, layout):
    """A held set of a dark current alone whose NaN / Inf pixels are invalid for every frame (include/azint.h): the same
    profiles on the held-aware kernel, on the kernels that see the set as a (dark, denominator) pair -- other layouts,
    fp64 accumulation, 16-bit frames -- and with the array passed per call."""
    cfg = workloads.tiny_config(130, 200, unit=workloads.Q_NM, name="held_dark", center_x=60.2, center_y=70.7, npt=150,
                                distance_m=0.03)
    rng = np.random.default_rng(31)
    img = rng.poisson(200.0, size=(cfg.height, cfg.width)).astype(np.float32)
    img16 = rng.poisson(300.0, size=(cfg.height, cfg.width)).astype(np.uint16)
    dark = rng.poisson(5.0, size=img.shape).astype(np.float32)
    dark[60, 70] = np.nan
    dark[61, 170] = np.inf
    dark[0, 0] = -np.inf
    dark[100:104, 20:90] = np.nan                 # enough weight to move several bins far beyond the tolerance
    arrays = (dark, None, None, None, None)
    want = _oracle(oracle, cfg, img, arrays)
    want16 = _oracle(oracle, cfg, img16, arrays)
    integ = B.Integrator(cfg)
    d_dark = torch.from_numpy(dark).cuda()
    t, t16 = torch.from_numpy(img).cuda(), torch.from_numpy(img16.view(np.int16)).cuda()
    assert_profile(_got(*integ.integrate1d(t, dark=d_dark)), want, what="dark per call")
    integ.hold_corrections(dark=d_dark)
    for accum in ("kahan", "f64"):
        integ.set_options(LAYOUTS[layout], ACCUMS[accum], 0.0)
        assert_profile(_got(*integ.integrate1d(t)), want, what=f"held dark only via {layout}/{accum}")
        i, s, c = integ.outputs()
        B.ai_integrate1d(integ.ctx, t16, None, None, None, None, None, None, i, s, c, dtype=B.AI_U16)
        torch.cuda.synchronize()
        assert_profile(_got(i, s, c), want16, what=f"held dark only, uint16 via {layout}/{accum}")
    integ.close()


def test_held_replaced_dropped_and_overridden(torch, B, oracle, workloads):
    """A second ai_hold_corrections replaces the set, all-NULL drops it, and a call with arrays of its own ignores it."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.R_MM, name="held2", **SMALL)
    img = np.random.default_rng(9).poisson(120.0, size=(cfg.height, cfg.width)).astype(np.int32)
    t = torch.from_numpy(img).cuda()
    set_a, set_b = _arrays((cfg.height, cfg.width), 1), _arrays((cfg.height, cfg.width), 2, edge=False)
    none = (None,) * 5
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, set_a))
    assert_profile(_got(*integ.integrate1d(t)), _oracle(oracle, cfg, img, set_a), what="set a")
    dev_b = _dev(torch, set_b)
    assert_profile(_got(*integ.integrate1d(t, *dev_b)), _oracle(oracle, cfg, img, set_b), what="own arrays over held")
    assert B.ai_last_launch_count(integ.ctx) == 3          # the per-call path: pre-pass, single-frame kernel, finish
    integ.hold_corrections(*dev_b)
    assert_profile(_got(*integ.integrate1d(t)), _oracle(oracle, cfg, img, set_b), what="set b")
    integ.hold_corrections()
    plain = integ.integrate1d(t)
    assert_profile(_got(*plain), _oracle(oracle, cfg, img, none), what="dropped")
    fresh = B.Integrator(cfg)
    ref = fresh.integrate1d(t)
    torch.cuda.synchronize()
    assert all(torch.equal(x, y) for x, y in zip(plain, ref)), "after dropping the set the plain path is the plain path"
    integ.close()
    fresh.close()


@pytest.mark.parametrize("layout,accum", [("tiled", "kahan"), ("tiled", "f64"), ("tiled", "plain"), ("direct", "kahan"), ("csr", "kahan"),
                                          ("lut", "kahan")])
def test_held_set_through_the_other_kernels(torch, B, oracle, workloads, layout, accum):
    """Layouts and accumulators without a held-aware kernel see the held set as a (dark, denominator) pair: same
    profiles; so do 16-bit frames on the default layout, and 32-bit frames where two stages of (frame tile, dark tile,
    blob) do not fit the shared memory (this geometry: blobs of up to 84 KB)."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="held3", **SMALL)
    rng = np.random.default_rng(13)
    img = rng.poisson(90.0, size=(cfg.height, cfg.width)).astype(np.float32)
    arrays = _arrays((cfg.height, cfg.width), 17)
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    integ.set_options(LAYOUTS[layout], ACCUMS[accum], 0.0)
    tol = 2e-5 if accum == "plain" else None          # plain fp32 accumulation: reported, not a parity path
    got = _got(*integ.integrate1d(torch.from_numpy(img).cuda()))
    want = _oracle(oracle, cfg, img, arrays)
    if tol is None:
        assert_profile(got, want, what=f"held via {layout}/{accum}")
    else:
        ok = want["count"] > 0
        assert np.allclose(got["intensity"][ok], want["intensity"][ok], rtol=tol)
    integ.set_options(LAYOUTS["tiled"], ACCUMS["kahan"], 0.0)
    img16 = rng.poisson(300.0, size=(cfg.height, cfg.width)).astype(np.uint16)
    i, s, c = integ.outputs()
    B.ai_integrate1d(integ.ctx, torch.from_numpy(img16.view(np.int16)).cuda(), None, None, None, None, None, None, i, s, c,
                     dtype=B.AI_U16)
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 3          # pre-pass over frame, dark and denominator
    assert_profile(_got(i, s, c), _oracle(oracle, cfg, img16, arrays), what="held/uint16")
    integ.close()


@pytest.mark.parametrize("dtype,nframes", [("float32", 100), ("int32", 66)])
def test_held_batches(torch, B, oracle, workloads, monkeypatch, dtype, nframes):
    """Batches against a held set through the frame-lane kernel: the first call makes the scaled blobs and the static
    count (2 + 2 launches), later calls are the batch kernel and its finish kernel only; small batches take the general
    kernel with the (dark, denominator) pair."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="held4", **SMALL)
    rng = np.random.default_rng(29 + nframes)
    frames = rng.poisson(80.0, size=(nframes, cfg.height, cfg.width)).astype(dtype)
    arrays = _arrays((cfg.height, cfg.width), 31)
    if dtype == "float32":
        frames[2, 33, 44] = np.nan
        frames[0, 85, 95] = np.nan
        frames[nframes - 1, 120, 7] = np.inf
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    t = torch.from_numpy(frames).cuda()
    for call, launches in ((0, 4), (1, 2)):
        i, s, c = integ.integrate1d_batch(t)
        torch.cuda.synchronize()
        assert B.ai_last_launch_count(integ.ctx) == launches
        for f in sorted({0, 2, nframes // 2, nframes - 1}):
            assert_profile(_got(i[f], s[f], c[f]), _oracle(oracle, cfg, frames[f], arrays), what=f"held batch {dtype} call {call} frame {f}")
    # a new set: the frame-lane copies are made again
    other = _arrays((cfg.height, cfg.width), 37, edge=False)
    integ.hold_corrections(*_dev(torch, other))
    i, s, c = integ.integrate1d_batch(t[:64])
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 4
    assert_profile(_got(i[63], s[63], c[63]), _oracle(oracle, cfg, frames[63], other), what="held batch, second set")
    monkeypatch.setitem(B.PATH_DEFAULTS, "no_fl", 1)
    monkeypatch.delitem(B.PATH_DEFAULTS, "force_fl")
    small = B.Integrator(cfg)
    small.hold_corrections(*_dev(torch, arrays))
    i, s, c = small.integrate1d_batch(t[:3])
    torch.cuda.synchronize()
    for f in range(3):
        assert_profile(_got(i[f], s[f], c[f]), _oracle(oracle, cfg, frames[f], arrays), what=f"held small batch frame {f}")
    integ.close()
    small.close()


def test_held_host_frames(torch, B, oracle, workloads):
    """The end-to-end entry point with a held set: only the frames cross the bus."""
    cfg = workloads.CONFIGS["cfg1b"]
    rng = np.random.default_rng(41)
    frames = rng.poisson(60.0, size=(5, cfg.height, cfg.width)).astype(np.int32)
    arrays = _arrays((cfg.height, cfg.width), 43, edge=False)
    pinned = torch.from_numpy(frames).pin_memory()
    outs = [torch.empty((5, cfg.npt), dtype=torch.float32).pin_memory() for _ in range(3)]
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    B.ai_integrate1d_host_frames(integ.ctx, pinned.numpy(), 5, cfg.npix, None, None, None, None, None,
                                 *[o.numpy() for o in outs])
    for k in range(5):
        got = {"intensity": outs[0][k].numpy(), "sum_signal": outs[1][k].numpy(), "count": outs[2][k].numpy()}
        assert_profile(got, _oracle(oracle, cfg, frames[k], arrays), what=f"held host frame {k}")
    integ.close()


def test_held_full_size_and_reproducible(torch, B, oracle, workloads):
    """BASELINE.json configs[2] (2048 x 2048, q, 3000 bins, every correction and a mask) against a held set, at full
    size against the oracle, and a chain of overlapping calls on alternating frames gives the same bits every time."""
    cfg = workloads.CONFIGS["cfg3"]
    fr = workloads.make_frame(cfg)
    arrays = (fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    a = torch.from_numpy(fr.image).cuda()
    b = a * 0.5
    first = integ.integrate1d(a)
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 2
    assert_profile(_got(*first), _oracle(oracle, cfg, fr.image, arrays), what="held cfg3")
    outs = [integ.outputs() for _ in range(12)]
    for k in range(12):
        integ.integrate1d(a if k % 2 == 0 else b, out=outs[k])
    torch.cuda.synchronize()
    for k in range(0, 12, 2):
        assert all(torch.equal(x, y) for x, y in zip(outs[k], first)), f"call {k} differs"
    for k in range(3, 12, 2):
        assert all(torch.equal(x, y) for x, y in zip(outs[k], outs[1])), f"call {k} differs"
    integ.close()


def test_held_2d(torch, B, oracle, workloads):
    """A bidimensional context with a held set: the same single-frame kernel on the held copy of the 2D matrix."""
    import math
    W = workloads
    cfg = W.scaled(W.tiny_config(80, 112, center_x=40.4, center_y=61.7, unit=W.R_MM, npt=33, name="held2d"), npt_azim=48)
    rng = np.random.default_rng(47)
    img = rng.poisson(150.0, size=(cfg.height, cfg.width)).astype(np.float32)
    dark, flat, solid, pol, mask = _arrays((cfg.height, cfg.width), 53, edge=False)
    flat[10, 10] = 0.0
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, (dark, flat, solid, pol, mask)))
    i, s, c = integ.integrate2d(torch.from_numpy(img).cuda())
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 2
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    lo, w = oracle.pixel_chi_bounds(cfg)
    want = oracle.integrate2d_bounds(umin, umax, lo, w, cfg.npt, u0, u1, cfg.npt_azim, -math.pi, math.pi, img, dark, flat,
                                     solid, pol, mask)
    got = {"intensity": i.cpu().numpy().ravel(), "sum_signal": s.cpu().numpy().ravel(), "count": c.cpu().numpy().ravel()}
    assert_profile(got, {k: np.asarray(want[k]).ravel() for k in got}, what="held 2d")
    integ.close()


def test_held_with_split_normalisation(torch, B, oracle, workloads):
    """ai_set_normalization(AI_NORM_SPLIT) against a held set: sum c (I - dark) over sum c (flat * solidangle *
    polarization), the held set seen as a (dark, denominator) pair by the two passes."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="held5", **FITS)
    rng = np.random.default_rng(61)
    img = rng.poisson(90.0, size=(cfg.height, cfg.width)).astype(np.float32)
    arrays = _arrays((cfg.height, cfg.width), 67)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    want = oracle.integrate1d_bounds_split(umin, umax, cfg.npt, u0, u1, img, *arrays)
    integ = B.Integrator(cfg)
    integ.hold_corrections(*_dev(torch, arrays))
    B.ai_set_normalization(integ.ctx, B.AI_NORM_SPLIT)
    assert_profile(_got(*integ.integrate1d(torch.from_numpy(img).cuda())), want, what="held, split normalisation")
    integ.close()
