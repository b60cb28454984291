"""Parity of the frame-lane batched kernel (integrate_fl.cu: lane = two frames) against the CPU
oracle through the C ABI.  Large batches on matrices with more than ~2.2 entries per pixel take it by themselves
(BASELINE.json configs[3]: test_gpu_parity.py::test_batch_full_size_sampled); ai_path_options.force_fl sends every batch of plain
32-bit frames through it, ai_path_options.fl_chunk / fl_stages cuts the chunks short / caps the stages so that small cases cover
several work items per block and ring wrap-arounds.
"""
import numpy as np
import pytest

from parity import assert_profile

pytestmark = pytest.mark.gpu


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


_bounds = {}


def _want(oracle, cfg, image, empty=0.0):
    if cfg not in _bounds:
        umin, umax = oracle.pixel_bounds(cfg)
        _bounds.clear()
        _bounds[cfg] = (umin, umax) + tuple(oracle.auto_range(umin, umax))
    umin, umax, u0, u1 = _bounds[cfg]
    return oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, image, None, None, None, None, None, empty=empty)


def _batch(torch, B, integ, frames, stride=None):
    n = frames.shape[0]
    if frames.dtype == np.uint32:
        t, code = torch.from_numpy(frames.view(np.int32)).cuda(), B.AI_U32
    else:
        t, code = torch.from_numpy(frames).cuda(), None
    i, s, c = integ.outputs(n)
    B.ai_integrate1d_batch(integ.ctx, t, n, stride or frames[0].size, None, None, None, None, None, i, s, c, dtype=code)
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 2
    return i, s, c


def _row(i, s, c, f):
    return {"intensity": i[f].cpu().numpy(), "sum_signal": s[f].cpu().numpy(), "count": c[f].cpu().numpy()}


SMALL = dict(center_x=100.3, center_y=90.1, npt=257, distance_m=0.02)


@pytest.mark.parametrize("tune", [None, {"fl_chunk": 2}, {"fl_chunk": 1, "fl_stages": 2}, {"fl_owner": 1}])
@pytest.mark.parametrize("dtype,nframes", [("int32", 7), ("int32", 64), ("uint32", 65), ("float32", 130)])
def test_fl_batches_match_the_oracle(torch, B, oracle, workloads, monkeypatch, tune, dtype, nframes):
    """Every frame of a forced frame-lane batch against the oracle: one frame short of / one beyond a group of 64, a
    ragged image (264 = 8 tiles of 32 + 8 columns, 200 = 25 tiles of 8 rows), float frames with NaN and +-Inf."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    if tune:
        for k, v in tune.items():
            monkeypatch.setitem(B.PATH_DEFAULTS, k, v)
    cfg = workloads.tiny_config(200, 264, unit=workloads.Q_NM, name="fl_small", **SMALL)
    rng = np.random.default_rng(nframes)
    frames = rng.poisson(100.0, size=(nframes, cfg.height, cfg.width)).astype(dtype)
    if dtype == "float32":
        frames[1, 17, 33] = np.nan
        frames[nframes - 1, 100, 200] = np.inf
        frames[64, 199, 263] = -np.inf
        frames[3, 0, 0] = np.nan
        frames[70, 40:60, :] = np.nan            # whole bins of one frame without a valid pixel
    integ = B.Integrator(cfg)
    i, s, c = _batch(torch, B, integ, frames)
    step = 1 if nframes <= 16 else 9
    for f in sorted(set(range(0, nframes, step)) | {1, 3, 64, 70, nframes - 1} & set(range(nframes))):
        assert_profile(_row(i, s, c, f), _want(oracle, cfg, frames[f]), what=f"fl/{dtype}/{tune}/frame {f} of {nframes}")
    integ.close()


def test_fl_bins_without_a_valid_pixel_are_empty(torch, B, oracle, workloads, monkeypatch):
    """A float frame whose centre region is NaN: the bins that only see that region have count exactly 0 and
    intensity = empty_value (the invalid weight is subtracted from the row's coefficient sum in fixed point)."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    cfg = workloads.tiny_config(128, 128, center_x=64.0, center_y=64.0, unit=workloads.R_MM, npt=90, name="fl_hole")
    rng = np.random.default_rng(5)
    frames = rng.poisson(30.0, size=(66, cfg.height, cfg.width)).astype(np.float32)
    yy, xx = np.mgrid[0:128, 0:128]
    hole = (yy - 63.5) ** 2 + (xx - 63.5) ** 2 < 30.0 ** 2
    frames[5][hole] = np.nan
    frames[65][:] = np.nan
    integ = B.Integrator(cfg, empty_value=-7.0)
    i, s, c = _batch(torch, B, integ, frames)
    for f in (0, 5, 65):
        want = _want(oracle, cfg, frames[f], empty=-7.0)
        got = _row(i, s, c, f)
        assert (want["count"] <= 0).sum() > (10 if f == 5 else (89 if f == 65 else -1))
        assert_profile(got, want, what=f"hole frame {f}")
        assert np.array_equal(got["intensity"][want["count"] <= 0], np.full((want["count"] <= 0).sum(), -7.0, np.float32))
    integ.close()


def test_fl_rows_do_not_depend_on_the_batch(torch, B, workloads, monkeypatch):
    """A frame's profiles are the same bits wherever it sits in a batch (which lane, which half of the lane, which
    group), whatever the other frames are, and from run to run: every sum has a fixed order."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    monkeypatch.setitem(B.PATH_DEFAULTS, "fl_chunk", 3)
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="fl_repro", **SMALL)
    rng = np.random.default_rng(11)
    pool = rng.poisson(200.0, size=(5, cfg.height, cfg.width)).astype(np.int32)
    order = rng.integers(0, 5, size=150)
    frames = pool[order]
    integ = B.Integrator(cfg)
    i, s, c = _batch(torch, B, integ, frames)
    i2, s2, c2 = _batch(torch, B, integ, np.ascontiguousarray(frames[::-1]))
    for k in range(5):
        rows = np.nonzero(order == k)[0]
        for r in rows[1:]:
            assert torch.equal(i[r], i[rows[0]]) and torch.equal(s[r], s[rows[0]]) and torch.equal(c[r], c[rows[0]])
        assert torch.equal(i2[149 - rows[0]], i[rows[0]]) and torch.equal(s2[149 - rows[0]], s[rows[0]])
    integ.close()


def test_fl_compensation_keeps_small_terms(torch, B, workloads, monkeypatch):
    """PAPER.md:186-188 in the batched kernel: one pixel of 2^24 and 65535 pixels of 1 in one bin -- the per-product
    Kahan recurrence keeps every 1 (plain fp32 accumulation would lose those added after the big value)."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    cfg = workloads.scaled(workloads.CONFIGS["cfg1"], npt=1)
    img = np.ones((cfg.height, cfg.width), dtype=np.float32)
    img[0, 0] = 2.0 ** 24
    exact = 2.0 ** 24 + cfg.npix - 1
    frames = np.stack([img, img[::-1].copy(), img * np.float32(0.5)] * 22)
    integ = B.Integrator(cfg)
    i, s, c = _batch(torch, B, integ, frames)
    got = s.cpu().numpy()[:, 0]
    assert np.all(np.abs(got[0::3] - exact) <= 1.0) and np.all(np.abs(got[1::3] - exact) <= 1.0)      # fp32 output spacing is 2
    assert np.all(np.abs(got[2::3] - exact / 2) <= 0.5)
    integ.close()


def test_fl_frame_stride_and_the_other_kernels_agree(torch, B, oracle, workloads, monkeypatch):
    """Frames 12 elements apart more than a frame; the slice-per-lane batched kernel (ai_path_options.no_fl) gives the same
    profiles within the tolerance (different, equally fixed, summation orders)."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.R_MM, name="fl_stride", **SMALL)
    rng = np.random.default_rng(3)
    n, stride = 67, cfg.npix + 12
    buf = rng.poisson(50.0, size=(n, stride)).astype(np.int32)
    t = torch.from_numpy(buf).cuda()
    out = {}
    for name, switch in (("fl", "force_fl"), ("slices", "no_fl")):
        integ = B.Integrator(cfg, path={switch: 1})
        i, s, c = integ.outputs(n)
        B.ai_integrate1d_batch(integ.ctx, t, n, stride, None, None, None, None, None, i, s, c)
        torch.cuda.synchronize()
        out[name] = (i.cpu().numpy(), s.cpu().numpy(), c.cpu().numpy())
        integ.close()
    for f in (0, 33, 66):
        img = buf[f, :cfg.npix].reshape(cfg.height, cfg.width)
        want = _want(oracle, cfg, img)
        for name in out:
            got = {"intensity": out[name][0][f], "sum_signal": out[name][1][f], "count": out[name][2][f]}
            assert_profile(got, want, what=f"{name} frame {f}")
    assert np.allclose(out["fl"][1], out["slices"][1], rtol=1e-6, atol=0)


@pytest.mark.parametrize("name", ["cfg3", "cfg5"])
def test_fl_full_size_geometries_sampled(torch, B, oracle, workloads, name):
    """The frame-lane kernel on the two large q-unit matrices at full size (BASELINE.json configs[2] and configs[4]
    geometries: 3000 / 5000 bins, 3.5 / 2.3 entries per pixel, the latter with the beam centre off the image), taken by
    itself (no environment switch) on plain float frames from a pool of two; sampled frames against the oracle.
    112 frames = a full group of 64 and a tail of 48, enough for the kernel to take the tail as well; with 96 frames the
    tail of 32 goes to the slice-per-lane batch kernel (two more launches) -- same profiles, other summation order."""
    cfg = workloads.CONFIGS[name]
    base = workloads.make_frame(cfg).image
    pool = np.stack([base, base[::-1].copy() * np.float32(0.5)])
    dev = torch.from_numpy(pool).cuda()
    frames = dev.repeat(56, 1, 1)
    integ = B.Integrator(cfg)
    i, s, c = integ.integrate1d_batch(frames)
    torch.cuda.synchronize()
    assert B.ai_get_batch_layout_info(integ.ctx)["built"] == 1, "the frame-lane kernel did not take the batch"
    assert B.ai_last_launch_count(integ.ctx) == 2
    for f in (0, 111):
        want = _want(oracle, cfg, pool[f % 2])
        assert_profile(_row(i, s, c, f), want, what=f"{name} frame {f}")
    assert torch.equal(i[0], i[110]) and torch.equal(s[1], s[111]) and torch.equal(c[0], c[64])
    i, s, c = integ.integrate1d_batch(frames[:96])
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 4           # frame-lane kernel + finish, slice-per-lane kernel + stage 2
    for f in (63, 64, 95):
        assert_profile(_row(i, s, c, f), _want(oracle, cfg, pool[f % 2]), what=f"{name} frame {f} of 96")
    assert torch.equal(i[0], i[62]) and torch.equal(i[64], i[94]) and torch.equal(s[65], s[95])
    integ.close()


@pytest.mark.parametrize("dtype,nframes,tune", [("int32", 7, None), ("float32", 100, {"fl_chunk": 2}), ("uint32", 66, None)])
def test_fl_corrected_batches(torch, B, oracle, workloads, monkeypatch, dtype, nframes, tune):
    """Batches with every correction array and a mask (one set for all frames) through the frame-lane
    kernel: the division is folded into a per-call copy of the coefficients, the loaders subtract the dark current as
    they stage the tiles.  Pixels invalid for every frame (masked, flat = 0 or not finite, a dark current that is not
    finite, a whole masked band that empties bins) leave the counts once per call; non-finite raw pixels per frame."""
    monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    if tune:
        for k, v in tune.items():
            monkeypatch.setitem(B.PATH_DEFAULTS, k, v)
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="fl_corr", **SMALL)
    rng = np.random.default_rng(17 + nframes)
    shape = (cfg.height, cfg.width)
    frames = rng.poisson(80.0, size=(nframes,) + shape).astype(dtype)
    dark = rng.poisson(5.0, shape).astype(np.float32)
    flat = rng.uniform(0.9, 1.1, shape).astype(np.float32)
    solid = rng.uniform(0.7, 1.0, shape).astype(np.float32)
    pol = rng.uniform(0.95, 1.0, shape).astype(np.float32)
    mask = (rng.random(shape) < 0.04).astype(np.uint8)
    mask[80:100, 90:112] = 1                      # around the beam centre: the innermost bins lose every pixel
    flat[10, 10] = 0.0
    flat[150, 200] = np.inf
    dark[60, 70] = np.nan                         # a dark current that is not finite: invalid for every frame, any dtype
    dark[61, 170] = np.inf
    if dtype == "float32":
        frames[2, 33, 44] = np.nan
        frames[0, 85, 95] = np.nan                # under the mask: must not touch anything
        frames[nframes - 1, 120, 7] = np.inf
    integ = B.Integrator(cfg)
    n = frames.shape[0]
    if dtype == "uint32":
        t, code = torch.from_numpy(frames.view(np.int32)).cuda(), B.AI_U32
    else:
        t, code = torch.from_numpy(frames).cuda(), None
    cor = [torch.from_numpy(x).cuda() for x in (dark, flat, solid, pol, mask)]
    i, s, c = integ.outputs(n)
    B.ai_integrate1d_batch(integ.ctx, t, n, cfg.npix, *cor, i, s, c, dtype=code)
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 5 and B.ai_get_batch_layout_info(integ.ctx)["built"] == 1
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    for f in sorted({0, 2, n // 2, n - 1}):
        want = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, frames[f], dark, flat, solid, pol, mask)
        assert (want["count"] <= 0).sum() >= 3
        assert_profile(_row(i, s, c, f), want, what=f"corrected fl/{dtype}/frame {f} of {n}")
    integ.close()


@pytest.mark.parametrize("mode", ["plain", "percall", "held"])
def test_batch_sizes_around_the_kernel_thresholds(torch, B, oracle, workloads, mode):
    """ai_integrate1d_batch splits a batch by measured cost: the frame-lane kernel takes the leading groups
    of 64 frames and a tail that is long enough (plain 60 on this light matrix, per-call corrections 14, held 24), the rest
    goes to the slice-per-lane kernel (plain) or frame by frame through the single-frame kernels (corrected).  Sizes on
    both sides of every threshold, float frames with NaN / Inf pixels, sampled frames against the oracle, launch counts."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="thresholds", center_x=100.3, center_y=90.1,
                                npt=120, distance_m=0.03)
    rng = np.random.default_rng(5)
    shape = (cfg.height, cfg.width)
    dark = rng.poisson(5.0, shape).astype(np.float32)
    flat = rng.uniform(0.9, 1.1, shape).astype(np.float32)
    solid = rng.uniform(0.7, 1.0, shape).astype(np.float32)
    pol = rng.uniform(0.95, 1.0, shape).astype(np.float32)
    mask = (rng.random(shape) < 0.04).astype(np.uint8)
    flat[10, 10] = 0.0
    dark[60, 70] = np.nan
    arrays = (dark, flat, solid, pol, mask) if mode != "plain" else (None,) * 5
    dev = [None if a is None else torch.from_numpy(a).cuda() for a in arrays]
    pool = rng.poisson(80.0, size=(5,) + shape).astype(np.float32)
    pool[1, 33, 44] = np.nan
    pool[3, 120, 7] = np.inf
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    want = [oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, pool[k], *arrays) for k in range(5)]
    integ = B.Integrator(cfg)
    if mode == "held":
        integ.hold_corrections(*dev)
    per_frame = {"percall": 3, "held": 2}          # launches of a frame that goes through the single-frame kernels
    tail_min = {"plain": 60, "percall": 14, "held": 24}[mode]
    first = True
    for n in (32, 13, 14, 23, 24, 59, 60, 65, 77, 129):
        frames = torch.from_numpy(pool[[k % 5 for k in range(n)]]).cuda()
        i, s, c = integ.integrate1d_batch(frames, *(dev if mode == "percall" else [None] * 5))
        torch.cuda.synchronize()
        full, tail = n // 64 * 64, n % 64
        taken = full + (tail if tail >= tail_min else 0)
        expect = 0
        if taken:
            expect += 2 + (3 if mode == "percall" else 0) + (2 if mode == "held" and first else 0)
            first = False
        if n - taken:
            expect += 2 if mode == "plain" and n - taken > 1 else (n - taken) * per_frame.get(mode, 2)
        assert B.ai_last_launch_count(integ.ctx) == expect, (mode, n, taken)
        for f in sorted({0, 1, n // 2, n - 2, n - 1}):
            assert_profile(_row(i, s, c, f), want[f % 5], what=f"{mode} batch of {n}, frame {f}")
    integ.close()


@pytest.mark.parametrize("mode", ["percall", "held"])
def test_corrected_batches_at_full_size(torch, B, oracle, workloads, mode):
    """The configuration bench_extras times as batch_cfg3_*_frames_all_corrections: BASELINE.json configs[2] (2048 x 2048,
    3000 bins in q, dark / flat / solid angle / polarisation / mask) in one ai_integrate1d_batch call of 128 frames, with
    the arrays passed per call and held by the context.  14.6 M entries: the scaled copy of the frame-lane blobs, the
    static count of the pixels that are invalid for every frame and the finish kernel at full size; sampled frames
    against the oracle (PAPER.md:240 corrections, :122 sums)."""
    W = workloads
    cfg = W.CONFIGS["cfg3"]
    pool = [W.make_frame(cfg, k) for k in range(3)]
    arrays = (pool[0].dark, pool[0].flat, pool[0].solidangle, pool[0].polarization, pool[0].mask)
    n = 128
    frames = torch.empty((n, cfg.height, cfg.width), dtype=torch.float32, device="cuda")
    dev_pool = [torch.from_numpy(p.image).cuda() for p in pool]
    for f in range(n):
        frames[f].copy_(dev_pool[f % 3])
    frames[5, 700, 900] = float("nan")             # a frame's own invalid pixels on top of the static ones
    frames[127, 12, 2040] = float("inf")
    cor = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]
    integ = B.Integrator(cfg)
    if mode == "held":
        integ.hold_corrections(*cor)
        i, s, c = integ.integrate1d_batch(frames)
    else:
        i, s, c = integ.integrate1d_batch(frames, *cor)
    torch.cuda.synchronize()
    assert B.ai_get_batch_layout_info(integ.ctx)["built"] == 1          # the frame-lane kernel took the batch
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    for f in (0, 5, 64, 127):
        img = frames[f].cpu().numpy()
        want = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, *arrays, nthreads=8)
        assert_profile(_row(i, s, c, f), want, what=f"cfg3 x {n} {mode}, frame {f}")
    # frames with the same content give the same bits wherever they sit in the batch
    assert torch.equal(i[0], i[63]) and torch.equal(s[1], s[124]) and torch.equal(c[2], c[125])
    integ.close()


@pytest.mark.parametrize("mode", ["plain", "percall", "held"])
def test_prepared_batches_allocate_nothing(torch, B, oracle, workloads, mode):
    """ai_prepare_batch (include/azint.h) moves the one-time work of the batched path to start-up: the frame-lane layout and
    every scratch buffer a batch of up to max_frames frames can need.  After it the device's free memory does not move
    across batches of any size up to that -- through the frame-lane kernel, the slice-per-lane kernel and the frame-by-frame
    paths -- and the results are the oracle's."""
    cfg = workloads.tiny_config(200, 264, unit=workloads.TTH_DEG, name="prepared", center_x=100.3, center_y=90.1,
                                npt=120, distance_m=0.03)
    rng = np.random.default_rng(11)
    shape = (cfg.height, cfg.width)
    arrays = (rng.poisson(5.0, shape).astype(np.float32), rng.uniform(0.9, 1.1, shape).astype(np.float32),
              rng.uniform(0.7, 1.0, shape).astype(np.float32), rng.uniform(0.95, 1.0, shape).astype(np.float32),
              (rng.random(shape) < 0.04).astype(np.uint8)) if mode != "plain" else (None,) * 5
    dev = [None if a is None else torch.from_numpy(a).cuda() for a in arrays]
    pool = rng.poisson(80.0, size=(4,) + shape).astype(np.float32)
    pool[1, 33, 44] = np.nan
    nmax = 130
    frames = torch.from_numpy(pool[[k % 4 for k in range(nmax)]]).cuda()
    integ = B.Integrator(cfg)
    if mode == "held":
        integ.hold_corrections(*dev)
    call_arrays = dev if mode == "percall" else [None] * 5
    outs = {n: integ.outputs(n) for n in (130, 64, 40, 5, 2)}
    assert B.ai_get_batch_layout_info(integ.ctx)["built"] == 0
    B.ai_prepare_batch(integ.ctx, nmax)
    assert B.ai_get_batch_layout_info(integ.ctx)["built"] == 1
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for n in (130, 64, 40, 5, 2, 130):
        integ.integrate1d_batch(frames[:n], *call_arrays, out=outs[n])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, f"{mode}: {free0 - free1} bytes of device memory were allocated after ai_prepare_batch"
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    want = [oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, pool[k], *arrays) for k in range(4)]
    for n in (130, 40, 5):
        i, s, c = outs[n]
        for f in sorted({0, 1, n // 2, n - 1}):
            assert_profile(_row(i, s, c, f), want[f % 4], what=f"prepared {mode} batch of {n}, frame {f}")
    integ.close()
