"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same seeded inputs.
Bars (BASELINE.json north_star): per-bin relative error <= 1e-6 on intensity with compensated accumulation; CSR row
pointers and column sets identical except <= 1 ulp bin-edge ties (counted); coefficients within 1e-6 relative
(+1e-7 absolute for cancellation-limited tiny coefficients).  Run with `-m gpu` on the B200 box.
"""
import numpy as np
import pytest

from parity import assert_profile, compare_csr, rel_err

pytestmark = pytest.mark.gpu

LAYOUTS = {"tiled": 0, "csr": 1, "lut": 2, "direct": 3}
ACCUMS = {"kahan": 0, "plain": 1, "f64": 2}


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


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run(torch, integ, fr, radial=False):
    args = [_dev(torch, x) for x in (fr.image, fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)]
    rad = torch.empty(integ.npt, dtype=torch.float32, device="cuda") if radial else None
    i, s, c = integ.integrate1d(*args, radial=rad)
    torch.cuda.synchronize()
    out = {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}
    if radial:
        out["radial"] = rad.cpu().numpy()
    return out


_oracle_cache = {}


def _oracle_bounds(oracle, cfg, rng=None):
    key = (cfg, rng)
    if key not in _oracle_cache:
        umin, umax = oracle.pixel_bounds(cfg)
        u0, u1 = oracle.auto_range(umin, umax) if rng is None else rng
        if len(_oracle_cache) > 3:
            _oracle_cache.clear()
        _oracle_cache[key] = (umin, umax, u0, u1)
    return _oracle_cache[key]


def _oracle_profile(oracle, cfg, fr, rng=None, empty=0.0):
    umin, umax, u0, u1 = _oracle_bounds(oracle, cfg, rng)
    return oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, fr.image, fr.dark, fr.flat, fr.solidangle,
                                     fr.polarization, fr.mask, empty=empty)


# ----------------------------------------------------------------------------------------------------------------------
# B1-B5: the matrix
# ----------------------------------------------------------------------------------------------------------------------
def _ragged_cases(W):
    return [
        W.tiny_config(100, 130, center_x=61.3, center_y=40.7, unit=W.TTH_DEG, npt=57, name="ragged_tth"),
        W.tiny_config(67, 259, center_x=-12.5, center_y=300.0, unit=W.Q_NM, npt=301, name="ragged_q_offimage"),
        W.tiny_config(129, 65, center_x=32.0, center_y=64.0, unit=W.R_MM, npt=200, name="ragged_r_narrow_bins"),
        W.tiny_config(33, 31, center_x=15.5, center_y=16.5, unit=W.Q_A, npt=1, name="single_bin"),
        W.tiny_config(1, 1, center_x=0.5, center_y=0.5, unit=W.TTH_RAD, npt=3, name="one_pixel"),
        W.tiny_config(70, 70, center_x=35.0, center_y=35.0, unit=W.TTH_RAD, npt=4000, name="more_bins_than_pixels"),
    ]


@pytest.mark.parametrize("name", ["cfg1", "cfg1b", "cfg2", "cfg3", "cfg4", "cfg5", "ragged0", "ragged1", "ragged2",
                                  "ragged3", "ragged4", "ragged5"])
def test_csr_matches_oracle(torch, B, oracle, workloads, parity_report, name):
    cfg = _ragged_cases(workloads)[int(name[-1])] if name.startswith("ragged") else workloads.CONFIGS[name]
    integ = B.Integrator(cfg)
    gi, gx, gd, (u0, u1) = integ.csr()
    umin, umax, o0, o1 = _oracle_bounds(oracle, cfg)
    assert u0 == pytest.approx(o0, rel=1e-15, abs=1e-300) and u1 == pytest.approx(o1, rel=4e-16)
    ora = oracle.csr(umin, umax, cfg.npt, o0, o1)
    rep = compare_csr((gi, gx, gd), ora, cfg.npix)
    print(name, rep)
    parity_report.setdefault("csr_vs_oracle", {})[cfg.name] = dict(rep, unit=workloads.UNIT_NAMES[cfg.unit], npt=cfg.npt,
                                                                   shape=[cfg.height, cfg.width])
    if cfg.unit == workloads.R_MM:
        # sqrt, multiply and divide are correctly rounded on both sides: the r-unit matrix must match structurally
        assert rep["ties"] == 0
    integ.close()


def test_csr_with_explicit_range(torch, B, oracle, workloads):
    cfg = workloads.CONFIGS["cfg1b"]
    rng = (3.0, 41.5)
    integ = B.Integrator(cfg, radial_range=rng)
    gi, gx, gd, got_rng = integ.csr()
    assert got_rng == rng
    umin, umax, _, _ = _oracle_bounds(oracle, cfg, rng)
    rep = compare_csr((gi, gx, gd), oracle.csr(umin, umax, cfg.npt, *rng), cfg.npix)
    assert rep["nnz_gpu"] > 0
    fr = workloads.make_frame(cfg)
    got = _run(torch, integ, fr, radial=True)
    want = _oracle_profile(oracle, cfg, fr, rng)
    assert_profile(got, want, what="explicit range")
    assert np.allclose(got["radial"], want["radial"], rtol=2e-7)
    integ.close()


# ----------------------------------------------------------------------------------------------------------------------
# H1-H5: one frame, every layout and accumulator
# ----------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", ["tiled", "direct", "csr", "lut"])
@pytest.mark.parametrize("accum", ["kahan", "f64", "plain"])
@pytest.mark.parametrize("name", ["cfg1", "cfg1b", "cfg2"])
def test_profile_parity(torch, B, oracle, workloads, parity_report, name, layout, accum):
    cfg = workloads.CONFIGS[name]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg, layout=LAYOUTS[layout], accum=ACCUMS[accum])
    got = _run(torch, integ, fr, radial=True)
    want = _oracle_profile(oracle, cfg, fr)
    # uncompensated fp32 is reported, not held to 1e-6 (north_star: "and reported without it")
    worst = assert_profile(got, want, tol=1e-3 if accum == "plain" else 1e-6, what=f"{name}/{layout}/{accum}")
    assert np.allclose(got["radial"], want["radial"], rtol=2e-7)
    print(name, layout, accum, worst)
    parity_report.setdefault("max_per_bin_relative_error", {})[f"{name}/{layout}/{accum}"] = worst
    integ.close()


@pytest.mark.parametrize("layout", ["tiled", "direct", "csr"])
@pytest.mark.parametrize("accum", ["kahan", "plain"])
def test_profile_parity_full_corrections_cfg3(torch, B, oracle, workloads, parity_report, layout, accum):
    cfg = workloads.CONFIGS["cfg3"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg, layout=LAYOUTS[layout], accum=ACCUMS[accum])
    got = _run(torch, integ, fr)
    want = _oracle_profile(oracle, cfg, fr)
    worst = assert_profile(got, want, tol=1e-3 if accum == "plain" else 1e-6, what=f"cfg3/{layout}/{accum}")
    print("cfg3", layout, accum, worst)
    parity_report.setdefault("max_per_bin_relative_error", {})[f"cfg3/{layout}/{accum}"] = worst
    integ.close()


def test_profile_parity_cfg5_layouts_and_accumulators(torch, B, oracle, workloads, parity_report):
    """BASELINE.json configs[4]: compensated vs uncompensated fp32 and LUT vs CSR against the fp64 oracle."""
    cfg = workloads.CONFIGS["cfg5"]
    fr = workloads.make_frame(cfg)
    want = _oracle_profile(oracle, cfg, fr)
    integ = B.Integrator(cfg)
    report = {}
    for layout in ("tiled", "direct", "csr", "lut"):
        for accum in ("kahan", "f64", "plain"):
            integ.set_options(LAYOUTS[layout], ACCUMS[accum])
            got = _run(torch, integ, fr)
            # uncompensated fp32 is reported, not held to 1e-6 (north_star: "and reported without it")
            worst = assert_profile(got, want, tol=1e-3 if accum == "plain" else 1e-6, what=f"cfg5/{layout}/{accum}")
            report[(layout, accum)] = worst["intensity"]
            parity_report.setdefault("max_per_bin_relative_error", {})[f"cfg5/{layout}/{accum}"] = worst
    print("cfg5 max per-bin relative error on intensity:", report)
    # the thread-per-bin LUT sums sequentially: without compensation it is the worst of the lot
    assert report[("lut", "plain")] >= report[("lut", "kahan")]
    integ.close()


@pytest.mark.parametrize("dtype", ["int32", "uint16", "int16", "uint32", "float32"])
@pytest.mark.parametrize("layout", ["tiled", "csr"])
def test_raw_dtypes(torch, B, oracle, workloads, dtype, layout):
    cfg = workloads.scaled(workloads.CONFIGS["cfg1b"], dtype=dtype)
    fr = workloads.make_frame(cfg)
    assert fr.image.dtype == np.dtype(dtype)
    integ = B.Integrator(cfg, layout=LAYOUTS[layout])
    img = fr.image
    if dtype in ("uint16", "uint32"):        # torch has limited unsigned support: ship the bits, pass the dtype code
        t = torch.from_numpy(img.view(np.int16 if dtype == "uint16" else np.int32)).cuda()
        code = B.AI_U16 if dtype == "uint16" else B.AI_U32
    else:
        t = torch.from_numpy(img).cuda()
        code = None
    i, s, c = integ.outputs()
    B.ai_integrate1d(integ.ctx, t, None, None, None, None, None, None, i, s, c, dtype=code)
    torch.cuda.synchronize()
    got = {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}
    assert_profile(got, _oracle_profile(oracle, cfg, fr), what=f"{dtype}/{layout}")
    integ.close()


# ----------------------------------------------------------------------------------------------------------------------
# ragged shapes, unaligned buffers, masks, empty bins, non-finite data
# ----------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx", range(6))
@pytest.mark.parametrize("layout", ["tiled", "direct", "csr", "lut"])
def test_ragged_and_degenerate_shapes(torch, B, oracle, workloads, idx, layout):
    cfg = _ragged_cases(workloads)[idx]
    rng = np.random.default_rng(100 + idx)
    img = rng.poisson(50.0, size=(cfg.height, cfg.width)).astype(np.float32)
    mask = (rng.random(size=img.shape) < 0.1).astype(np.uint8)
    flat = rng.uniform(0.8, 1.2, size=img.shape).astype(np.float32)
    fr = workloads.Frame(image=img, flat=flat, mask=mask)
    integ = B.Integrator(cfg, layout=LAYOUTS[layout], empty_value=-7.0)
    got = _run(torch, integ, fr)
    want = _oracle_profile(oracle, cfg, fr, empty=-7.0)
    assert_profile(got, want, what=f"{cfg.name}/{layout}")
    empty = want["count"] <= 0
    assert np.all(got["intensity"][empty] == -7.0)
    integ.close()


def test_unaligned_buffers_take_the_scalar_path(torch, B, oracle, workloads):
    cfg = workloads.CONFIGS["cfg1b"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg)
    buf = torch.zeros(cfg.npix + 1, dtype=torch.float32, device="cuda")
    buf[1:] = torch.from_numpy(fr.image).cuda().ravel()          # 4-byte aligned only
    mbuf = torch.zeros(cfg.npix + 3, dtype=torch.uint8, device="cuda")
    mask = (np.random.default_rng(5).random(cfg.npix) < 0.05).astype(np.uint8)
    mbuf[3:] = torch.from_numpy(mask).cuda()
    i, s, c = integ.integrate1d(buf[1:], mask=mbuf[3:])
    torch.cuda.synchronize()
    got = {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}
    want = _oracle_profile(oracle, cfg, workloads.Frame(image=fr.image, mask=mask.reshape(cfg.height, cfg.width)))
    assert_profile(got, want, what="unaligned")
    integ.close()


@pytest.mark.parametrize("layout", ["tiled", "direct", "csr", "lut"])
def test_all_masked_and_non_finite_pixels(torch, B, oracle, workloads, layout):
    cfg = workloads.CONFIGS["cfg1b"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg, layout=LAYOUTS[layout], empty_value=-1.0)
    everything = np.ones((cfg.height, cfg.width), dtype=np.uint8)
    got = _run(torch, integ, workloads.Frame(image=fr.image, mask=everything))
    assert np.all(got["intensity"] == -1.0) and np.all(got["count"] == 0) and np.all(got["sum_signal"] == 0)
    # NaN / Inf pixels and zero flat-field behave like masked pixels (reading 8; oracle O5)
    img = fr.image.copy()
    img[5, 7] = np.nan
    img[100, 100] = np.inf
    flat = np.ones_like(img)
    flat[200, 13] = 0.0
    fr2 = workloads.Frame(image=img, flat=flat)
    assert_profile(_run(torch, integ, fr2), _oracle_profile(oracle, cfg, fr2, empty=-1.0), what="non-finite")
    integ.close()


def test_results_are_bit_reproducible(torch, B, workloads):
    cfg = workloads.CONFIGS["cfg2"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg)
    a = _run(torch, integ, fr)
    for _ in range(3):
        b = _run(torch, integ, fr)
        for k in a:
            assert np.array_equal(a[k], b[k])
    integ.close()


@pytest.mark.parametrize("corrected", [False, True])
def test_back_to_back_launches_do_not_interfere(torch, B, workloads, corrected):
    """Launches chained by programmatic dependent launch overlap (the next kernel's prologue runs while the previous
    one drains) and share the context's partial buffer, ticket counter and barrier counter: a train of calls on
    rotating frames and two contexts must give, bit for bit, what the same calls give one at a time."""
    cfg = workloads.CONFIGS["cfg2"]
    rng = np.random.default_rng(11)
    base = workloads.make_frame(cfg).image
    frames = [torch.from_numpy(base * np.float32(s)).cuda() for s in (1.0, 0.5, 2.0, 3.0, 0.25)]
    mask = torch.from_numpy((rng.random(base.shape) < 0.03).astype(np.uint8)).cuda() if corrected else None
    integs = [B.Integrator(cfg), B.Integrator(cfg)]
    ref = []
    for k in range(len(frames)):
        out = integs[0].integrate1d(frames[k], mask=mask)
        torch.cuda.synchronize()
        ref.append([o.clone() for o in out])
    n = 60
    outs = [[integs[j].outputs() for _ in range(n)] for j in range(2)]
    for k in range(n):
        integs[k % 2].integrate1d(frames[k % len(frames)], mask=mask, out=outs[k % 2][k])
    torch.cuda.synchronize()
    for k in range(n):
        for a, b in zip(outs[k % 2][k], ref[k % len(frames)]):
            assert torch.equal(a, b), f"call {k} differs from the same call run alone"
    for it in integs:
        it.close()


def test_mixed_call_sequence_is_bit_reproducible(torch, B, workloads):
    """A random sequence of plain, masked and batched calls on two contexts (one of them with rows off 16-byte
    boundaries), enqueued without synchronising: every result equals, bit for bit, the result of the same call run
    alone.  Exercises the launch chain across all streamed kernels and the pre-pass."""
    rng = np.random.default_rng(5)
    cfgs = [workloads.CONFIGS["cfg1b"],
            workloads.tiny_config(333, 301, center_x=150.2, center_y=170.9, unit=workloads.TTH_DEG, npt=400,
                                  distance_m=0.03, name="odd_width")]
    ctxs = [B.Integrator(c) for c in cfgs]
    frames = [[torch.from_numpy(rng.poisson(50.0, size=(c.height, c.width)).astype(np.float32)).cuda() for _ in range(3)]
              for c in cfgs]
    masks = [torch.from_numpy((rng.random((c.height, c.width)) < 0.05).astype(np.uint8)).cuda() for c in cfgs]
    batches = [torch.stack(f) for f in frames]

    def run(kind, j, k):
        if kind == 0:
            return ctxs[j].integrate1d(frames[j][k])
        if kind == 1:
            return ctxs[j].integrate1d(frames[j][k], mask=masks[j])
        return ctxs[j].integrate1d_batch(batches[j])

    ref = {}
    for kind in range(3):
        for j in range(2):
            for k in range(3):
                out = run(kind, j, k)
                torch.cuda.synchronize()
                ref[(kind, j, k)] = [t.clone() for t in out]
    plan = [(int(rng.integers(0, 3)), int(rng.integers(0, 2)), int(rng.integers(0, 3))) for _ in range(300)]
    outs = [(key, run(*key)) for key in plan]
    torch.cuda.synchronize()
    for n, (key, out) in enumerate(outs):
        for a, b in zip(out, ref[key]):
            assert torch.equal(a, b), f"call {n} {key} differs from the same call run alone"
    for it in ctxs:
        it.close()


@pytest.mark.parametrize("masked", [False, True])
def test_two_contexts_on_two_streams(torch, B, workloads, masked):
    """Two contexts driven from two streams at once (another tenant on the GPU): blocks of either context's stream kernel
    become resident out of turn, so the launch chain's "one block per SM" argument for re-using a set of partial sums
    (and a corrected frame) every second call does not hold by itself -- the kernels check the count of ended finish
    kernels.  3000 bins (BASELINE.json configs[2]'s shape), a few hundred calls per context, every call's result compared
    with the context's isolated result for that frame, bit for bit."""
    cfg = workloads.CONFIGS["cfg3"]
    base = workloads.make_frame(cfg)
    rng = np.random.default_rng(42)
    frames = [torch.from_numpy(base.image * np.float32(s)).cuda() for s in (1.0, 0.5, 2.0)]
    mask = torch.from_numpy(base.mask).cuda() if masked else None
    ctxs = [B.Integrator(cfg), B.Integrator(cfg)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ref = []
    for it in ctxs:                                  # isolated results, one call at a time
        r = []
        for f in frames:
            o = it.integrate1d(f, mask=mask)
            torch.cuda.synchronize()
            r.append(tuple(t.clone() for t in o))
        ref.append(r)
    ncalls = 240
    outs = [[tuple(torch.empty(cfg.npt, dtype=torch.float32, device="cuda") for _ in range(3)) for _ in range(ncalls)]
            for _ in ctxs]
    order = rng.integers(0, 3, size=(2, ncalls))
    torch.cuda.synchronize()
    k = [0, 0]
    while k[0] < ncalls or k[1] < ncalls:            # enqueue in uneven bursts so that the two chains drift past each other
        j = int(rng.integers(0, 2))
        for _ in range(int(rng.integers(1, 9))):
            if k[j] < ncalls:
                with torch.cuda.stream(streams[j]):
                    ctxs[j].integrate1d(frames[order[j, k[j]]], mask=mask, out=outs[j][k[j]])
                k[j] += 1
    torch.cuda.synchronize()
    for j in range(2):
        for n in range(ncalls):
            want = ref[j][order[j, n]]
            got = outs[j][n]
            assert torch.equal(got[0], want[0]) and torch.equal(got[1], want[1]) and torch.equal(got[2], want[2]), (j, n)
    for it in ctxs:
        it.close()


def test_compensation_keeps_small_terms(torch, B, workloads):
    """Kahan summation lets single precision give accurate sums.  One bin, one pixel of 2^24 and
    65535 pixels of 1: the exact sum is 2^24 + 65535; every lane that holds the big value would drop the ones without
    compensation."""
    cfg = workloads.scaled(workloads.CONFIGS["cfg1"], npt=1)
    img = np.ones((cfg.height, cfg.width), dtype=np.float32)
    img[0, 0] = 2.0 ** 24
    exact = 2.0 ** 24 + cfg.npix - 1
    for layout in ("tiled", "csr", "lut"):
        for accum in ("kahan", "f64"):
            integ = B.Integrator(cfg, layout=LAYOUTS[layout], accum=ACCUMS[accum])
            got = _run(torch, integ, workloads.Frame(image=img))
            assert abs(float(got["sum_signal"][0]) - exact) <= 1.0, (layout, accum)      # fp32 output spacing is 2
            integ.close()
    integ = B.Integrator(cfg, layout=LAYOUTS["lut"], accum=ACCUMS["plain"])
    got = _run(torch, integ, workloads.Frame(image=img))
    # sequential uncompensated fp32 loses every 1 added after the big value: it is visibly wrong
    assert abs(float(got["sum_signal"][0]) - exact) > 1000.0
    integ.close()


# ----------------------------------------------------------------------------------------------------------------------
# the two pipelined stage-1 kernels: single-frame stream kernel (default for plain 32-bit frames) and the general one
# ----------------------------------------------------------------------------------------------------------------------
def _run_raw(torch, B, integ, img, dtype):
    if dtype == "uint32":
        t, code = torch.from_numpy(img.view(np.int32)).cuda(), B.AI_U32
    else:
        t, code = torch.from_numpy(img).cuda(), None
    i, s, c = integ.outputs()
    B.ai_integrate1d(integ.ctx, t, None, None, None, None, None, None, i, s, c, dtype=code)
    torch.cuda.synchronize()
    return {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}


@pytest.mark.parametrize("path", ["stream", "pipe"])
@pytest.mark.parametrize("dtype", ["float32", "int32", "uint32"])
@pytest.mark.parametrize("shape", [(256, 256), (130, 200), (70, 1028), (97, 131)])
def test_single_frame_kernels(torch, B, oracle, workloads, monkeypatch, path, dtype, shape):
    """ai_path_options.no_stream sends single plain frames through the general pipelined kernel.  A width
    that is not a multiple of 4 (rows off 16-byte boundaries) reaches the single-frame kernel through the pre-pass,
    which re-pitches the frame."""
    if path == "pipe":
        monkeypatch.setitem(B.PATH_DEFAULTS, "no_stream", 1)
    h, w = shape
    cfg = workloads.tiny_config(h, w, center_x=w * 0.41, center_y=h * 0.57, unit=workloads.Q_NM, npt=173,
                                distance_m=0.02, name=f"single_{h}x{w}")
    rng = np.random.default_rng(h * 1000 + w)
    img = rng.poisson(200.0, size=(h, w)).astype(dtype)
    integ = B.Integrator(cfg)
    for acc in ("kahan", "f64"):
        integ.set_options(LAYOUTS["tiled"], ACCUMS[acc])
        got = _run_raw(torch, B, integ, img, dtype)
        assert_profile(got, _oracle_profile(oracle, cfg, workloads.Frame(image=img)), what=f"{path}/{dtype}/{shape}/{acc}")
    integ.close()


@pytest.mark.parametrize("path", ["prepass", "pipe"])
@pytest.mark.parametrize("dtype", ["float32", "uint16", "int32"])
@pytest.mark.parametrize("shape", [(256, 256), (130, 200)])
def test_corrected_frame_kernels(torch, B, oracle, workloads, monkeypatch, path, dtype, shape):
    """One frame with every correction array and a mask: by default H1 + H2 run as a pre-pass and the single-frame
    kernel consumes the corrected frame; ai_path_options.no_prepass stages the corrections inside the general kernel."""
    if path == "pipe":
        monkeypatch.setitem(B.PATH_DEFAULTS, "no_prepass", 1)
    h, w = shape
    cfg = workloads.tiny_config(h, w, center_x=w * 0.3, center_y=h * 0.6, unit=workloads.TTH_DEG, npt=211,
                                distance_m=0.03, name=f"corr_{h}x{w}")
    rng = np.random.default_rng(h + 7 * w)
    img = rng.poisson(300.0, size=(h, w)).astype(dtype)
    fr = workloads.Frame(image=img, dark=rng.poisson(5.0, size=(h, w)).astype(np.float32),
                         flat=rng.uniform(0.9, 1.1, size=(h, w)).astype(np.float32),
                         solidangle=rng.uniform(0.7, 1.0, size=(h, w)).astype(np.float32),
                         polarization=rng.uniform(0.95, 1.0, size=(h, w)).astype(np.float32),
                         mask=(rng.random(size=(h, w)) < 0.05).astype(np.uint8))
    fr.flat[3, 5] = 0.0                      # zero denominator: invalid pixel
    integ = B.Integrator(cfg, empty_value=-2.0)
    args = [_dev(torch, x) for x in (fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)]
    if dtype == "uint16":
        t, code = torch.from_numpy(img.view(np.int16)).cuda(), B.AI_U16
    else:
        t, code = torch.from_numpy(img).cuda(), None
    for acc in ("kahan", "f64"):
        integ.set_options(LAYOUTS["tiled"], ACCUMS[acc], -2.0)
        i, s, c = integ.outputs()
        B.ai_integrate1d(integ.ctx, t, *args, None, i, s, c, dtype=code)
        torch.cuda.synchronize()
        got = {"intensity": i.cpu().numpy(), "sum_signal": s.cpu().numpy(), "count": c.cpu().numpy()}
        assert_profile(got, _oracle_profile(oracle, cfg, fr, empty=-2.0), what=f"{path}/{dtype}/{shape}/{acc}")
    assert B.ai_last_launch_count(integ.ctx) == (3 if path == "prepass" else 2)
    integ.close()


@pytest.mark.parametrize("path", ["stream", "pipe"])
def test_non_finite_pixels_in_plain_float_frames(torch, B, oracle, workloads, monkeypatch, path):
    """No mask, no corrections: NaN / Inf pixels are found lazily (a non-finite lane sum repeats the block with the
    tracked variant) and behave like masked pixels (oracle O5)."""
    if path == "pipe":
        monkeypatch.setitem(B.PATH_DEFAULTS, "no_stream", 1)
    cfg = workloads.CONFIGS["cfg1b"]
    img = workloads.make_frame(cfg).image.copy()
    rng = np.random.default_rng(77)
    bad = rng.integers(0, cfg.npix, size=40)
    img.ravel()[bad[:20]] = np.nan
    img.ravel()[bad[20:30]] = np.inf
    img.ravel()[bad[30:]] = -np.inf
    img[0, 0] = np.inf                      # pixel 0 of a tile: where padding entries point
    integ = B.Integrator(cfg, empty_value=-3.0)
    fr = workloads.Frame(image=img)
    assert_profile(_run(torch, integ, fr), _oracle_profile(oracle, cfg, fr, empty=-3.0), what=f"non-finite/{path}")
    integ.close()


# ----------------------------------------------------------------------------------------------------------------------
# H6: batch
# ----------------------------------------------------------------------------------------------------------------------
def test_batch_matches_oracle_small(torch, B, oracle, workloads):
    cfg = workloads.scaled(workloads.CONFIGS["cfg4"], height=256, width=256, center_x_px=128.0, center_y_px=128.0,
                           distance_m=0.025, npt=300)
    frames = workloads.make_frames(cfg, 5)
    integ = B.Integrator(cfg)
    i, s, c = integ.integrate1d_batch(torch.from_numpy(frames).cuda())
    torch.cuda.synchronize()
    for f in range(5):
        want = _oracle_profile(oracle, cfg, workloads.Frame(image=frames[f]))
        got = {"intensity": i[f].cpu().numpy(), "sum_signal": s[f].cpu().numpy(), "count": c[f].cpu().numpy()}
        assert_profile(got, want, what=f"batch frame {f}")
    integ.close()


@pytest.mark.parametrize("path", ["bstream", "pipe", "fl"])
@pytest.mark.parametrize("dtype,nframes", [("int32", 7), ("float32", 6), ("uint32", 2), ("float32", 33)])
def test_batch_kernels(torch, B, oracle, workloads, monkeypatch, path, dtype, nframes):
    """Batches of plain 32-bit frames take the two-frames-at-a-time stream kernel; ai_path_options.no_stream sends them
    through the general pipelined kernel, ai_path_options.force_fl through the frame-lane kernel (tests/test_gpu_parity_fl.py has
    more of those).  Odd counts leave a single last frame; float frames carry NaN / Inf."""
    if path == "pipe":
        monkeypatch.setitem(B.PATH_DEFAULTS, "no_stream", 1)
    if path == "fl":
        monkeypatch.setitem(B.PATH_DEFAULTS, "force_fl", 1)
    cfg = workloads.tiny_config(200, 264, center_x=100.3, center_y=90.1, unit=workloads.Q_NM, npt=257,
                                distance_m=0.02, name="batch_small")
    rng = np.random.default_rng(nframes)
    frames = rng.poisson(100.0, size=(nframes, cfg.height, cfg.width)).astype(dtype)
    if dtype == "float32":
        frames[1, 17, 33] = np.nan
        frames[nframes - 1, 100, 200] = np.inf
    if dtype == "uint32":
        t, code = torch.from_numpy(frames.view(np.int32)).cuda(), B.AI_U32
    else:
        t, code = torch.from_numpy(frames).cuda(), None
    integ = B.Integrator(cfg)
    i, s, c = integ.outputs(nframes)
    B.ai_integrate1d_batch(integ.ctx, t, nframes, cfg.npix, None, None, None, None, None, i, s, c, dtype=code)
    torch.cuda.synchronize()
    for f in range(nframes):
        want = _oracle_profile(oracle, cfg, workloads.Frame(image=frames[f]))
        got = {"intensity": i[f].cpu().numpy(), "sum_signal": s[f].cpu().numpy(), "count": c[f].cpu().numpy()}
        assert_profile(got, want, what=f"{path}/{dtype}/frame {f} of {nframes}")
    integ.close()


def test_batch_equals_single_frame_calls_bit_for_bit(torch, B, oracle, workloads):
    """BASELINE.json configs[1] frames through ai_integrate1d_batch in a small batch (the slice-per-lane batch kernel,
    bench.py's `batch_cfg2_64_frames.slice_per_lane_kernel_no_fl`): every frame's profiles equal, bit for bit,
    what ai_integrate1d gives for it (same accumulation order in both kernels), and a sampled frame matches the oracle."""
    cfg = workloads.CONFIGS["cfg2"]
    base = workloads.make_frame(cfg).image
    frames = np.stack([base * np.float32(s) for s in (1.0, 0.5, 2.0, 0.75, 3.0)])
    dev = torch.from_numpy(frames).cuda()
    integ = B.Integrator(cfg)
    bi, bs, bc = integ.integrate1d_batch(dev)
    torch.cuda.synchronize()
    for f in range(frames.shape[0]):
        i, s, c = integ.integrate1d(dev[f])
        torch.cuda.synchronize()
        assert torch.equal(bi[f], i) and torch.equal(bs[f], s) and torch.equal(bc[f], c), f"frame {f}"
    want = _oracle_profile(oracle, cfg, workloads.Frame(image=frames[3]))
    got = {"intensity": bi[3].cpu().numpy(), "sum_signal": bs[3].cpu().numpy(), "count": bc[3].cpu().numpy()}
    assert_profile(got, want, what="cfg2 batch frame 3")
    integ.close()


@pytest.mark.parametrize("path", ["frame by frame", "general kernel"])
def test_small_batch_with_mask(torch, B, oracle, workloads, monkeypatch, path):
    """A small batch with a mask: frame by frame through the pre-pass + single-frame kernel (3 launches per frame), or,
    without the pre-pass (ai_path_options.no_prepass), the general batched kernel that stages the corrections itself."""
    if path == "general kernel":
        monkeypatch.setitem(B.PATH_DEFAULTS, "no_prepass", 1)
    cfg = workloads.tiny_config(130, 200, center_x=60.0, center_y=70.0, unit=workloads.TTH_DEG, npt=150,
                                distance_m=0.03, name="batch_mask")
    rng = np.random.default_rng(3)
    frames = rng.poisson(50.0, size=(4, cfg.height, cfg.width)).astype(np.int32)
    mask = (rng.random(size=(cfg.height, cfg.width)) < 0.1).astype(np.uint8)
    integ = B.Integrator(cfg)
    i, s, c = integ.integrate1d_batch(torch.from_numpy(frames).cuda(), mask=torch.from_numpy(mask).cuda())
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == (12 if path == "frame by frame" else 2)
    for f in range(4):
        want = _oracle_profile(oracle, cfg, workloads.Frame(image=frames[f], mask=mask))
        got = {"intensity": i[f].cpu().numpy(), "sum_signal": s[f].cpu().numpy(), "count": c[f].cpu().numpy()}
        assert_profile(got, want, what=f"masked batch frame {f}")
    integ.close()


def test_batch_full_size_sampled(torch, B, oracle, workloads):
    """BASELINE.json configs[3] at full size: 1024 frames of 1024x1024 int32 in one call (the launch configuration
    bench.py times).  The frames cycle through a pool of 8 distinct seeded frames; sampled outputs are compared with
    the oracle, and every output row must equal the row of its pool frame bit for bit."""
    cfg = workloads.CONFIGS["cfg4"]
    pool = workloads.make_frames(cfg, 8)
    dev_pool = torch.from_numpy(pool).cuda()
    frames = dev_pool.repeat(cfg.nframes // 8, 1, 1)
    assert frames.shape[0] == 1024
    integ = B.Integrator(cfg)
    i, s, c = integ.integrate1d_batch(frames)
    torch.cuda.synchronize()
    for f in (0, 3, 517, 1023):
        want = _oracle_profile(oracle, cfg, workloads.Frame(image=pool[f % 8]))
        got = {"intensity": i[f].cpu().numpy(), "sum_signal": s[f].cpu().numpy(), "count": c[f].cpu().numpy()}
        assert_profile(got, want, what=f"cfg4 frame {f}")
    ref = i[:8].repeat(cfg.nframes // 8, 1)
    assert torch.equal(i, ref)
    integ.close()


# ----------------------------------------------------------------------------------------------------------------------
# end-to-end host entry point and error behaviour
# ----------------------------------------------------------------------------------------------------------------------
def test_host_entry_point(torch, B, oracle, workloads):
    cfg = workloads.CONFIGS["cfg1b"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg)
    host = torch.from_numpy(fr.image).pin_memory()
    out = [torch.empty(cfg.npt, dtype=torch.float32).pin_memory() for _ in range(3)]
    B.ai_integrate1d_host(integ.ctx, host.numpy(), None, None, None, None, None, out[0].numpy(), out[1].numpy(),
                          out[2].numpy(), dtype=B.AI_F32)
    got = {"intensity": out[0].numpy(), "sum_signal": out[1].numpy(), "count": out[2].numpy()}
    assert_profile(got, _oracle_profile(oracle, cfg, fr), what="host entry")
    assert B.ai_last_launch_count(integ.ctx) >= 1
    integ.close()


def test_host_frames_entry_point(torch, B, oracle, workloads):
    """ai_integrate1d_host_frames: pinned host frames in, host profiles out, uploads overlapping the kernels."""
    cfg = workloads.CONFIGS["cfg1b"]
    frames = np.stack([workloads.make_frame(cfg, frame_index=k).image for k in range(5)])
    pinned = torch.from_numpy(frames).pin_memory()
    outs = [torch.empty((5, cfg.npt), dtype=torch.float32).pin_memory() for _ in range(3)]
    integ = B.Integrator(cfg)
    for _ in range(2):       # second call reuses the staging buffers
        B.ai_integrate1d_host_frames(integ.ctx, pinned.numpy(), 5, cfg.npix, None, None, None, None, None,
                                     *[o.numpy() for o in outs])
    for k in range(5):
        got = {"intensity": outs[0][k].numpy(), "sum_signal": outs[1][k].numpy(), "count": outs[2][k].numpy()}
        assert_profile(got, _oracle_profile(oracle, cfg, workloads.Frame(image=frames[k])), what=f"host frame {k}")
    integ.close()


def test_host_frames_in_chunks_with_a_mask_and_a_stride(torch, B, oracle, workloads):
    """19 frames = two chunks of 8 and one of 3, each one batched launch; frames 2 elements apart more than a frame."""
    cfg = workloads.CONFIGS["cfg1b"]
    nf, stride = 19, cfg.npix + 8
    rng = np.random.default_rng(31)
    buf = np.zeros(nf * stride, dtype=np.float32)
    frames = []
    for k in range(nf):
        fr = rng.poisson(40.0 + 3 * k, size=cfg.npix).astype(np.float32)
        buf[k * stride:k * stride + cfg.npix] = fr
        frames.append(fr.reshape(cfg.height, cfg.width))
    mask = (rng.random((cfg.height, cfg.width)) < 0.05).astype(np.uint8)
    pinned = torch.from_numpy(buf).pin_memory()
    outs = [torch.empty((nf, cfg.npt), dtype=torch.float32).pin_memory() for _ in range(3)]
    integ = B.Integrator(cfg)
    B.ai_integrate1d_host_frames(integ.ctx, pinned.numpy(), nf, stride, None, None, None, None, _dev(torch, mask),
                                 *[o.numpy() for o in outs])
    for k in (0, 7, 8, 15, 16, 18):
        got = {"intensity": outs[0][k].numpy(), "sum_signal": outs[1][k].numpy(), "count": outs[2][k].numpy()}
        assert_profile(got, _oracle_profile(oracle, cfg, workloads.Frame(image=frames[k], mask=mask)), what=f"host frame {k}")
    integ.close()


@pytest.mark.parametrize("name", ["cfg1b", "cfg2", "cfg3"])
def test_scatter_comparison_path(torch, B, oracle, workloads, parity_report, name):
    """AI_LAYOUT_SCATTER: forward scatter with fp32 atomics -- uncompensated, order not fixed: held
    to 2e-5 and reported."""
    cfg = workloads.CONFIGS[name]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg, layout=B.AI_LAYOUT_SCATTER)
    got = _run(torch, integ, fr, radial=True)
    want = _oracle_profile(oracle, cfg, fr)
    worst = assert_profile(got, want, tol=2e-5, what=f"scatter/{name}")
    again = _run(torch, integ, fr)
    worst["bit_reproducible_in_this_run"] = bool(np.array_equal(got["sum_signal"], again["sum_signal"]))
    print("scatter", name, worst)
    parity_report.setdefault("scatter_with_atomics", {})[name] = worst
    # a small batch through the same path
    if name == "cfg1b":
        frames = np.stack([fr.image, fr.image * 2]).astype(np.float32)
        i, s, c = integ.integrate1d_batch(_dev(torch, frames))
        torch.cuda.synchronize()
        got1 = {"intensity": i[1].cpu().numpy(), "sum_signal": s[1].cpu().numpy(), "count": c[1].cpu().numpy()}
        assert_profile(got1, _oracle_profile(oracle, cfg, workloads.Frame(image=frames[1])), tol=2e-5, what="scatter batch")
    integ.close()


@pytest.mark.parametrize("name", ["cfg1b", "cfg3"])
def test_split_normalisation(torch, B, oracle, workloads, name):
    """ai_set_normalization(AI_NORM_SPLIT): sum c (I - dark) over sum c (flat * solidangle * polarization)."""
    cfg = workloads.CONFIGS[name]
    fr = workloads.make_frame(cfg)
    if not cfg.corrections:
        rng = np.random.default_rng(41)
        shape = fr.image.shape
        fr = workloads.Frame(image=fr.image, dark=rng.poisson(5.0, shape).astype(np.float32),
                             flat=rng.uniform(0.9, 1.1, shape).astype(np.float32),
                             solidangle=rng.uniform(0.8, 1.0, shape).astype(np.float32),
                             polarization=rng.uniform(0.95, 1.0, shape).astype(np.float32),
                             mask=(rng.random(shape) < 0.04).astype(np.uint8))
    umin, umax, u0, u1 = _oracle_bounds(oracle, cfg)
    want = oracle.integrate1d_bounds_split(umin, umax, cfg.npt, u0, u1, fr.image, fr.dark, fr.flat, fr.solidangle,
                                           fr.polarization, fr.mask)
    integ = B.Integrator(cfg)
    B.ai_set_normalization(integ.ctx, B.AI_NORM_SPLIT)
    got = _run(torch, integ, fr)
    for key in ("intensity", "sum_signal", "count"):
        e = rel_err(got[key], want[key])
        assert e.max() <= 1e-6, (name, key, float(e.max()))
    # a frame without corrections: the two estimators coincide
    plain = workloads.Frame(image=fr.image)
    got_p = _run(torch, integ, plain)
    B.ai_set_normalization(integ.ctx, B.AI_NORM_PIXEL)
    ref_p = _run(torch, integ, plain)
    assert np.allclose(got_p["intensity"], ref_p["intensity"], rtol=1e-6)
    # batches are refused in this mode, not silently computed with the other estimator
    B.ai_set_normalization(integ.ctx, B.AI_NORM_SPLIT)
    with pytest.raises(B.AzintError):
        integ.integrate1d_batch(_dev(torch, np.stack([fr.image, fr.image])))
    integ.close()


def test_layout_info(torch, B, workloads):
    """ai_get_layout_info: sizes of the execution layout, consistent with the canonical CSR."""
    cfg = workloads.CONFIGS["cfg2"]
    integ = B.Integrator(cfg)
    info = B.ai_get_layout_info(integ.ctx)
    nnz = B.ai_get_csr(integ.ctx)[3]
    assert info["tile_h"] in (8, 16, 32, 64)
    assert info["ntiles"] == ((cfg.height + info["tile_h"] - 1) // info["tile_h"]) * ((cfg.width + 63) // 64)
    assert nnz <= info["padded_entries"] <= nnz + 4 * info["nseg"]          # segments padded to multiples of 4
    assert 6 * info["padded_entries"] <= info["blob_bytes"] <= 8 * info["padded_entries"]   # < the CSR's 8 B/entry
    assert info["max_blob_bytes"] * info["ntiles"] >= info["blob_bytes"]
    assert info["nseg"] <= info["nslot"] <= 4 * info["nseg"]
    assert info["stream_stages"] >= 2
    integ.close()


def test_error_codes_on_device(torch, B, workloads):
    cfg = workloads.CONFIGS["cfg1"]
    integ = B.Integrator(cfg)
    i, s, c = integ.outputs()
    with pytest.raises(B.AzintError) as e:
        B.ai_integrate1d(integ.ctx, None, None, None, None, None, None, None, i, s, c, dtype=B.AI_F32)
    assert e.value.code == B.AI_EINVAL
    with pytest.raises(B.AzintError) as e:
        B.ai_set_options(integ.ctx, 9, 0, 0.0)
    assert e.value.code == B.AI_EINVAL
    integ.close()


@pytest.mark.parametrize("layout", ["csr", "lut", "scatter"])
def test_comparison_layouts_refuse_more_frames_than_the_grid_holds(torch, B, workloads, layout):
    """Frames ride on gridDim.y (<= 65535) in the comparison layouts: a larger batch is refused, not mis-launched."""
    W = workloads
    cfg = W.tiny_config(4, 4, center_x=2.0, center_y=2.0, unit=W.R_MM, npt=3, name="many_frames")
    code = {"csr": B.AI_LAYOUT_CSR, "lut": B.AI_LAYOUT_LUT, "scatter": B.AI_LAYOUT_SCATTER}[layout]
    integ = B.Integrator(cfg, layout=code)
    n = 65536
    frames = torch.ones((n, 4, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(B.AzintError) as e:
        integ.integrate1d_batch(frames)
    assert e.value.code == B.AI_EUNSUPPORTED and "65535" in str(e.value)
    i, s, c = integ.integrate1d_batch(frames[:65535])
    torch.cuda.synchronize()
    assert torch.allclose(i, torch.ones_like(i), rtol=1e-6)
    integ.close()


def test_train_with_a_producer_kernel_before_every_call(torch, B, workloads):
    """include/azint.h (ai_integrate1d, reading 25 of DESIGN.md 3.2): consecutive calls overlap on the GPU, and a call may
    read its frame as soon as the kernel enqueued right before it has completed or triggered its dependents early; an
    ordinary kernel never triggers early, so it gives plain stream ordering.  The everyday pipeline "a kernel writes the
    frame (decompression, a cast), then integrate": 200 calls on one buffer that an elementwise torch kernel rewrites
    immediately before every call with one of two contents -- every profile bit-equal to the isolated call's."""
    W = workloads
    cfg = W.CONFIGS["cfg2"]
    integ = B.Integrator(cfg)
    src = [torch.from_numpy(W.make_frame(cfg, k).image).cuda() for k in range(2)]
    ref = []
    for k in range(2):
        out = integ.integrate1d(src[k], out=integ.outputs())
        torch.cuda.synchronize()
        ref.append(out)
    assert not torch.equal(ref[0][1], ref[1][1])
    buf = torch.empty_like(src[0])
    n = 200
    outs = integ.outputs(n)
    for k in range(n):
        torch.mul(src[k % 2], 1.0, out=buf)                 # an ordinary kernel, same stream, no synchronisation
        integ.integrate1d(buf, out=(outs[0][k], outs[1][k], outs[2][k]))
    torch.cuda.synchronize()
    assert B.ai_last_launch_count(integ.ctx) == 2           # the single-frame kernel chain, not a fallback
    for k in range(n):
        for q in range(3):
            assert torch.equal(outs[q][k], ref[k % 2][q]), (k, q)
    # the same with corrections: the library's own pre-pass sits between the producer and the stream kernel
    cfg3 = W.CONFIGS["cfg3"]
    fr = [W.make_frame(cfg3, k) for k in range(2)]
    cor = [_dev(torch, x) for x in (fr[0].dark, fr[0].flat, fr[0].solidangle, fr[0].polarization, fr[0].mask)]
    integ3 = B.Integrator(cfg3)
    src = [_dev(torch, f.image) for f in fr]
    ref = []
    for k in range(2):
        out = integ3.integrate1d(src[k], *cor, out=integ3.outputs())
        torch.cuda.synchronize()
        ref.append(out)
    outs = integ3.outputs(n)
    for k in range(n):
        torch.mul(src[k % 2], 1.0, out=buf)
        integ3.integrate1d(buf, *cor, out=(outs[0][k], outs[1][k], outs[2][k]))
    torch.cuda.synchronize()
    for k in range(n):
        for q in range(3):
            assert torch.equal(outs[q][k], ref[k % 2][q]), ("corrected", k, q)
    integ.close()
    integ3.close()
