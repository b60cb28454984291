"""ai_integrate1d_noalloc (include/azint.h, csrc/integrate_noalloc.cu): the entry point for callers that cannot allocate
device memory while they run -- a process in which another component (a framework's caching allocator, a per-tenant
budget) already owns all of it, so that a cudaMalloc inside the library fails; a real-time acquisition loop that a
cudaMalloc or a device-wide cudaFree in mid-run would stall.  Its partial sums live in a fixed 8 MiB array inside the
library instead of a buffer the context allocates; everything else (inputs, outputs, arithmetic) is ai_integrate1d's.

Checked here: the profiles against the existing path (the default layout within the 1e-6 per-bin bar of the other parity
tests, the block-per-tile layout bit for bit) and against the oracle, on two calls in a row that share the array -- the
second on another context with a different matrix, so that records the first left behind would show; that repeated calls
leave the device's free memory unchanged; that a matrix beyond the array's size is refused with a text that says so.
The file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity tests.
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


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _host(out):
    return {"intensity": out[0].cpu().numpy(), "sum_signal": out[1].cpu().numpy(), "count": out[2].cpu().numpy()}


def _as_want(d):
    return {k: v.astype(np.float64) for k, v in d.items()}


def _corrections(shape, seed):
    rng = np.random.default_rng(seed)
    dark = rng.poisson(5.0, shape).astype(np.float32)
    flat = rng.uniform(0.9, 1.1, shape).astype(np.float32)
    solid = rng.uniform(0.7, 1.0, shape).astype(np.float32)
    pol = rng.uniform(0.95, 1.0, shape).astype(np.float32)
    mask = (rng.random(shape) < 0.04).astype(np.uint8)
    mask[shape[0] // 2 - 8:shape[0] // 2 + 8, :] = 1        # a gap stripe: whole tiles without a valid pixel
    flat[3, 5] = 0.0                                         # the degenerate pixels of the method
    flat[17, 40] = np.inf
    dark[29, 11] = np.nan
    return dark, flat, solid, pol, mask


def _oracle(oracle, cfg, image, arrays):
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    return oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, image, *arrays)


def test_two_calls_in_a_row_match_the_existing_path(torch, B, oracle, workloads):
    W = workloads
    # two detectors with different matrices (several tiles each, ragged edges, one width off the 4-pixel boundary)
    cfg_a = W.tiny_config(300, 264, center_x=120.3, center_y=140.7, unit=W.Q_NM, npt=257, distance_m=0.03, name="na_a")
    cfg_b = W.tiny_config(203, 331, center_x=-20.5, center_y=90.0, unit=W.TTH_DEG, npt=90, name="na_b")
    rng = np.random.default_rng(20261106)
    img_a = rng.poisson(200.0, (cfg_a.height, cfg_a.width)).astype(np.float32)
    img_b = rng.poisson(50.0, (cfg_b.height, cfg_b.width)).astype(np.int32)
    arr_a = _corrections(img_a.shape, 1)
    arr_b = (None,) * 5
    ia, ib = B.Integrator(cfg_a), B.Integrator(cfg_b)
    da, db = [_dev(torch, x) for x in (img_a, *arr_a)], [_dev(torch, x) for x in (img_b, *arr_b)]

    # the existing path first (default layout, then the block-per-tile layout the new entry is a variant of)
    ref_a = _host(ia.integrate1d(*da))
    ref_b = _host(ib.integrate1d(*db))
    ia.set_options(layout=B.AI_LAYOUT_TILED_DIRECT)
    ib.set_options(layout=B.AI_LAYOUT_TILED_DIRECT)
    dir_a = _host(ia.integrate1d(*da))
    dir_b = _host(ib.integrate1d(*db))
    ia.set_options()
    ib.set_options()

    # two calls in a row on the shared array, no synchronisation between them (same stream: ordered)
    rad = torch.empty(cfg_a.npt, dtype=torch.float32, device="cuda")
    out_a, out_b = ia.outputs(), ib.outputs()
    ia.integrate1d_noalloc(*da, out=out_a, radial=rad)
    ib.integrate1d_noalloc(*db, out=out_b)
    torch.cuda.synchronize()
    got_a, got_b = _host(out_a), _host(out_b)
    # ... and the first one again: the array now holds the records of the other matrix
    again_a = _host(ia.integrate1d_noalloc(*da))
    torch.cuda.synchronize()

    for got, ref, direct, what in ((got_a, ref_a, dir_a, "first call"), (got_b, ref_b, dir_b, "second call"),
                                   (again_a, ref_a, dir_a, "first call repeated")):
        assert_profile(got, _as_want(ref), what=what + " vs default layout")           # the tests' 1e-6 per-bin bar
        for k in ("intensity", "sum_signal", "count"):
            assert np.array_equal(got[k], direct[k]), (what, k, "not bit-identical to AI_LAYOUT_TILED_DIRECT")
    assert_profile(got_a, _oracle(oracle, cfg_a, img_a, arr_a), what="first call vs oracle")
    assert_profile(got_b, _oracle(oracle, cfg_b, img_b, arr_b), what="second call vs oracle")
    umin, umax = oracle.pixel_bounds(cfg_a)
    u0, u1 = oracle.auto_range(umin, umax)
    centres = u0 + (np.arange(cfg_a.npt) + 0.5) * (u1 - u0) / cfg_a.npt
    assert np.allclose(rad.cpu().numpy(), centres, rtol=1e-6)
    assert B.ai_last_launch_count(ia.ctx) == 2


@pytest.mark.parametrize("accum", ["kahan", "plain", "f64"])
@pytest.mark.parametrize("dtype", ["float32", "int32", "uint16", "int16", "uint32"])
def test_every_dtype_and_accumulator(torch, B, workloads, dtype, accum):
    W = workloads
    cfg = W.tiny_config(130, 200, center_x=61.3, center_y=40.7, unit=W.R_MM, npt=77, name="na_dt")
    rng = np.random.default_rng(7)
    img = rng.poisson(300.0, (cfg.height, cfg.width)).astype(dtype)
    acc = {"kahan": B.AI_ACC_F32_KAHAN, "plain": B.AI_ACC_F32_PLAIN, "f64": B.AI_ACC_F64}[accum]
    integ = B.Integrator(cfg, layout=B.AI_LAYOUT_TILED_DIRECT, accum=acc)
    if dtype in ("uint16", "uint32") and not hasattr(torch, dtype):
        pytest.skip("torch without " + dtype)
    d = _dev(torch, img)
    want = _host(integ.integrate1d(d))
    got = _host(integ.integrate1d_noalloc(d))
    for k in ("intensity", "sum_signal", "count"):
        assert np.array_equal(got[k], want[k]), k


def test_headline_frame_and_no_allocation(torch, B, workloads):
    """cfg2 (2048 x 2048, 1000 bins: 103 132 records of 16 bytes, well inside the array) against the default path, and
    the device's free memory before and after a run of calls."""
    W = workloads
    cfg = W.CONFIGS["cfg2"]
    integ = B.Integrator(cfg)
    records = B.ai_get_layout_info(integ.ctx)["nslot"]
    assert 0 < records * 16 <= B.AI_NOALLOC_SCRATCH_BYTES
    frame = _dev(torch, W.make_frame(cfg).image)
    other = _dev(torch, W.make_frame(cfg, 1).image)
    ref = _host(integ.integrate1d(frame))
    ref_other = _host(integ.integrate1d(other))
    out, out2 = integ.outputs(), integ.outputs()
    integ.integrate1d_noalloc(frame, out=out)                  # the first call on the device: set-up included
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(10):
        integ.integrate1d_noalloc(other, out=out2)
        integ.integrate1d_noalloc(frame, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, "device memory changed hands during ai_integrate1d_noalloc calls"
    assert_profile(_host(out), _as_want(ref), what="cfg2 vs default layout")
    assert_profile(_host(out2), _as_want(ref_other), what="cfg2, other frame vs default layout")


def test_a_matrix_beyond_the_array_is_refused(torch, B, workloads):
    W = workloads
    # many narrow bins over a 2048 x 2048 detector: more (tile, bin) records than the array holds
    cfg = W.scaled(W.CONFIGS["cfg2"], npt=12000, name="na_big")
    integ = B.Integrator(cfg)
    records = B.ai_get_layout_info(integ.ctx)["nslot"]
    assert records * 16 > B.AI_NOALLOC_SCRATCH_BYTES, records
    frame = _dev(torch, W.make_frame(W.CONFIGS["cfg2"]).image)
    out = tuple(torch.full((cfg.npt,), -7.0, dtype=torch.float32, device="cuda") for _ in range(3))
    with pytest.raises(B.AzintError) as e:
        integ.integrate1d_noalloc(frame, out=out)
    assert e.value.code == B.AI_EUNSUPPORTED
    text = str(e.value)
    assert str(records * 16) in text and str(B.AI_NOALLOC_SCRATCH_BYTES) in text, text
    torch.cuda.synchronize()
    assert all(bool((o == -7.0).all()) for o in out), "a refused call wrote its outputs"
    # the ordinary entry point still serves this matrix
    ref = integ.integrate1d(frame)
    torch.cuda.synchronize()
    assert float(ref[2].sum()) > 0


def test_refusals_that_need_no_launch(torch, B, workloads):
    W = workloads
    cfg = W.tiny_config(64, 64, center_x=30.0, center_y=31.0, unit=W.R_MM, npt=20, name="na_small")
    img = torch.ones((64, 64), dtype=torch.float32, device="cuda")
    cake = B.Integrator(W.scaled(cfg, npt_azim=12))
    with pytest.raises(B.AzintError) as e:
        cake.integrate1d_noalloc(img)
    assert e.value.code == B.AI_EUNSUPPORTED
    integ = B.Integrator(cfg)
    dark = torch.zeros((64, 64), dtype=torch.float32, device="cuda")
    integ.hold_corrections(dark=dark)
    with pytest.raises(B.AzintError) as e:
        integ.integrate1d_noalloc(img)
    assert e.value.code == B.AI_EUNSUPPORTED
    got = _host(integ.integrate1d_noalloc(img, dark=dark))     # arrays of its own: served
    torch.cuda.synchronize()
    assert np.allclose(got["intensity"][got["count"] > 0], 1.0, rtol=1e-6)
