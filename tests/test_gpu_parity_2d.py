"""Parity of bidimensional ("cake") integration on the CUDA path (ai_setup2d / ai_integrate2d through the C ABI) against
the CPU oracle (oracle/azint_oracle.c, pinned in tests/test_oracle_pins_2d.py): the matrix (rows = azimuthal x radial
bins, column sets identical except bin-edge ties, coefficients within 1e-6 relative + 1e-7) and the per-bin results
(relative error <= 1e-6 with compensated accumulation).  PAPER.md:29, :114-116 (Fig. 3), :39, :120.
"""
import math

import numpy as np
import pytest

from parity import assert_profile, compare_csr

pytestmark = pytest.mark.gpu

LAYOUTS = {"tiled": 0, "csr": 1, "direct": 3}
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


def _cases(W):
    def c(name, h, w, cx, cy, npt, na, unit=W.R_MM):
        return W.scaled(W.tiny_config(h, w, center_x=cx, center_y=cy, unit=unit, npt=npt, name=name), npt_azim=na)
    return {
        "centred": c("centred", 96, 96, 48.0, 48.0, 40, 36),                 # centre on a pixel corner
        "inside_a_pixel": c("inside_a_pixel", 80, 112, 40.4, 61.7, 33, 48),  # one pixel covers the full circle
        "on_an_edge": c("on_an_edge", 64, 64, 20.0, 30.5, 25, 30),
        "seam_only": c("seam_only", 70, 130, 150.5, 33.3, 50, 90, W.Q_NM),   # beam right of the image: all chi near +-pi
        "off_image": c("off_image", 67, 259, -12.5, 300.0, 41, 180, W.TTH_DEG),
        "many_bins": c("many_bins", 48, 48, 24.0, 24.0, 64, 360),            # more bins than pixels near the centre
        "one_azim_bin": c("one_azim_bin", 60, 72, 30.3, 29.6, 45, 1),        # pixels across the seam: both images in bin 0
    }


def _oracle2d(oracle, cfg, azim_range=None):
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    lo, w = oracle.pixel_chi_bounds(cfg)
    c0, c1 = (-math.pi, math.pi) if azim_range is None else azim_range
    return umin, umax, lo, w, u0, u1, c0, c1


def _dev(torch, a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _run2d(torch, integ, fr):
    args = [_dev(torch, x) for x in (fr.image, fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)]
    rad = torch.empty(integ.npt_rad, dtype=torch.float32, device="cuda")
    azi = torch.empty(integ.npt_azim, dtype=torch.float32, device="cuda")
    i, s, c = integ.integrate2d(*args, radial=rad, azimuthal=azi)
    torch.cuda.synchronize()
    return {"intensity": i.cpu().numpy().ravel(), "sum_signal": s.cpu().numpy().ravel(), "count": c.cpu().numpy().ravel(),
            "radial": rad.cpu().numpy(), "azimuthal": azi.cpu().numpy()}


def _flat(want):
    return {k: np.asarray(want[k]).ravel() for k in ("intensity", "sum_signal", "count")}


@pytest.mark.parametrize("name", ["centred", "inside_a_pixel", "on_an_edge", "seam_only", "off_image", "many_bins",
                                  "one_azim_bin"])
def test_csr2d_matches_oracle(torch, B, oracle, workloads, parity_report, name):
    cfg = _cases(workloads)[name]
    integ = B.Integrator(cfg)
    gi, gx, gd, (u0, u1) = integ.csr()
    umin, umax, lo, w, o0, o1, c0, c1 = _oracle2d(oracle, cfg)
    assert u0 == pytest.approx(o0, rel=1e-15, abs=1e-300) and u1 == pytest.approx(o1, rel=4e-16)
    ora = oracle.csr2d(umin, umax, lo, w, cfg.npt, o0, o1, cfg.npt_azim, c0, c1)
    # pixel edges that lie ON the x or y axis through the beam centre have chi exactly on a bin edge whenever 0, pi/2, pi
    # are bin edges: the zero-width overlap is an entry on one side and none on the other (atan2 differs by an ulp
    # between glibc and CUDA).  Such ties are counted, and bounded by the number of pixels along the two axes.
    rep = compare_csr((gi, gx, gd), ora, cfg.npix, max_ties=4 * (cfg.height + cfg.width))
    print(name, rep)
    parity_report.setdefault("csr2d_vs_oracle", {})[name] = dict(rep, npt_rad=cfg.npt, npt_azim=cfg.npt_azim,
                                                                 shape=[cfg.height, cfg.width])
    integ.close()


@pytest.mark.parametrize("layout", ["tiled", "direct", "csr"])
@pytest.mark.parametrize("name", ["centred", "inside_a_pixel", "on_an_edge", "seam_only", "off_image", "many_bins",
                                  "one_azim_bin"])
def test_profile2d_parity_small(torch, B, oracle, workloads, name, layout):
    cfg = _cases(workloads)[name]
    rng = np.random.default_rng(11)
    shape = (cfg.height, cfg.width)
    fr = workloads.Frame(image=rng.poisson(200.0, size=shape).astype(np.float32),
                         dark=rng.poisson(5.0, size=shape).astype(np.float32),
                         flat=rng.uniform(0.9, 1.1, size=shape).astype(np.float32),
                         mask=(rng.random(shape) < 0.05).astype(np.uint8))
    plain = workloads.Frame(image=fr.image)
    for accum in ("kahan", "f64"):
        integ = B.Integrator(cfg, layout=LAYOUTS[layout], accum=ACCUMS[accum], empty_value=-1.0)
        for f in (plain, fr):
            got = _run2d(torch, integ, f)
            want = oracle.integrate2d(cfg, f, empty=-1.0)
            assert_profile(got, _flat(want), what=f"{name}/{layout}/{accum}")
            assert np.allclose(got["radial"], want["radial"], rtol=2e-7)
            assert np.allclose(got["azimuthal"], want["azimuthal"], rtol=2e-7, atol=1e-7)
            # bins nothing falls into carry the empty value
            empty = _flat(want)["count"] <= 0
            assert np.all(got["intensity"][empty] == -1.0)
        integ.close()


def test_restricted_azimuthal_range(torch, B, oracle, workloads):
    cfg = _cases(workloads)["inside_a_pixel"]
    rng = np.random.default_rng(12)
    fr = workloads.Frame(image=rng.poisson(100.0, size=(cfg.height, cfg.width)).astype(np.float32))
    for arange in ((0.0, math.pi / 2), (math.pi / 2, 2.5 * math.pi), (-3.0, 1.0)):
        integ = B.Integrator(cfg, azim_range=arange)
        got = _run2d(torch, integ, fr)
        want = oracle.integrate2d(cfg, fr, azim_range=arange)
        assert_profile(got, _flat(want), what=f"azim range {arange}")
        integ.close()


def test_cake_full_size(torch, B, oracle, workloads, parity_report):
    """2048 x 2048 gold-ring frame into 360 azimuthal x 500 radial bins: the matrix and the result."""
    cfg = workloads.CONFIGS["cake2"]
    fr = workloads.make_frame(cfg)
    integ = B.Integrator(cfg)
    gi, gx, gd, (u0, u1) = integ.csr()
    umin, umax, lo, w, o0, o1, c0, c1 = _oracle2d(oracle, cfg)
    ora = oracle.csr2d(umin, umax, lo, w, cfg.npt, o0, o1, cfg.npt_azim, c0, c1)
    rep = compare_csr((gi, gx, gd), ora, cfg.npix, max_ties=4 * (cfg.height + cfg.width))
    print("cake2 matrix", rep, B.ai_get_layout_info(integ.ctx))
    del ora, gi, gx, gd
    want = oracle.integrate2d_bounds(umin, umax, lo, w, cfg.npt, o0, o1, cfg.npt_azim, c0, c1, fr.image)
    worst = {}
    for layout in ("tiled", "direct"):
        for accum in ("kahan", "plain"):
            integ.set_options(LAYOUTS[layout], ACCUMS[accum])
            got = _run2d(torch, integ, fr)
            worst[f"{layout}/{accum}"] = assert_profile(got, _flat(want), tol=1e-3 if accum == "plain" else 1e-6,
                                                        what=f"cake2/{layout}/{accum}")
    print("cake2", worst)
    # collapsing the azimuthal axis gives the 1D profile of the same frame (500 bins)
    integ.set_options()
    got = _run2d(torch, integ, fr)
    want1 = oracle.integrate1d(cfg, fr)
    s1 = got["sum_signal"].reshape(cfg.npt_azim, cfg.npt).astype(np.float64).sum(axis=0)
    assert np.allclose(s1, want1["sum_signal"], rtol=2e-6)
    parity_report["cake2_2048x2048_360x500"] = {"matrix": rep, "max_per_bin_relative_error": worst,
                                                "layout": B.ai_get_layout_info(integ.ctx)}
    integ.close()


def test_2d_and_1d_entry_points_do_not_mix(torch, B, workloads):
    cfg = _cases(workloads)["centred"]
    integ = B.Integrator(cfg)
    img = torch.zeros((cfg.height, cfg.width), dtype=torch.float32, device="cuda")
    out = [torch.empty(integ.npt, dtype=torch.float32, device="cuda") for _ in range(3)]
    with pytest.raises(B.AzintError):
        B.ai_integrate1d(integ.ctx, img, None, None, None, None, None, None, *out)
    integ.close()
    one = B.Integrator(workloads.CONFIGS["cfg1"])
    img = torch.zeros((256, 256), dtype=torch.float32, device="cuda")
    with pytest.raises(B.AzintError):
        B.ai_integrate2d(one.ctx, img, None, None, None, None, None, None, None, *out)
    one.close()
