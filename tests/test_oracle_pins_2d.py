"""Pins of the oracle's bidimensional ("cake") routines (oracle/azint_oracle.c, last section) against things that are
not the oracle: the already pinned 1D oracle (summing the 2D result over the azimuthal bins must give the 1D result bin
by bin), what the paper fixes (conservation of signal and of pixels), a hand-worked image, symmetry,
and an mpmath brute force of the azimuthal extents.  All `-m "not gpu"`.
"""
import math

import numpy as np
import pytest


@pytest.fixture(scope="module")
def W(workloads):
    return workloads


def _cfg(W, h, w, cx, cy, npt, npt_azim, unit=None, **kw):
    c = W.tiny_config(h, w, center_x=cx, center_y=cy, unit=W.R_MM if unit is None else unit, npt=npt, **kw)
    return W.scaled(c, npt_azim=npt_azim)


# ----------------------------------------------------------------------------------------------------------------
# azimuthal extent of a pixel: chi = atan2(y, x) over the pixel rectangle
# ----------------------------------------------------------------------------------------------------------------
def _brute_extent(cfg, i, j):
    """(lo, width) of the set of directions of pixel (i, j) by mpmath: the boundary of the rectangle is sampled densely
    and the largest gap between consecutive directions (on the circle) is what the pixel does NOT cover."""
    import mpmath as mp
    mp.mp.dps = 30
    x0, x1 = (j - cfg.center_x_px), (j + 1 - cfg.center_x_px)
    y0, y1 = (i - cfg.center_y_px), (i + 1 - cfg.center_y_px)
    if x0 < 0 < x1 and y0 < 0 < y1:
        return -math.pi, 2 * math.pi
    pts = []
    n = 64
    for k in range(n + 1):
        t = mp.mpf(k) / n
        for (x, y) in ((x0 + t * (x1 - x0), y0), (x0 + t * (x1 - x0), y1), (x0, y0 + t * (y1 - y0)), (x1, y0 + t * (y1 - y0))):
            if x == 0 and y == 0:
                continue
            pts.append(mp.atan2(y, x))
    pts = sorted(set(pts))
    gaps = [(pts[(k + 1) % len(pts)] - pts[k]) % (2 * mp.pi) for k in range(len(pts))]
    k = max(range(len(pts)), key=lambda q: gaps[q])
    lo = pts[(k + 1) % len(pts)]
    return float(lo), float(2 * mp.pi - gaps[k])


@pytest.mark.parametrize("cx,cy", [(4.0, 4.0), (3.5, 4.5), (3.3, 2.7), (-2.0, 3.0), (12.0, 4.0), (4.0, 3.25), (2.5, -1.0)])
def test_azimuthal_extents_against_mpmath(oracle, W, cx, cy):
    # centre on a pixel corner, inside a pixel, on an edge, off the image on either side (seam crossing), ...
    cfg = _cfg(W, 8, 8, cx, cy, 4, 8)
    lo, w = oracle.pixel_chi_bounds(cfg)
    for i in range(8):
        for j in range(8):
            blo, bw = _brute_extent(cfg, i, j)
            p = i * 8 + j
            assert w[p] == pytest.approx(bw, abs=1e-12), (i, j)
            d = (lo[p] - blo + math.pi) % (2 * math.pi) - math.pi
            assert abs(d) < 1e-12, (i, j, lo[p], blo)
            assert -math.pi <= lo[p] < math.pi + 1e-15


def test_azimuthal_extent_special_cases(oracle, W):
    cfg = _cfg(W, 2, 2, 1.0, 1.0, 1, 4)                       # centre on the corner shared by the four pixels
    lo, w = oracle.pixel_chi_bounds(cfg)
    assert w == pytest.approx([math.pi / 2] * 4, abs=1e-15)
    assert lo == pytest.approx([-math.pi, -math.pi / 2, math.pi / 2, 0.0], abs=1e-15)     # (0,0) (0,1) (1,0) (1,1)
    cfg = _cfg(W, 1, 2, 1.0, 0.5, 1, 4)                       # centre on the edge between two pixels
    lo, w = oracle.pixel_chi_bounds(cfg)
    assert w == pytest.approx([math.pi, math.pi], abs=1e-15)
    assert lo[1] == pytest.approx(-math.pi / 2, abs=1e-15)   # right pixel: x >= 0
    assert lo[0] == pytest.approx(math.pi / 2, abs=1e-15)    # left pixel: [pi/2, 3pi/2], across the seam
    cfg = _cfg(W, 1, 1, 0.5, 0.5, 1, 4)                       # centre strictly inside
    lo, w = oracle.pixel_chi_bounds(cfg)
    assert lo[0] == -math.pi and w[0] == 2 * math.pi


def test_periodic_split_hand_cases(oracle):
    pi = math.pi
    # four bins on the full circle: [-pi,-pi/2) [-pi/2,0) [0,pi/2) [pi/2,pi]
    assert oracle.split_azim(0.1, 0.2, -pi, pi, 4) == ([2], [1.0])
    b, c = oracle.split_azim(-0.1, 0.4, -pi, pi, 4)           # straddles 0: 1/4 below, 3/4 above
    assert b == [1, 2] and c == pytest.approx([0.25, 0.75], abs=1e-15)
    b, c = oracle.split_azim(pi - 0.3, 0.4, -pi, pi, 4)       # across the seam: 3/4 in the last bin, 1/4 in the first
    assert b == [0, 3] and c == pytest.approx([0.25, 0.75], abs=1e-12)
    b, c = oracle.split_azim(-pi, 2 * pi, -pi, pi, 4)         # the whole circle: a quarter each
    assert b == [0, 1, 2, 3] and c == pytest.approx([0.25] * 4, abs=1e-15)
    # a restricted range keeps only what falls inside it (weights relative to the whole pixel)
    b, c = oracle.split_azim(-0.1, 0.4, 0.0, pi / 2, 2)
    assert b == [0] and c == pytest.approx([0.75], abs=1e-15)
    # a range that starts elsewhere on the circle: [pi/2, 5pi/2] -- the same pixel, seen one turn later
    b, c = oracle.split_azim(-0.1, 0.4, pi / 2, 5 * pi / 2, 4)
    assert b == [2, 3] and c == pytest.approx([0.25, 0.75], abs=1e-12)


# ----------------------------------------------------------------------------------------------------------------
# the 2D result
# ----------------------------------------------------------------------------------------------------------------
def test_worked_2x2_image(oracle, W):
    # 2 x 2 image, centre on the shared corner, 4 azimuthal x 1 radial bin: each pixel is exactly one quadrant.
    # chi bins: [-pi,-pi/2) -> pixel (0,0) = 1;  [-pi/2,0) -> pixel (0,1) = 2;  [0,pi/2) -> pixel (1,1) = 4;
    # [pi/2,pi] -> pixel (1,0) = 3
    cfg = _cfg(W, 2, 2, 1.0, 1.0, 1, 4)
    r = oracle.integrate2d(cfg, W.Frame(image=np.array([[1.0, 2.0], [3.0, 4.0]])))
    assert r["count"].ravel() == pytest.approx([1, 1, 1, 1], abs=1e-15)
    assert r["sum_signal"].ravel() == pytest.approx([1, 2, 4, 3], abs=1e-15)
    assert r["intensity"].ravel() == pytest.approx([1, 2, 4, 3], abs=1e-15)
    assert r["azimuthal"] == pytest.approx([-0.75 * math.pi, -0.25 * math.pi, 0.25 * math.pi, 0.75 * math.pi])


@pytest.mark.parametrize("case", ["centred", "offcentre", "offimage", "q_units"])
def test_sum_over_azimuth_equals_the_1d_result(oracle, W, case):
    # the 1D oracle is pinned on its own (tests/test_oracle_pins.py); the azimuthal weights of a pixel sum to 1 on the
    # full circle, so collapsing the azimuthal axis must reproduce it bin by bin
    cfg = {"centred": _cfg(W, 48, 48, 24.0, 24.0, 37, 24),
           "offcentre": _cfg(W, 40, 56, 17.3, 29.6, 41, 36),
           "offimage": _cfg(W, 32, 48, -9.5, 60.0, 29, 90),
           "q_units": _cfg(W, 33, 47, 20.25, 11.5, 53, 17, unit=W.Q_NM)}[case]
    rng = np.random.default_rng(5)
    fr = W.Frame(image=rng.poisson(100.0, size=(cfg.height, cfg.width)).astype(np.float64),
                 dark=rng.poisson(5.0, size=(cfg.height, cfg.width)).astype(np.float64),
                 flat=rng.uniform(0.9, 1.1, size=(cfg.height, cfg.width)),
                 mask=(rng.random((cfg.height, cfg.width)) < 0.05).astype(np.uint8))
    r2 = oracle.integrate2d(cfg, fr)
    r1 = oracle.integrate1d(cfg, fr)
    assert r2["sum_signal"].sum(axis=0) == pytest.approx(r1["sum_signal"], rel=1e-12, abs=1e-9)
    assert r2["count"].sum(axis=0) == pytest.approx(r1["count"], rel=1e-12, abs=1e-12)
    assert r2["radial"] == pytest.approx(r1["radial"], rel=1e-15)


def test_conservation_and_unit_weights(oracle, W):
    # sum(image) = sum(weighted histogram), sum(unweighted histogram) = number of pixels; equivalently
    # every pixel's weights sum to 1 (checked per pixel on the CSR)
    cfg = _cfg(W, 40, 40, 13.7, 22.2, 31, 45)
    rng = np.random.default_rng(6)
    img = rng.poisson(50.0, size=(40, 40)).astype(np.float64)
    r = oracle.integrate2d(cfg, W.Frame(image=img))
    assert r["sum_signal"].sum() == pytest.approx(img.sum(), rel=1e-13)
    assert r["count"].sum() == pytest.approx(cfg.npix, rel=1e-13)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    lo, w = oracle.pixel_chi_bounds(cfg)
    indptr, indices, data = oracle.csr2d(umin, umax, lo, w, cfg.npt, u0, u1, cfg.npt_azim, -math.pi, math.pi)
    assert np.bincount(indices, weights=data, minlength=cfg.npix) == pytest.approx(np.ones(cfg.npix), abs=1e-13)
    # the CSR applied to the image is the weighted histogram; columns ascend within a row
    import scipy.sparse as sp
    m = sp.csr_matrix((data, indices, indptr), shape=(cfg.npt * cfg.npt_azim, cfg.npix))
    assert m @ img.ravel() == pytest.approx(r["sum_signal"].ravel(), rel=1e-12, abs=1e-12)
    for b in range(0, cfg.npt * cfg.npt_azim, 97):
        assert np.all(np.diff(indices[indptr[b]:indptr[b + 1]]) > 0)


def test_fourfold_symmetry(oracle, W):
    # centred square detector: rotating the frame by 90 degrees shifts the azimuthal bins by npt_azim / 4
    cfg = _cfg(W, 32, 32, 16.0, 16.0, 19, 16)
    rng = np.random.default_rng(8)
    img = rng.poisson(80.0, size=(32, 32)).astype(np.float64)
    r = oracle.integrate2d(cfg, W.Frame(image=img))
    # a quarter turn of the frame in the (x, y) plane; its sense only decides the sign of the shift
    rr = oracle.integrate2d(cfg, W.Frame(image=np.ascontiguousarray(np.rot90(img, k=-1))))
    assert any(np.allclose(r["sum_signal"], np.roll(rr["sum_signal"], s, axis=0), rtol=1e-12, atol=1e-9) for s in (4, -4))
    assert not np.allclose(r["sum_signal"], rr["sum_signal"], rtol=1e-6)
    # the geometry alone is 4-fold symmetric: the unweighted histogram is invariant under a shift by a quarter turn
    assert np.allclose(r["count"], np.roll(r["count"], 4, axis=0), rtol=1e-12, atol=1e-12)


def test_uniform_image_and_restricted_ranges(oracle, W):
    cfg = _cfg(W, 30, 44, 10.0, 33.0, 23, 40)
    fr = W.Frame(image=np.full((30, 44), 7.5))
    r = oracle.integrate2d(cfg, fr)
    ok = r["count"] > 0
    assert r["intensity"][ok] == pytest.approx(np.full(ok.sum(), 7.5), rel=1e-13)
    assert np.all(r["intensity"][~ok] == 0.0)
    # a sector: only the pixels' parts inside it count; the sector's bins equal the matching bins of a full-circle run
    # with aligned edges (40 bins on the circle, 10 bins on a quarter)
    q = oracle.integrate2d(W.scaled(cfg, npt_azim=10), fr, azim_range=(0.0, math.pi / 2))
    assert q["count"] == pytest.approx(r["count"][20:30], rel=1e-12, abs=1e-13)
