"""Pins of the oracle's full pixel splitting (oracle/azint_oracle.c) against things that are not the
oracle: an independent polygon clipper (Sutherland-Hodgman against the two edges of a bin, shoelace area), hand-worked
quadrilaterals, unit row sums, and containment in the bounding-box matrix.  All `-m "not gpu"`.
"""
import math

import numpy as np
import pytest


def _clip_area(pts, lo, hi):
    """area of the polygon `pts` [(f, chi), ...] between f = lo and f = hi: Sutherland-Hodgman, then the shoelace formula"""
    def clip(poly, bound, keep_above):
        out = []
        for k in range(len(poly)):
            a, b = poly[k], poly[(k + 1) % len(poly)]
            ina = a[0] >= bound if keep_above else a[0] <= bound
            inb = b[0] >= bound if keep_above else b[0] <= bound
            if ina:
                out.append(a)
            if ina != inb:
                t = (bound - a[0]) / (b[0] - a[0])
                out.append((bound, a[1] + t * (b[1] - a[1])))
        return out
    poly = clip(clip(list(pts), lo, True), hi, False)
    if len(poly) < 3:
        return 0.0
    s = 0.0
    for k in range(len(poly)):
        a, b = poly[k], poly[(k + 1) % len(poly)]
        s += a[0] * b[1] - b[0] * a[1]
    return abs(s) / 2.0


def test_hand_worked_quadrilaterals(oracle):
    # an axis-parallel rectangle f in [2.25, 4.75]: the bounding-box answer 0.3, 0.4, 0.3 (u0 = 0, u1 = npt: bin units)
    b, c = oracle.split_full([2.25, 4.75, 4.75, 2.25], [0.0, 0.0, 1.0, 1.0], 0.0, 10.0, 10)
    assert b == [2, 3, 4] and c == pytest.approx([0.3, 0.4, 0.3], abs=1e-15)
    # the triangle (0,0) (2,0) (2,2) (a corner repeated): area 2; under chi = f, bin 0 holds 1/2, bin 1 holds 3/2
    b, c = oracle.split_full([0.0, 2.0, 2.0, 0.0], [0.0, 0.0, 2.0, 0.0], 0.0, 10.0, 10)
    assert b == [0, 1] and c == pytest.approx([0.25, 0.75], abs=1e-15)
    # a diamond centred on a bin edge: (3,0) (4,1) (5,0) (4,-1): half in bin 3, half in bin 4
    b, c = oracle.split_full([3.0, 4.0, 5.0, 4.0], [0.0, 1.0, 0.0, -1.0], 0.0, 10.0, 10)
    assert b == [3, 4] and c == pytest.approx([0.5, 0.5], abs=1e-15)
    # entirely inside one bin -> no splitting
    assert oracle.split_full([3.1, 3.6, 3.7, 3.2], [0.0, 0.1, 1.0, 0.9], 0.0, 10.0, 10) == ([3], [1.0])
    # partly below the range: only the part inside counts, weights relative to the whole quadrilateral
    b, c = oracle.split_full([-1.0, 1.0, 1.0, -1.0], [0.0, 0.0, 1.0, 1.0], 0.0, 10.0, 10)
    assert b == [0] and c == pytest.approx([0.5], abs=1e-15)


def test_random_quadrilaterals_against_polygon_clipping(oracle):
    rng = np.random.default_rng(77)
    for _ in range(300):
        # a convex quadrilateral: a jittered parallelogram, in bin units
        o = rng.uniform(1.0, 6.0), rng.uniform(-1.0, 1.0)
        e1 = rng.uniform(0.2, 2.5), rng.uniform(-0.3, 0.3)
        e2 = rng.uniform(-0.8, 0.8), rng.uniform(0.3, 1.5)
        pts = [(o[0], o[1]), (o[0] + e1[0], o[1] + e1[1]), (o[0] + e1[0] + e2[0], o[1] + e1[1] + e2[1]),
               (o[0] + e2[0], o[1] + e2[1])]
        pts = [(p[0] + rng.uniform(-0.05, 0.05), p[1] + rng.uniform(-0.05, 0.05)) for p in pts]
        total = _clip_area(pts, -100.0, 100.0)
        bins, coefs = oracle.split_full([p[0] for p in pts], [p[1] for p in pts], 0.0, 12.0, 12)
        want = {b: _clip_area(pts, float(b), float(b + 1)) / total for b in range(12)}
        want = {b: v for b, v in want.items() if v > 0}
        assert bins == sorted(want)
        assert coefs == pytest.approx([want[b] for b in bins], rel=1e-11, abs=1e-13)
        assert sum(coefs) == pytest.approx(1.0, abs=1e-12)


@pytest.mark.parametrize("case", ["centred", "offcentre_q", "offimage_tth"])
def test_detector_pixels_against_polygon_clipping_and_row_sums(oracle, workloads, case):
    W = workloads
    cfg = {"centred": W.tiny_config(16, 16, center_x=8.0, center_y=8.0, unit=W.R_MM, npt=23),
           "offcentre_q": W.tiny_config(14, 18, center_x=5.3, center_y=9.6, unit=W.Q_NM, npt=31),
           "offimage_tth": W.tiny_config(12, 20, center_x=-6.5, center_y=30.0, unit=W.TTH_DEG, npt=40)}[case]
    u4, c4, q = oracle.pixel_corners(cfg)
    indptr, indices, data, (u0, u1) = oracle.csr_full(cfg)
    delta = (u1 - u0) / cfg.npt
    dense = np.zeros((cfg.npt, cfg.npix))
    for b in range(cfg.npt):
        dense[b, indices[indptr[b]:indptr[b + 1]]] = data[indptr[b]:indptr[b + 1]]
        assert np.all(np.diff(indices[indptr[b]:indptr[b + 1]]) > 0)
    # every pixel's weights sum to 1 (PAPER.md:116 conservation of pixels)
    assert dense.sum(axis=0) == pytest.approx(np.ones(cfg.npix), abs=1e-12)
    # each weight is the clipped area of the quadrilateral over its total area
    for p in range(cfg.npix):
        if not q[p]:
            continue
        pts = [((u4[p, k] - u0) / delta, c4[p, k]) for k in range(4)]
        total = _clip_area(pts, -1e9, 1e9)
        if total < 1e-14:
            continue
        for b in np.nonzero(dense[:, p])[0]:
            assert dense[b, p] == pytest.approx(_clip_area(pts, float(b), float(b + 1)) / total, rel=1e-9, abs=1e-12)
    # the quadrilateral lies inside its bounding box: the matrix is a subset of the bounding-box one, never larger
    umin, umax = oracle.pixel_bounds(cfg)
    bi, bx, bd = oracle.csr(umin, umax, cfg.npt, u0, u1)
    bbox = np.zeros((cfg.npt, cfg.npix), dtype=bool)
    for b in range(cfg.npt):
        bbox[b, bx[bi[b]:bi[b + 1]]] = True
    assert not np.any((dense > 0) & ~bbox)
    assert indptr[-1] <= bi[-1]


def test_corner_geometry(oracle, workloads):
    W = workloads
    cfg = W.tiny_config(2, 2, center_x=1.0, center_y=1.0, unit=W.R_MM, npt=2, pixel_m=1e-3)
    u4, c4, q = oracle.pixel_corners(cfg)
    assert np.all(q == 1)
    # pixel (1,1): corners (0,0) (1,0) (1,1) (0,1) mm -> r = 0, 1, sqrt 2, 1; chi = (centre direction pi/4), 0, pi/4, pi/2
    assert u4[3] == pytest.approx([0.0, 1.0, math.sqrt(2.0), 1.0], abs=1e-15)
    assert c4[3] == pytest.approx([math.pi / 4, 0.0, math.pi / 4, math.pi / 2], abs=1e-15)
    # a pixel that holds the beam centre has no quadrilateral and falls back to its bounding box
    cfg = W.tiny_config(3, 3, center_x=1.5, center_y=1.5, unit=W.R_MM, npt=4)
    u4, c4, q = oracle.pixel_corners(cfg)
    assert q.tolist() == [1, 1, 1, 1, 0, 1, 1, 1, 1]
    # the pixel left of the centre crosses the seam: its corner angles stay within half a turn of one another
    assert np.ptp(c4[3]) < math.pi


# ---- aio_integrate1d_full: the per-pixel forward scatter of PAPER.md:126-130 ------------------------------------------------
def _full_cases(W):
    return {"centred": W.tiny_config(16, 16, center_x=8.0, center_y=8.0, unit=W.R_MM, npt=23),
            "offcentre_q": W.tiny_config(14, 18, center_x=5.3, center_y=9.6, unit=W.Q_NM, npt=31),
            "offimage_tth": W.tiny_config(12, 20, center_x=-6.5, center_y=30.0, unit=W.TTH_DEG, npt=40)}


def _corrected_frame(W, cfg, seed):
    rng = np.random.default_rng(seed)
    shape = (cfg.height, cfg.width)
    return W.Frame(image=rng.poisson(300.0, size=shape).astype(np.float64),
                   dark=rng.poisson(5.0, size=shape).astype(np.float64),
                   flat=rng.uniform(0.9, 1.1, size=shape), solidangle=rng.uniform(0.7, 1.0, size=shape),
                   polarization=rng.uniform(0.95, 1.0, size=shape), mask=(rng.random(shape) < 0.1).astype(np.uint8))


def _value_and_validity(fr):
    """O5 written out once more, for the pins only: v = (I - dark) / (flat solid pol), valid = unmasked."""
    v = (fr.image - fr.dark) / (fr.flat * fr.solidangle * fr.polarization)
    ok = fr.mask == 0
    return np.where(ok, v, 0.0).ravel(), ok.ravel()


@pytest.mark.parametrize("case", ["centred", "offcentre_q", "offimage_tth"])
def test_full_profile_uniform_image_and_conservation(oracle, workloads, case):
    """the splitting conserves the signal and the pixels.  Over the automatic range every pixel lies inside
    the range, so sum_b sum_signal = sum_p v_p and sum_b count = number of valid pixels; a uniform image gives a constant
    profile wherever a bin holds any pixel."""
    W = workloads
    cfg = _full_cases(W)[case]
    fr = _corrected_frame(W, cfg, 3)
    v, ok = _value_and_validity(fr)
    out = oracle.integrate1d_full(cfg, fr)
    assert out["sum_signal"].sum() == pytest.approx(v.sum(), rel=1e-12)
    assert out["count"].sum() == pytest.approx(ok.sum(), rel=1e-12)
    uni = oracle.integrate1d_full(cfg, W.Frame(image=np.full((cfg.height, cfg.width), 7.25)))
    filled = uni["count"] > 0
    assert filled.sum() >= cfg.npt // 2
    assert uni["intensity"][filled] == pytest.approx(7.25, rel=1e-13)
    assert np.all(uni["intensity"][~filled] == 0.0)
    assert uni["count"].sum() == pytest.approx(cfg.npix, rel=1e-12)
    u0, u1 = out["range"]
    assert out["radial"] == pytest.approx(u0 + (np.arange(cfg.npt) + 0.5) * (u1 - u0) / cfg.npt, rel=1e-15)


@pytest.mark.parametrize("case", ["centred", "offcentre_q", "offimage_tth"])
def test_full_profile_equals_pinned_matrix_times_frame(oracle, workloads, case):
    """The scatter and the (clipper-pinned) matrix of aio_csr_full are two routes to the same sums: S = M v, C = M valid.
    A dropped validity test, a swapped mask polarity or a missing dark current in the scatter shows here."""
    W = workloads
    cfg = _full_cases(W)[case]
    fr = _corrected_frame(W, cfg, 9)
    v, ok = _value_and_validity(fr)
    indptr, indices, data, _ = oracle.csr_full(cfg)
    out = oracle.integrate1d_full(cfg, fr, empty=-3.0)
    for b in range(cfg.npt):
        cols, c = indices[indptr[b]:indptr[b + 1]], data[indptr[b]:indptr[b + 1]]
        S, Cn = float(np.dot(c, v[cols])), float(np.dot(c, ok[cols].astype(np.float64)))
        assert out["sum_signal"][b] == pytest.approx(S, rel=1e-12, abs=1e-12)
        assert out["count"][b] == pytest.approx(Cn, rel=1e-12, abs=1e-12)
        assert out["intensity"][b] == (pytest.approx(S / Cn, rel=1e-12) if Cn > 0 else -3.0)
    # every pixel masked: both histograms empty, intensity = the empty value
    dead = W.Frame(image=fr.image, mask=np.ones_like(fr.mask))
    out = oracle.integrate1d_full(cfg, dead, empty=-3.0)
    assert np.all(out["count"] == 0.0) and np.all(out["sum_signal"] == 0.0) and np.all(out["intensity"] == -3.0)


def test_full_profile_one_bin_is_the_mean_and_no_quadrilateral_is_the_bounding_box(oracle, workloads):
    W = workloads
    cfg = W.tiny_config(14, 18, center_x=5.3, center_y=9.6, unit=W.TTH_DEG, npt=1)
    fr = _corrected_frame(W, cfg, 21)
    v, ok = _value_and_validity(fr)
    out = oracle.integrate1d_full(cfg, fr)
    assert out["count"][0] == pytest.approx(ok.sum(), rel=1e-13)
    assert out["intensity"][0] == pytest.approx(v.sum() / ok.sum(), rel=1e-12)
    # with no pixel given a quadrilateral the routine is bounding-box splitting: equal to the pinned 1D oracle
    cfg = _full_cases(W)["offcentre_q"]
    fr = _corrected_frame(W, cfg, 22)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    u4, c4, q = oracle.pixel_corners(cfg)
    args = (fr.image, fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask)
    got = oracle.integrate1d_full_corners(u4, c4, np.zeros_like(q), umin, umax, cfg.npt, u0, u1, *args)
    want = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, *args)
    for k in ("sum_signal", "count", "intensity"):
        assert np.array_equal(got[k], want[k]), k
    # ... and with the quadrilaterals it is not (the pin above would be empty otherwise)
    full = oracle.integrate1d_full_corners(u4, c4, q, umin, umax, cfg.npt, u0, u1, *args)
    assert np.abs(full["count"] - want["count"]).max() > 1e-3
