"""Pins for the CPU oracle (oracle/azint_oracle.c): everything here checks it against something other than itself --
values worked by hand from the paper's procedure, closed forms, invariants the paper states, an independent mpmath
brute force, numpy / scipy routines on special cases, and the statistics derived independently in SURVEY.md §8(a).
CPU only (`-m "not gpu"`).
"""
import json
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def gold(name):
    with open(os.path.join(GOLD, name)) as f:
        return json.load(f)


# ----------------------------------------------------------------------------------------------------------------
# O4: the split itself
# ----------------------------------------------------------------------------------------------------------------
def test_hand_worked_split(oracle):
    g = gold("worked_examples.json")["split"]
    # bins of unit width on [0, 10]: f == u
    bins, coefs = oracle.split(g["f_min"], g["f_max"], 0.0, 10.0, 10)
    assert bins == g["bins"]
    assert np.allclose(coefs, g["coefs"], rtol=0, atol=1e-15)


def test_split_special_cases(oracle):
    # PAPER.md:122 "When the whole pixel falls into only one bin, there is no pixel splitting"
    assert oracle.split(3.1, 3.9, 0.0, 10.0, 10) == ([3], [1.0])
    # two outermost bins only, no internal bin
    b, c = oracle.split(3.5, 4.25, 0.0, 10.0, 10)
    assert b == [3, 4] and np.allclose(c, [0.5 / 0.75, 0.25 / 0.75], atol=1e-15)
    # four internal bins share the remainder evenly: each gets 1/w
    b, c = oracle.split(1.5, 6.5, 0.0, 10.0, 10)
    assert b == [1, 2, 3, 4, 5, 6] and np.allclose(c, [0.1, 0.2, 0.2, 0.2, 0.2, 0.1], atol=1e-15)
    # upper bound exactly on a bin edge: zero-width overlap emits no entry (reading 5)
    assert oracle.split(2.5, 4.0, 0.0, 10.0, 10)[0] == [2, 3]
    # lower bound exactly on a bin edge
    assert oracle.split(3.0, 3.5, 0.0, 10.0, 10) == ([3], [1.0])
    # last bin is closed: a pixel ending exactly at u1 lands in bin npt-1
    b, c = oracle.split(9.5, 10.0, 0.0, 10.0, 10)
    assert b == [9] and c == [1.0]
    # entirely outside an explicit range
    assert oracle.split(-2.0, -1.0, 0.0, 10.0, 10) == ([], [])
    assert oracle.split(10.0, 11.0, 0.0, 10.0, 10) == ([], [])
    # partly outside: the outside part is lost, coefficients sum to the inside fraction
    b, c = oracle.split(-0.5, 1.5, 0.0, 10.0, 10)
    assert b == [0, 1] and np.allclose(c, [0.5, 0.25], atol=1e-15)
    b, c = oracle.split(9.25, 10.75, 0.0, 10.0, 10)
    assert b == [9] and np.allclose(c, [0.5], atol=1e-15)
    # non-trivial origin and bin width
    b, c = oracle.split(1.0 + 0.25 * 2.25, 1.0 + 0.25 * 4.75, 1.0, 3.5, 10)
    assert b == [2, 3, 4] and np.allclose(c, [0.3, 0.4, 0.3], atol=1e-12)


def test_worked_2x2_image(oracle, workloads):
    g = gold("worked_examples.json")["image_2x2"]
    cfg = workloads.tiny_config(2, 2, center_x=g["center"][0], center_y=g["center"][1], unit=workloads.R_MM,
                                npt=g["npt"], pixel_m=g["pixel"])
    fr = workloads.Frame(image=np.array(g["image"], dtype=np.float64))
    r = oracle.integrate1d(cfg, fr)
    assert np.allclose(r["count"], g["count"], atol=1e-14)
    assert np.allclose(r["sum_signal"], g["sum_signal"], atol=1e-13)
    assert np.allclose(r["intensity"], g["intensity"], atol=1e-13)
    # radial = bin centres of [0, sqrt(2)] m expressed in mm
    assert np.allclose(r["radial"], np.array([0.25, 0.75]) * math.sqrt(2.0) * 1e3, rtol=1e-14)


# ----------------------------------------------------------------------------------------------------------------
# O1-O4 against an independent brute force (mpmath, 50 digits, O(npt * N), written in u space not f space)
# ----------------------------------------------------------------------------------------------------------------
def _brute_force_matrix(cfg, u0, u1, W):
    import mpmath as mp
    mp.mp.dps = 50
    D, lam, pix = mp.mpf(cfg.distance_m), mp.mpf(cfg.wavelength_m), mp.mpf(cfg.pixel_m)
    cx, cy = mp.mpf(cfg.center_x_px), mp.mpf(cfg.center_y_px)

    def u_of(r):
        if cfg.unit == W.R_MM:
            return 1000 * r
        tth = mp.atan(r / D)
        if cfg.unit == W.TTH_RAD:
            return tth
        if cfg.unit == W.TTH_DEG:
            return tth * 180 / mp.pi
        q = 4 * mp.pi * mp.sin(tth / 2) / lam
        return q * (mp.mpf(10) ** -9 if cfg.unit == W.Q_NM else mp.mpf(10) ** -10)

    u0, u1 = mp.mpf(u0), mp.mpf(u1)
    edges = [u0 + (u1 - u0) * b / cfg.npt for b in range(cfg.npt + 1)]
    M = np.zeros((cfg.npt, cfg.npix))
    for i in range(cfg.height):
        for j in range(cfg.width):
            xs = [(j - cx) * pix, (j + 1 - cx) * pix]
            ys = [(i - cy) * pix, (i + 1 - cy) * pix]
            # nearest point of the rectangle to the origin: clamp 0 into each interval
            nx = min(max(mp.mpf(0), xs[0]), xs[1])
            ny = min(max(mp.mpf(0), ys[0]), ys[1])
            rmin = mp.sqrt(nx * nx + ny * ny)
            rmax = max(mp.sqrt(x * x + y * y) for x in xs for y in ys)
            a, z = u_of(rmin), u_of(rmax)
            for b in range(cfg.npt):
                ov = min(z, edges[b + 1]) - max(a, edges[b])
                if ov > 0:
                    M[b, i * cfg.width + j] = float(ov / (z - a))
    return M


TINY = [
    # (H, W, cx, cy, unit, npt, explicit range as fractions of the auto range or None)
    (8, 8, 4.0, 4.0, "R_MM", 7, None),
    (6, 9, 2.3, 3.7, "TTH_DEG", 11, None),            # non-integer centre inside a pixel
    (7, 5, -3.0, 2.0, "Q_NM", 9, None),               # centre off the image
    (5, 7, 3.5, 2.5, "TTH_RAD", 13, None),            # centre at a pixel centre
    (8, 6, 3.0, 9.5, "Q_A", 6, None),
    (8, 8, 4.0, 4.0, "R_MM", 5, (0.21, 0.77)),        # explicit range cutting pixels at both ends
    (16, 16, 7.25, 8.5, "Q_NM", 40, None),            # bins much narrower than a pixel
    (4, 4, 2.0, 2.0, "R_MM", 1, None),
]


@pytest.mark.parametrize("H,Wd,cx,cy,unit,npt,rng", TINY)
def test_coefficients_vs_mpmath_brute_force(oracle, workloads, H, Wd, cx, cy, unit, npt, rng):
    W = workloads
    # a short distance makes atan / sin visibly non-linear over the tiny detector
    cfg = W.tiny_config(H, Wd, center_x=cx, center_y=cy, unit=getattr(W, unit), npt=npt, distance_m=1.2e-3)
    umin, umax = oracle.pixel_bounds(cfg)
    a0, a1 = oracle.auto_range(umin, umax)
    u0, u1 = (a0, a1) if rng is None else (a0 + rng[0] * (a1 - a0), a0 + rng[1] * (a1 - a0))
    indptr, indices, data = oracle.csr(umin, umax, npt, u0, u1)
    import scipy.sparse as sp
    got = sp.csr_matrix((data, indices, indptr), shape=(npt, cfg.npix)).toarray()
    want = _brute_force_matrix(cfg, u0, u1, W)
    # entries whose overlap is below 1e-12 of a bin are bin-edge ties (reading 5): ignore them on both sides
    tie = (np.abs(got - want) < 1e-11) & ((got == 0) != (want == 0))
    assert np.array_equal((got != 0) | tie, (want != 0) | tie)
    assert np.allclose(got, want, rtol=1e-10, atol=1e-12)
    # and indices ascend within each row (scipy "sorted indices")
    for b in range(npt):
        row = indices[indptr[b]:indptr[b + 1]]
        assert np.all(np.diff(row) > 0)


# ----------------------------------------------------------------------------------------------------------------
# O1-O3: ranges in closed form and the statistics SURVEY.md derived independently
# ----------------------------------------------------------------------------------------------------------------
def _closed_form_range(cfg, W):
    xs = np.array([0.0 - cfg.center_x_px, cfg.width - cfg.center_x_px]) * cfg.pixel_m
    ys = np.array([0.0 - cfg.center_y_px, cfg.height - cfg.center_y_px]) * cfg.pixel_m
    rmax = math.sqrt(max(xs ** 2) + max(ys ** 2))
    dx = 0.0 if xs[0] <= 0 <= xs[1] else min(abs(xs))
    dy = 0.0 if ys[0] <= 0 <= ys[1] else min(abs(ys))
    rmin = math.hypot(dx, dy)

    def u(r):
        tth = math.atan(r / cfg.distance_m)
        return {W.R_MM: 1e3 * r, W.TTH_RAD: tth, W.TTH_DEG: math.degrees(tth),
                W.Q_NM: 4e-9 * math.pi * math.sin(tth / 2) / cfg.wavelength_m,
                W.Q_A: 4e-10 * math.pi * math.sin(tth / 2) / cfg.wavelength_m}[cfg.unit]
    return u(rmin), u(rmax)


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_ranges_and_matrix_statistics(oracle, workloads, name):
    cfg = workloads.CONFIGS[name]
    ref = gold("survey_table_8a.json")[name]
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    c0, c1 = _closed_form_range(cfg, workloads)
    assert u0 == pytest.approx(c0, rel=1e-14, abs=1e-300)
    assert u1 == pytest.approx(c1, rel=1e-14)
    # the survey prints 6 significant digits
    assert u0 == pytest.approx(ref["range"][0], rel=6e-6, abs=1e-12)
    assert u1 == pytest.approx(ref["range"][1], rel=6e-6)
    assert (u1 - u0) / cfg.npt == pytest.approx(ref["delta"], rel=6e-6)
    indptr, _, _ = oracle.csr(umin, umax, cfg.npt, u0, u1) if cfg.npix <= 2048 * 2048 else _csr_indptr_only(
        oracle, umin, umax, cfg, u0, u1)
    assert int(indptr[-1]) == ref["nnz"]
    rl = np.diff(indptr)
    assert int(rl.min()) == ref["row_len"]["min"]
    assert int(rl.max()) == ref["row_len"]["max"]
    assert float(np.median(rl)) == pytest.approx(ref["row_len"]["median"], abs=1.0)
    assert float(rl.mean()) == pytest.approx(ref["row_len"]["mean"], abs=1.0)


def _csr_indptr_only(oracle, umin, umax, cfg, u0, u1):
    import ctypes as C
    indptr = np.zeros(cfg.npt + 1, dtype=np.int64)
    dp = C.POINTER(C.c_double)
    oracle.lib().aio_csr(umin.ctypes.data_as(dp), umax.ctypes.data_as(dp), umin.size, cfg.npt, u0, u1,
                         indptr.ctypes.data_as(C.POINTER(C.c_int64)), None, None)
    return indptr, None, None


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
def test_bins_per_pixel_histogram(oracle, workloads, name):
    cfg = workloads.CONFIGS[name]
    ref = gold("survey_table_8a.json")[name]["bins_per_pixel"]
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    _, indices, _ = oracle.csr(umin, umax, cfg.npt, u0, u1)
    per_pixel = np.bincount(indices, minlength=cfg.npix)
    hist = np.bincount(per_pixel)
    for k, v in ref.items():
        assert (int(hist[int(k)]) if int(k) < hist.size else 0) == v
    assert hist.sum() == cfg.npix and hist[0] == 0


def test_lut_to_csr_size_ratio_matches_paper(oracle, workloads):
    # CSR "reduces the size of the storage needed, as compared to the LUT, by a factor two to three"
    cfg = workloads.CONFIGS["cfg2"]
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    indptr, _, _ = _csr_indptr_only(oracle, umin, umax, cfg, u0, u1)
    rl = np.diff(indptr)
    ratio = cfg.npt * rl.max() / rl.sum()
    assert 1.7 < ratio < 3.0


def test_eightfold_symmetry_and_scale_invariance(oracle, workloads):
    W = workloads
    cfg = W.tiny_config(32, 32, center_x=16.0, center_y=16.0, unit=W.TTH_DEG, npt=25)
    umin, umax = oracle.pixel_bounds(cfg)
    a, b = umin.reshape(32, 32), umax.reshape(32, 32)
    for arr in (a, b):
        assert np.array_equal(arr, arr[::-1, :]) and np.array_equal(arr, arr[:, ::-1]) and np.array_equal(arr, arr.T)
    # scaling pixel size and distance by the same factor leaves 2theta untouched (power of two: exact)
    cfg2 = W.scaled(cfg, pixel_m=cfg.pixel_m * 4, distance_m=cfg.distance_m * 4)
    umin2, umax2 = oracle.pixel_bounds(cfg2)
    assert np.array_equal(umin, umin2) and np.array_equal(umax, umax2)


# ----------------------------------------------------------------------------------------------------------------
# O5-O7: invariants the paper states, and special cases that reduce to numpy / scipy
# ----------------------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def cfg1b_case(oracle, workloads):
    cfg = workloads.CONFIGS["cfg1b"]
    fr = workloads.make_frame(cfg)
    return cfg, fr, oracle.integrate1d(cfg, fr)


def test_conservation_of_signal_and_pixels(cfg1b_case):
    # sum(image) = sum(weighted histogram); sum(unweighted histogram) = number of pixels
    cfg, fr, r = cfg1b_case
    assert r["sum_signal"].sum() == pytest.approx(fr.image.astype(np.float64).sum(), rel=1e-13)
    assert r["count"].sum() == pytest.approx(cfg.npix, rel=1e-13)


def test_every_pixel_coefficients_sum_to_one(oracle, workloads):
    cfg = workloads.CONFIGS["cfg1"]
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    _, indices, data = oracle.csr(umin, umax, cfg.npt, u0, u1)
    sums = np.bincount(indices, weights=data, minlength=cfg.npix)
    assert np.allclose(sums, 1.0, rtol=0, atol=1e-12)


def test_uniform_image_gives_constant_profile(oracle, workloads):
    cfg = workloads.CONFIGS["cfg1"]
    r = oracle.integrate1d(cfg, workloads.Frame(image=np.full((cfg.height, cfg.width), 7.25)))
    assert np.all(r["count"] > 0)
    assert np.allclose(r["intensity"], 7.25, rtol=1e-13)


def test_single_bin_is_the_plain_mean(oracle, workloads):
    # mean = sum / number of contributing pixels
    cfg = workloads.scaled(workloads.CONFIGS["cfg1b"], npt=1)
    fr = workloads.make_frame(cfg)
    r = oracle.integrate1d(cfg, fr)
    assert r["intensity"][0] == pytest.approx(fr.image.astype(np.float64).mean(), rel=1e-13)
    assert r["count"][0] == pytest.approx(cfg.npix, rel=1e-14)


def test_profile_equals_scipy_csr_product(oracle, workloads, cfg1b_case):
    # data / indices / indptr are "fully compatible with the scipy.sparse.csr.csr_matrix constructor"
    import scipy.sparse as sp
    cfg, fr, r = cfg1b_case
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = r["range"]
    indptr, indices, data = oracle.csr(umin, umax, cfg.npt, u0, u1)
    M = sp.csr_matrix((data, indices, indptr), shape=(cfg.npt, cfg.npix))
    assert M.has_sorted_indices
    v = fr.image.astype(np.float64).ravel()
    assert np.allclose(M @ v, r["sum_signal"], rtol=1e-12)
    assert np.allclose(M @ np.ones(cfg.npix), r["count"], rtol=1e-12)


def test_no_split_limit_matches_numpy_histogram(oracle, workloads):
    # PAPER.md:88-91 azimint_hist: with bins much wider than a pixel almost no pixel is split, so the split profile
    # must approach the two-histogram result on pixel-centre radii.
    W = workloads
    cfg = W.scaled(W.CONFIGS["cfg1b"], npt=4, unit=W.R_MM)
    fr = W.make_frame(cfg)
    r = oracle.integrate1d(cfg, fr)
    x = (np.arange(cfg.width) + 0.5 - cfg.center_x_px) * cfg.pixel_m
    y = (np.arange(cfg.height) + 0.5 - cfg.center_y_px) * cfg.pixel_m
    radius = 1e3 * np.sqrt(x[None, :] ** 2 + y[:, None] ** 2).ravel()
    histu = np.histogram(radius, 4, range=r["range"])[0]
    histw = np.histogram(radius, 4, range=r["range"], weights=fr.image.astype(np.float64).ravel())[0]
    assert np.allclose(r["count"], histu, rtol=0.03)
    assert np.allclose(r["intensity"], histw / histu, rtol=0.03)


@pytest.mark.parametrize("unit,key", [("TTH_DEG", "tth_deg"), ("Q_NM", "q_nm"), ("R_MM", "r_mm")])
def test_noise_free_rings_peak_at_bragg_positions(oracle, workloads, unit, key):
    # PAPER.md:25 Bragg's law + PAPER.md:40-41, 50 unit formulas; positions from tests/golden/bragg_gold.json
    W = workloads
    g = gold("bragg_gold.json")
    cfg = W.scaled(W.CONFIGS["cfg2"], height=1024, width=1024, center_x_px=0.0, center_y_px=0.0,
                   unit=getattr(W, unit), npt=1500)
    fr = W.make_frame(cfg, noise=False)
    r = oracle.integrate1d(cfg, fr)
    delta = r["radial"][1] - r["radial"][0]
    peaks = [b for b in range(1, cfg.npt - 1)
             if r["intensity"][b] > 200 and r["intensity"][b] >= r["intensity"][b - 1]
             and r["intensity"][b] > r["intensity"][b + 1]]
    expect = [u for u in g[key] if r["range"][0] + 5 * delta < u < r["range"][1] - 5 * delta]
    assert len(expect) >= 4 and len(peaks) == len(expect)
    for b, u in zip(peaks, expect):
        assert abs(r["radial"][b] - u) <= 1.01 * delta + 5e-4 * u     # golden values carry 5 digits


def test_generalised_uniform_with_corrections(oracle, workloads):
    # I = k * flat * solidangle * polarization + dark  =>  profile == k everywhere (O5 with PAPER.md:240's corrections)
    W = workloads
    cfg = W.scaled(W.CONFIGS["cfg1b"], corrections=True, unit=W.Q_NM, npt=80)
    dark, flat, solid, pol, mask = W.correction_arrays(cfg)
    k = 3.5
    img = k * flat.astype(np.float64) * solid.astype(np.float64) * pol.astype(np.float64) + dark.astype(np.float64)
    fr = W.Frame(image=img, dark=dark, flat=flat, solidangle=solid, polarization=pol, mask=mask)
    r = oracle.integrate1d(cfg, fr)
    ok = r["count"] > 0
    assert ok.sum() > 70
    assert np.allclose(r["intensity"][ok], k, rtol=1e-12)


def test_mask_removes_exactly_the_masked_coefficients(oracle, workloads):
    W = workloads
    cfg = W.CONFIGS["cfg1b"]
    fr = W.make_frame(cfg)
    full = oracle.integrate1d(cfg, fr)
    mask = np.zeros((cfg.height, cfg.width), dtype=np.uint8)
    masked = [(10, 20), (100, 100), (128, 127), (255, 0)]
    for i, j in masked:
        mask[i, j] = 1
    part = oracle.integrate1d(cfg, W.Frame(image=fr.image, mask=mask))
    umin, umax = oracle.pixel_bounds(cfg)
    dC = np.zeros(cfg.npt)
    dS = np.zeros(cfg.npt)
    for i, j in masked:
        p = i * cfg.width + j
        bins, coefs = oracle.split(umin[p], umax[p], *full["range"], cfg.npt)
        for b, c in zip(bins, coefs):
            dC[b] += c
            dS[b] += c * float(fr.image[i, j])
    assert np.allclose(full["count"] - part["count"], dC, atol=1e-10)
    assert np.allclose(full["sum_signal"] - part["sum_signal"], dS, atol=1e-7)
    assert part["range"] == full["range"]          # the automatic range ignores the mask (reading 4)


def test_invalid_denominator_and_empty_bins(oracle, workloads):
    W = workloads
    cfg = W.tiny_config(8, 8, center_x=4.0, center_y=4.0, unit=W.R_MM, npt=6)
    img = np.arange(64, dtype=np.float64).reshape(8, 8)
    flat = np.ones((8, 8)); flat[2, 3] = 0.0
    a = oracle.integrate1d(cfg, W.Frame(image=img, flat=flat))
    m = np.zeros((8, 8), dtype=np.uint8); m[2, 3] = 1
    b = oracle.integrate1d(cfg, W.Frame(image=img, mask=m))
    assert np.array_equal(a["intensity"], b["intensity"]) and np.array_equal(a["count"], b["count"])
    # everything masked -> every bin empty -> empty value, zero sums (reading 6)
    e = oracle.integrate1d(cfg, W.Frame(image=img, mask=np.ones((8, 8), dtype=np.uint8)), empty=-1.0)
    assert np.all(e["intensity"] == -1.0) and np.all(e["count"] == 0) and np.all(e["sum_signal"] == 0)


def test_threaded_variant_agrees_with_single_thread(oracle, workloads):
    # one private histogram pair per thread, merged at the end -- only the summation order changes
    cfg = workloads.CONFIGS["cfg1b"]
    fr = workloads.make_frame(cfg)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    r1 = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, fr.image, nthreads=1)
    r4 = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, fr.image, nthreads=4)
    assert np.allclose(r1["sum_signal"], r4["sum_signal"], rtol=1e-13)
    assert np.allclose(r1["count"], r4["count"], rtol=1e-13)


def test_a_pixel_spanning_more_bins_than_the_oracle_buffers_is_an_error_not_a_clamp(oracle, workloads):
    # one pixel over 5000 bins: both the scatter and the CSR routine refuse (-3) instead of dropping contributions
    W = workloads
    cfg = W.tiny_config(1, 1, center_x=0.5, center_y=0.5, unit=W.R_MM, npt=5000)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    with pytest.raises(ValueError, match="-3"):
        oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, np.ones(1))
    with pytest.raises(ValueError, match="-3"):
        oracle.csr(umin, umax, cfg.npt, u0, u1)
    # 4096 bins is still fine, and the pixel is spread evenly: every coefficient 1 / 4096
    cfg = W.scaled(cfg, npt=4096)
    r = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, np.full(1, 3.0))
    assert r["count"] == pytest.approx(np.full(4096, 1.0 / 4096), rel=1e-9)
    assert r["intensity"] == pytest.approx(np.full(4096, 3.0), rel=1e-12)


# ----------------------------------------------------------------------------------------------------------------
# the split-normalisation estimator (sum c (I - dark) over sum c flat Omega P)
# ----------------------------------------------------------------------------------------------------------------
def test_split_normalisation_against_scipy_products_and_closed_forms(oracle, workloads):
    W = workloads
    cfg = W.tiny_config(40, 52, center_x=20.3, center_y=31.1, unit=W.TTH_DEG, npt=37)
    rng = np.random.default_rng(21)
    shape = (cfg.height, cfg.width)
    img = rng.poisson(300.0, size=shape).astype(np.float64)
    dark = rng.poisson(5.0, size=shape).astype(np.float64)
    flat = rng.uniform(0.8, 1.2, size=shape)
    sa = rng.uniform(0.7, 1.0, size=shape)
    pol = rng.uniform(0.9, 1.0, size=shape)
    mask = (rng.random(shape) < 0.07).astype(np.uint8)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)
    r = oracle.integrate1d_bounds_split(umin, umax, cfg.npt, u0, u1, img, dark, flat, sa, pol, mask)
    # the same sums as two products of the (separately pinned) CSR matrix with masked vectors
    import scipy.sparse as sp
    indptr, indices, data = oracle.csr(umin, umax, cfg.npt, u0, u1)
    m = sp.csr_matrix((data, indices, indptr), shape=(cfg.npt, cfg.npix))
    ok = (mask.ravel() == 0)
    num = np.where(ok, (img - dark).ravel(), 0.0)
    den = np.where(ok, (flat * sa * pol).ravel(), 0.0)
    assert r["sum_signal"] == pytest.approx(m @ num, rel=1e-12)
    assert r["sum_norm"] == pytest.approx(m @ den, rel=1e-12)
    assert r["intensity"] == pytest.approx((m @ num) / (m @ den), rel=1e-12)
    # I = k * flat * Omega * P + dark  =>  the ratio of the sums is k in every bin, whatever the mask
    k = 12.5
    r2 = oracle.integrate1d_bounds_split(umin, umax, cfg.npt, u0, u1, k * flat * sa * pol + dark, dark, flat, sa, pol, mask)
    assert r2["intensity"] == pytest.approx(np.full(cfg.npt, k), rel=1e-13)
    # without a denominator the normalisation is the unweighted histogram: the default estimator
    r3 = oracle.integrate1d_bounds_split(umin, umax, cfg.npt, u0, u1, img, dark, None, None, None, mask)
    r4 = oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, img, dark, None, None, None, mask)
    assert r3["intensity"] == pytest.approx(r4["intensity"], rel=1e-14)
    assert r3["sum_norm"] == pytest.approx(r4["count"], rel=1e-14)


def test_non_finite_inputs_are_exactly_a_masked_pixel(oracle, workloads):
    """DESIGN.md reading 8 of PAPER.md:240: a pixel whose numerator I - dark or whose denominator flat x solid angle x
    polarisation is not finite (or whose denominator is 0) is an invalid pixel.  Hand case: each of a NaN pixel, an Inf
    pixel, an Inf / NaN dark current, an Inf / NaN / zero flat, solid angle or polarisation gives bit for bit the profile of
    the clean inputs with that one pixel masked -- also in count, which would keep the pixel's weight if only the signal
    were dropped."""
    W = workloads
    cfg = W.tiny_config(12, 15, center_x=4.2, center_y=6.9, unit=W.TTH_DEG, npt=9)
    rng = np.random.default_rng(77)
    shape = (cfg.height, cfg.width)
    clean = dict(image=rng.poisson(100.0, size=shape).astype(np.float64), dark=rng.poisson(5.0, size=shape).astype(np.float64),
                 flat=rng.uniform(0.9, 1.1, size=shape), solidangle=rng.uniform(0.7, 1.0, size=shape),
                 polarization=rng.uniform(0.95, 1.0, size=shape))
    base_mask = (rng.random(shape) < 0.1).astype(np.uint8)
    umin, umax = oracle.pixel_bounds(cfg)
    u0, u1 = oracle.auto_range(umin, umax)

    def run(arrays, mask):
        return oracle.integrate1d_bounds(umin, umax, cfg.npt, u0, u1, arrays["image"], arrays["dark"], arrays["flat"],
                                         arrays["solidangle"], arrays["polarization"], mask, empty=-1.0)
    spot = (5, 7)
    assert base_mask[spot] == 0
    masked = base_mask.copy()
    masked[spot] = 1
    want = run(clean, masked)
    unmasked = run(clean, base_mask)
    assert np.abs(want["count"] - unmasked["count"]).max() > 0.1          # the pixel matters
    cases = [("image", np.nan), ("image", np.inf), ("image", -np.inf), ("dark", np.inf), ("dark", np.nan),
             ("flat", np.inf), ("flat", np.nan), ("flat", 0.0), ("solidangle", np.nan), ("solidangle", 0.0),
             ("polarization", -np.inf), ("polarization", 0.0)]
    for name, bad in cases:
        arrays = {k: v.copy() for k, v in clean.items()}
        arrays[name][spot] = bad
        got = run(arrays, base_mask)
        for k in ("sum_signal", "count", "intensity"):
            assert np.array_equal(got[k], want[k]), (name, bad, k)
    # Inf - Inf in the numerator, and a non-finite value under the mask (must stay harmless)
    arrays = {k: v.copy() for k, v in clean.items()}
    arrays["image"][spot] = np.inf
    arrays["dark"][spot] = np.inf
    arrays["image"][np.nonzero(base_mask)[0][0], np.nonzero(base_mask)[1][0]] = np.nan
    got = run(arrays, base_mask)
    for k in ("sum_signal", "count", "intensity"):
        assert np.array_equal(got[k], want[k]), k
