"""Comparators used by the GPU parity tests (tolerances are north_star's, restated in DESIGN.md section 7)."""
import numpy as np

REL_TOL = 1e-6          # per-bin relative error on intensity with compensated accumulation (BASELINE.json north_star)
COEF_ABS = 1e-7         # coefficients: |dc| <= 1e-6 c + 1e-7 (SURVEY.md section 8(c) "Numerics the builder should expect")
TIE_COEF = 1e-9         # an entry present on one side only must be a bin-edge tie: coefficient below this


def rel_err(got, want, floor=0.0):
    got = np.asarray(got, dtype=np.float64)
    want = np.asarray(want, dtype=np.float64)
    den = np.maximum(np.abs(want), floor)
    out = np.zeros_like(want)
    nz = den > 0
    out[nz] = np.abs(got[nz] - want[nz]) / den[nz]
    out[~nz] = np.abs(got[~nz])
    return out


def assert_profile(got, want, tol=REL_TOL, what="", floor_rel=0.0):
    """got: dict of float32 arrays from the CUDA path; want: oracle dict (float64).

    Pure per-bin relative error |got - want| / |want| <= tol on intensity, sum_signal and count for every bin the oracle
    fills.  floor_rel (default 0: none) is only for data whose dark-subtracted sums cancel to ~0 in some bin: there the
    denominator is max(|want|, floor_rel * max|want|), and the number of bins that needed it is returned as
    `floored_bins` so that the caller can report it.  None of the five configs needs it."""
    empty = want["count"] <= 0
    # bins the oracle calls empty must be empty on the GPU too (count exactly 0)
    assert np.array_equal(np.asarray(got["count"])[empty], np.zeros(empty.sum(), dtype=np.float32)), what
    ok = ~empty
    i_scale = np.abs(want["intensity"][ok]).max() if ok.any() else 1.0
    s_scale = np.abs(want["sum_signal"][ok]).max() if ok.any() else 1.0
    e_int = rel_err(np.asarray(got["intensity"])[ok], want["intensity"][ok], floor=floor_rel * i_scale)
    e_cnt = rel_err(np.asarray(got["count"])[ok], want["count"][ok])
    e_sum = rel_err(np.asarray(got["sum_signal"])[ok], want["sum_signal"][ok], floor=floor_rel * s_scale)
    floored = int((np.abs(want["intensity"][ok]) < floor_rel * i_scale).sum() +
                  (np.abs(want["sum_signal"][ok]) < floor_rel * s_scale).sum())
    worst = {"intensity": float(e_int.max(initial=0)), "count": float(e_cnt.max(initial=0)),
             "sum_signal": float(e_sum.max(initial=0)), "floored_bins": floored}
    for k in ("intensity", "count", "sum_signal"):
        assert worst[k] <= tol, (what, k, worst)
    return worst


def compare_csr(gpu, ora, npix, max_ties=None):
    """gpu: (indptr int32, indices int32, data float32); ora: (indptr int64, indices int32, data float64).
    Returns a report dict; raises AssertionError on a real difference.  max_ties: how many bin-edge ties (entries present
    on one side only, coefficient < TIE_COEF) are plausible; default max(8, 1e-5 nnz)."""
    gi, gx, gd = gpu
    oi, ox, od = ora
    rep = {"nnz_gpu": int(gi[-1]), "nnz_oracle": int(oi[-1]), "ties": 0, "coef_rel_fail": 0, "coef_max_rel": 0.0}
    if np.array_equal(gi, oi) and np.array_equal(gx, ox):
        g_d, o_d = gd.astype(np.float64), od
    else:
        npt = gi.size - 1
        grow = np.repeat(np.arange(npt, dtype=np.int64), np.diff(gi))
        orow = np.repeat(np.arange(npt, dtype=np.int64), np.diff(oi))
        gkey = grow * npix + gx
        okey = orow * npix + ox
        assert np.all(np.diff(gkey) > 0), "GPU CSR rows are not in ascending pixel order"
        only_g = ~np.isin(gkey, okey, assume_unique=True)
        only_o = ~np.isin(okey, gkey, assume_unique=True)
        rep["ties"] = int(only_g.sum() + only_o.sum())
        assert np.all(gd[only_g] < TIE_COEF), "GPU-only entries that are not bin-edge ties"
        assert np.all(od[only_o] < TIE_COEF), "oracle-only entries that are not bin-edge ties"
        cap = max(8, int(1e-5 * oi[-1])) if max_ties is None else max_ties
        assert rep["ties"] <= cap, f"too many edge ties: {rep['ties']}"
        g_d, o_d = gd[~only_g].astype(np.float64), od[~only_o]
    d = np.abs(g_d - o_d)
    assert np.all(d <= REL_TOL * np.abs(o_d) + COEF_ABS), f"coefficient mismatch, max abs diff {d.max()}"
    rel = d / np.maximum(np.abs(o_d), 1e-300)
    rep["coef_rel_fail"] = int((rel > REL_TOL).sum())
    rep["coef_max_rel"] = float(rel.max(initial=0))
    return rep
