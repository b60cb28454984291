"""ctypes front-end of oracle/azint_oracle.c -- TEST INFRASTRUCTURE, not the product.

Argument marshalling only (dtype conversion to float64 is exact for the float32 / int32 / uint16 inputs used); every
step of O1-O7 runs in the C file, which cites the paper passage it follows.  Imports nothing from
paper_1412_6367_b200 (the seeded input generators are passed in by the caller as plain numpy arrays).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build


class Geometry(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("distance_m", "pixel_y_m", "pixel_x_m", "center_y_px", "center_x_px", "wavelength_m")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, u8p = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_uint8)
        L.aio_pixel_bounds.argtypes = [C.POINTER(Geometry), C.c_int, C.c_int, C.c_int, dp, dp]
        L.aio_auto_range.argtypes = [dp, dp, C.c_int64, dp, dp]
        L.aio_split.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, ip, dp, C.c_int]
        L.aio_integrate1d_bounds.argtypes = [dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double,
                                             dp, dp, dp, dp, dp, u8p, C.c_double, C.c_int, dp, dp, dp, dp]
        L.aio_integrate1d_bounds_split.argtypes = [dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double,
                                                   dp, dp, dp, dp, dp, u8p, C.c_double, dp, dp, dp]
        L.aio_integrate1d.argtypes = [C.POINTER(Geometry), C.c_int, C.c_int, C.c_int, C.c_int, dp,
                                      dp, dp, dp, dp, dp, u8p, C.c_double, dp, dp, dp, dp, dp]
        L.aio_csr.argtypes = [dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double,
                              C.POINTER(C.c_int64), C.POINTER(C.c_int32), dp]
        L.aio_csr.restype = C.c_int64
        L.aio_pixel_chi_bounds.argtypes = [C.POINTER(Geometry), C.c_int, C.c_int, dp, dp]
        L.aio_split_azim.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, ip, dp, C.c_int]
        L.aio_integrate2d_bounds.argtypes = [dp, dp, dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double, C.c_int,
                                             C.c_double, C.c_double, dp, dp, dp, dp, dp, u8p, C.c_double, dp, dp, dp]
        L.aio_csr2d.argtypes = [dp, dp, dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double, C.c_int, C.c_double,
                                C.c_double, C.POINTER(C.c_int64), C.POINTER(C.c_int32), dp]
        L.aio_csr2d.restype = C.c_int64
        L.aio_pixel_corners.argtypes = [C.POINTER(Geometry), C.c_int, C.c_int, C.c_int, dp, dp, u8p]
        L.aio_split_full.argtypes = [dp, dp, C.c_double, C.c_double, C.c_int, ip, dp, C.c_int]
        L.aio_csr_full.argtypes = [dp, dp, u8p, dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double,
                                   C.POINTER(C.c_int64), C.POINTER(C.c_int32), dp]
        L.aio_csr_full.restype = C.c_int64
        L.aio_integrate1d_full.argtypes = [dp, dp, u8p, dp, dp, C.c_int64, C.c_int, C.c_double, C.c_double,
                                           dp, dp, dp, dp, dp, u8p, C.c_double, dp, dp, dp, dp]
        _lib = L
    return _lib


def _d(a):
    """float64 C-contiguous copy (or None) and its pointer."""
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.float64).ravel()
    return arr, arr.ctypes.data_as(C.POINTER(C.c_double))


def _m(a):
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.uint8).ravel()
    return arr, arr.ctypes.data_as(C.POINTER(C.c_uint8))


def geometry(cfg) -> Geometry:
    """cfg: any object with distance_m, pixel_m, center_x_px, center_y_px, wavelength_m (e.g. workloads.Config)."""
    return Geometry(cfg.distance_m, cfg.pixel_m, cfg.pixel_m, cfg.center_y_px, cfg.center_x_px, cfg.wavelength_m)


def pixel_bounds(cfg):
    n = cfg.height * cfg.width
    umin, umax = np.empty(n), np.empty(n)
    g = geometry(cfg)
    rc = lib().aio_pixel_bounds(C.byref(g), cfg.height, cfg.width, cfg.unit,
                                umin.ctypes.data_as(C.POINTER(C.c_double)), umax.ctypes.data_as(C.POINTER(C.c_double)))
    if rc:
        raise ValueError(f"aio_pixel_bounds: {rc}")
    return umin, umax


def auto_range(umin, umax):
    u0, u1 = C.c_double(), C.c_double()
    _, pmin = _d(umin)
    _, pmax = _d(umax)
    lib().aio_auto_range(pmin, pmax, umin.size, C.byref(u0), C.byref(u1))
    return u0.value, u1.value


def split(u_min, u_max, u0, u1, npt, cap=4096):
    bins = (C.c_int * cap)()
    coefs = (C.c_double * cap)()
    n = lib().aio_split(u_min, u_max, u0, u1, npt, bins, coefs, cap)
    return list(bins[:n]), list(coefs[:n])


def integrate1d_bounds(umin, umax, npt, u0, u1, image, dark=None, flat=None, solidangle=None, polarization=None,
                       mask=None, empty=0.0, nthreads=1):
    """O4-O7 over precomputed bounds; returns dict(radial, intensity, sum_signal, count) of float64 arrays."""
    keep = [_d(umin), _d(umax), _d(image), _d(dark), _d(flat), _d(solidangle), _d(polarization), _m(mask)]
    out = {k: np.empty(npt) for k in ("radial", "intensity", "sum_signal", "count")}
    po = [out[k].ctypes.data_as(C.POINTER(C.c_double)) for k in ("radial", "intensity", "sum_signal", "count")]
    rc = lib().aio_integrate1d_bounds(keep[0][1], keep[1][1], keep[0][0].size, npt, u0, u1,
                                      *[k[1] for k in keep[2:]], empty, nthreads, *po)
    if rc:
        raise ValueError(f"aio_integrate1d_bounds: {rc}")
    return out


def integrate1d_bounds_split(umin, umax, npt, u0, u1, image, dark=None, flat=None, solidangle=None, polarization=None,
                             mask=None, empty=0.0):
    """The split-normalisation estimator: dict(intensity, sum_signal, sum_norm); `count` is an alias of sum_norm."""
    keep = [_d(umin), _d(umax), _d(image), _d(dark), _d(flat), _d(solidangle), _d(polarization), _m(mask)]
    out = {k: np.empty(npt) for k in ("intensity", "sum_signal", "sum_norm")}
    po = [out[k].ctypes.data_as(C.POINTER(C.c_double)) for k in ("intensity", "sum_signal", "sum_norm")]
    rc = lib().aio_integrate1d_bounds_split(keep[0][1], keep[1][1], keep[0][0].size, npt, u0, u1,
                                            *[k[1] for k in keep[2:]], empty, *po)
    if rc:
        raise ValueError(f"aio_integrate1d_bounds_split: {rc}")
    out["count"] = out["sum_norm"]
    return out


def integrate1d(cfg, frame, radial_range=None, empty=0.0):
    """O1-O7 for a workloads.Config-like `cfg` and a workloads.Frame-like `frame`."""
    keep = [_d(frame.image), _d(frame.dark), _d(frame.flat), _d(frame.solidangle), _d(frame.polarization),
            _m(frame.mask)]
    npt = cfg.npt
    out = {k: np.empty(npt) for k in ("radial", "intensity", "sum_signal", "count")}
    po = [out[k].ctypes.data_as(C.POINTER(C.c_double)) for k in ("radial", "intensity", "sum_signal", "count")]
    rng = None if radial_range is None else (C.c_double * 2)(*radial_range)
    rout = (C.c_double * 2)()
    g = geometry(cfg)
    rc = lib().aio_integrate1d(C.byref(g), cfg.height, cfg.width, npt, cfg.unit, rng, *[k[1] for k in keep], empty,
                               *po, rout)
    if rc:
        raise ValueError(f"aio_integrate1d: {rc}")
    out["range"] = (rout[0], rout[1])
    return out


def csr(umin, umax, npt, u0, u1):
    """Oracle CSR: (indptr int64[npt+1], indices int32[nnz], data float64[nnz])."""
    keep = [_d(umin), _d(umax)]
    indptr = np.zeros(npt + 1, dtype=np.int64)
    pi = indptr.ctypes.data_as(C.POINTER(C.c_int64))
    nnz = lib().aio_csr(keep[0][1], keep[1][1], keep[0][0].size, npt, u0, u1, pi, None, None)
    if nnz < 0:
        raise ValueError(f"aio_csr: {nnz}")
    indices = np.empty(nnz, dtype=np.int32)
    data = np.empty(nnz, dtype=np.float64)
    lib().aio_csr(keep[0][1], keep[1][1], keep[0][0].size, npt, u0, u1, pi,
                  indices.ctypes.data_as(C.POINTER(C.c_int32)), data.ctypes.data_as(C.POINTER(C.c_double)))
    return indptr, indices, data


# ---- bidimensional integration (azimuthal x radial bins) ----------------------------------------------------------------
FULL_CIRCLE = (-np.pi, np.pi)


def pixel_chi_bounds(cfg):
    """(chi_lo, chi_w): every pixel covers [chi_lo, chi_lo + chi_w] on the periodic azimuthal axis, radians."""
    n = cfg.height * cfg.width
    lo, w = np.empty(n), np.empty(n)
    g = geometry(cfg)
    rc = lib().aio_pixel_chi_bounds(C.byref(g), cfg.height, cfg.width, lo.ctypes.data_as(C.POINTER(C.c_double)),
                                    w.ctypes.data_as(C.POINTER(C.c_double)))
    if rc:
        raise ValueError(f"aio_pixel_chi_bounds: {rc}")
    return lo, w


def split_azim(chi_lo, w, c0, c1, npt, cap=4096):
    bins = (C.c_int * cap)()
    coefs = (C.c_double * cap)()
    n = lib().aio_split_azim(chi_lo, w, c0, c1, npt, bins, coefs, cap)
    return list(bins[:n]), list(coefs[:n])


def integrate2d_bounds(umin, umax, chi_lo, chi_w, npt_rad, u0, u1, npt_azim, c0, c1, image, dark=None, flat=None,
                       solidangle=None, polarization=None, mask=None, empty=0.0):
    """Forward scatter into [npt_azim][npt_rad] bins; dict(radial, azimuthal, intensity, sum_signal, count)."""
    keep = [_d(umin), _d(umax), _d(chi_lo), _d(chi_w), _d(image), _d(dark), _d(flat), _d(solidangle),
            _d(polarization), _m(mask)]
    out = {k: np.empty((npt_azim, npt_rad)) for k in ("intensity", "sum_signal", "count")}
    po = [out[k].ctypes.data_as(C.POINTER(C.c_double)) for k in ("intensity", "sum_signal", "count")]
    rc = lib().aio_integrate2d_bounds(keep[0][1], keep[1][1], keep[2][1], keep[3][1], keep[0][0].size, npt_rad, u0, u1,
                                      npt_azim, c0, c1, *[k[1] for k in keep[4:]], empty, *po)
    if rc:
        raise ValueError(f"aio_integrate2d_bounds: {rc}")
    out["radial"] = u0 + (np.arange(npt_rad) + 0.5) * (u1 - u0) / npt_rad
    out["azimuthal"] = c0 + (np.arange(npt_azim) + 0.5) * (c1 - c0) / npt_azim
    return out


def integrate2d(cfg, frame, radial_range=None, azim_range=None, empty=0.0):
    """O1-O7 on both axes for a workloads.Config-like `cfg` with npt (radial) and npt_azim bins."""
    umin, umax = pixel_bounds(cfg)
    u0, u1 = auto_range(umin, umax) if radial_range is None else radial_range
    c0, c1 = FULL_CIRCLE if azim_range is None else azim_range
    lo, w = pixel_chi_bounds(cfg)
    out = integrate2d_bounds(umin, umax, lo, w, cfg.npt, u0, u1, cfg.npt_azim, c0, c1, frame.image, frame.dark,
                             frame.flat, frame.solidangle, frame.polarization, frame.mask, empty=empty)
    out["range"] = (u0, u1)
    out["azim_range"] = (c0, c1)
    return out


def csr2d(umin, umax, chi_lo, chi_w, npt_rad, u0, u1, npt_azim, c0, c1):
    """Oracle CSR of the 2D matrix, row = a * npt_rad + r: (indptr int64, indices int32, data float64)."""
    keep = [_d(umin), _d(umax), _d(chi_lo), _d(chi_w)]
    nb = npt_rad * npt_azim
    indptr = np.zeros(nb + 1, dtype=np.int64)
    pi = indptr.ctypes.data_as(C.POINTER(C.c_int64))
    a = [k[1] for k in keep]
    nnz = lib().aio_csr2d(*a, keep[0][0].size, npt_rad, u0, u1, npt_azim, c0, c1, pi, None, None)
    if nnz < 0:
        raise ValueError(f"aio_csr2d: {nnz}")
    indices = np.empty(nnz, dtype=np.int32)
    data = np.empty(nnz, dtype=np.float64)
    lib().aio_csr2d(*a, keep[0][0].size, npt_rad, u0, u1, npt_azim, c0, c1, pi,
                    indices.ctypes.data_as(C.POINTER(C.c_int32)), data.ctypes.data_as(C.POINTER(C.c_double)))
    return indptr, indices, data


# ---- full pixel splitting -------------------------------------------------------------------------------
def pixel_corners(cfg):
    """(u4 [npix][4], chi4 [npix][4], has_quad [npix]): the pixels' corners in the (radial unit, chi) plane."""
    n = cfg.height * cfg.width
    u4, c4, q = np.empty((n, 4)), np.empty((n, 4)), np.empty(n, dtype=np.uint8)
    g = geometry(cfg)
    dp = C.POINTER(C.c_double)
    rc = lib().aio_pixel_corners(C.byref(g), cfg.height, cfg.width, cfg.unit, u4.ctypes.data_as(dp), c4.ctypes.data_as(dp),
                                 q.ctypes.data_as(C.POINTER(C.c_uint8)))
    if rc:
        raise ValueError(f"aio_pixel_corners: {rc}")
    return u4, c4, q


def split_full(u4, chi4, u0, u1, npt, cap=4096):
    bins = (C.c_int * cap)()
    coefs = (C.c_double * cap)()
    dp = C.POINTER(C.c_double)
    a, b = np.ascontiguousarray(u4, dtype=np.float64), np.ascontiguousarray(chi4, dtype=np.float64)
    n = lib().aio_split_full(a.ctypes.data_as(dp), b.ctypes.data_as(dp), u0, u1, npt, bins, coefs, cap)
    return list(bins[:n]), list(coefs[:n])


def csr_full(cfg, u0=None, u1=None):
    """Oracle CSR of the full-splitting matrix (the range defaults to the bounding-box automatic range)."""
    umin, umax = pixel_bounds(cfg)
    if u0 is None:
        u0, u1 = auto_range(umin, umax)
    u4, c4, q = pixel_corners(cfg)
    dp = C.POINTER(C.c_double)
    indptr = np.zeros(cfg.npt + 1, dtype=np.int64)
    pi = indptr.ctypes.data_as(C.POINTER(C.c_int64))
    args = (u4.ctypes.data_as(dp), c4.ctypes.data_as(dp), q.ctypes.data_as(C.POINTER(C.c_uint8)),
            umin.ctypes.data_as(dp), umax.ctypes.data_as(dp), umin.size, cfg.npt, u0, u1, pi)
    nnz = lib().aio_csr_full(*args, None, None)
    if nnz < 0:
        raise ValueError(f"aio_csr_full: {nnz}")
    indices = np.empty(nnz, dtype=np.int32)
    data = np.empty(nnz, dtype=np.float64)
    lib().aio_csr_full(*args, indices.ctypes.data_as(C.POINTER(C.c_int32)), data.ctypes.data_as(dp))
    return indptr, indices, data, (u0, u1)


def integrate1d_full(cfg, frame, empty=0.0):
    """Full pixel splitting of one frame (aio_integrate1d_full: the per-pixel forward scatter of PAPER.md:126-130) over
    the bounding-box automatic range: dict(radial, intensity, sum_signal, count).  Marshalling only."""
    umin, umax = pixel_bounds(cfg)
    u0, u1 = auto_range(umin, umax)
    u4, c4, q = pixel_corners(cfg)
    return integrate1d_full_corners(u4, c4, q, umin, umax, cfg.npt, u0, u1, frame.image, frame.dark, frame.flat,
                                    frame.solidangle, frame.polarization, frame.mask, empty=empty)


def integrate1d_full_corners(u4, c4, has_quad, umin, umax, npt, u0, u1, image, dark=None, flat=None, solidangle=None,
                             polarization=None, mask=None, empty=0.0):
    keep = [_d(u4), _d(c4), _m(has_quad), _d(umin), _d(umax), _d(image), _d(dark), _d(flat), _d(solidangle),
            _d(polarization), _m(mask)]
    out = {k: np.empty(npt) for k in ("radial", "intensity", "sum_signal", "count")}
    po = [out[k].ctypes.data_as(C.POINTER(C.c_double)) for k in ("radial", "intensity", "sum_signal", "count")]
    rc = lib().aio_integrate1d_full(keep[0][1], keep[1][1], keep[2][1], keep[3][1], keep[4][1], keep[3][0].size, npt,
                                    u0, u1, *[k[1] for k in keep[5:]], empty, *po)
    if rc:
        raise ValueError(f"aio_integrate1d_full: {rc}")
    out["range"] = (u0, u1)
    return out


def num_threads_available() -> int:
    return int(lib().aio_num_threads_available())
