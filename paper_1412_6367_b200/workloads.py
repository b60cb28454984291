"""Seeded synthetic inputs shared by the oracle (tests) and the CUDA path (tests, bench).

This module holds NONE of the method's arithmetic (no pixel bounds, no bin
assignment, no splitting, no accumulation): it only draws detector frames and
correction arrays with the shape, dtype and structure of the paper's workloads.
It imports neither ``oracle/`` nor the CUDA binding.

The paper benchmarks on real frames from the pyFAI test-suite (§6),
which are not available; these inputs stand in for them.  They follow the
paper's simulated test case (§3.1: gold powder, lambda = 1e-10 m,
all rings of equal intensity, 2048x2048 pixels of 1e-4 m at 0.1 m) and the image
sizes / integer dtypes of PAPER.md:194 and PAPER.md:257 (Table 3).  The ring
model, seeds and mask layout are the recipe of SURVEY.md §8(d) / DESIGN.md §4.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
import math

import numpy as np

BASE_SEED = 14126367
A_GOLD_M = 4.078e-10          # fcc gold lattice constant (BASELINE.json configs[0])
RING_SIGMA_PX = 1.5
RING_PEAK = 1000.0
BACKGROUND = 10.0

# unit names follow include/azint.h (ai_unit)
R_MM, TTH_DEG, TTH_RAD, Q_NM, Q_A = 0, 1, 2, 3, 4
UNIT_NAMES = {R_MM: "r_mm", TTH_DEG: "2th_deg", TTH_RAD: "2th_rad", Q_NM: "q_nm^-1", Q_A: "q_A^-1"}


@dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json `configs` (geometry + binning + input recipe)."""
    name: str
    height: int
    width: int
    pixel_m: float
    distance_m: float
    wavelength_m: float
    center_x_px: float          # along the fast (column, j) axis
    center_y_px: float          # along the slow (row, i) axis
    unit: int
    npt: int
    dtype: str = "float32"      # dtype of the raw frame
    nframes: int = 1
    corrections: bool = False   # dark / flat / solid angle / polarisation / mask
    seed_index: int = 0
    note: str = ""
    npt_azim: int = 0           # > 0: bidimensional integration, azimuthal x radial bins (npt = radial bins)

    @property
    def npix(self) -> int:
        return self.height * self.width


CONFIGS = {
    # BASELINE.json configs[0]; literally has no ring on the image (SURVEY.md §8(c) reading 18)
    "cfg1": Config("cfg1", 256, 256, 1e-4, 0.1, 1e-10, 128.0, 128.0, TTH_DEG, 100, seed_index=1),
    # same detector, distance scaled by 1/8 so that five rings fall on the image
    "cfg1b": Config("cfg1b", 256, 256, 1e-4, 0.0125, 1e-10, 128.0, 128.0, TTH_DEG, 100, seed_index=11),
    # BASELINE.json configs[1]: the headline configuration (PAPER.md:50 test case)
    "cfg2": Config("cfg2", 2048, 2048, 1e-4, 0.1, 1e-10, 1024.0, 1024.0, R_MM, 1000, seed_index=2),
    # configs[2]: full preprocessing
    "cfg3": Config("cfg3", 2048, 2048, 1e-4, 0.1, 1e-10, 1024.0, 1024.0, Q_NM, 3000,
                   corrections=True, seed_index=3),
    # configs[3]: streaming batch of int32 frames
    "cfg4": Config("cfg4", 1024, 1024, 1e-4, 0.1, 1e-10, 512.0, 512.0, TTH_DEG, 1000,
                   dtype="int32", nframes=1024, seed_index=4),
    # configs[4]: off-image beam centre, rings are arcs
    "cfg5": Config("cfg5", 4096, 4096, 75e-6, 0.2, 1e-10, -200.0, 2048.0, Q_NM, 5000, seed_index=5),
    # bidimensional ("cake") integration of the headline frame (Fig. 3): 360 azimuthal x 500
    # radial bins over the full circle
    "cake2": Config("cake2", 2048, 2048, 1e-4, 0.1, 1e-10, 1024.0, 1024.0, R_MM, 500, seed_index=2, npt_azim=360),
    # Pilatus-1M shape of PAPER.md:257 (Table 3); pixel size is a reading
    "t3": Config("t3", 981, 1043, 172e-6, 0.1, 1e-10, 521.5, 490.5, TTH_DEG, 1000,
                 dtype="int32", seed_index=6),
}


def tiny_config(height: int, width: int, *, center_x: float, center_y: float, unit: int, npt: int,
                pixel_m: float = 1e-4, distance_m: float = 0.1, wavelength_m: float = 1e-10,
                name: str = "tiny") -> Config:
    return Config(name, height, width, pixel_m, distance_m, wavelength_m, center_x, center_y, unit, npt)


def fcc_reflections(max_n: int = 64):
    """(h,k,l) of the fcc-allowed reflections (all even or all odd), one per distinct h^2+k^2+l^2."""
    seen = {}
    hmax = int(math.isqrt(max_n)) + 1
    for h in range(hmax + 1):
        for k in range(h + 1):
            for l in range(k + 1):
                n = h * h + k * k + l * l
                if n == 0 or n > max_n:
                    continue
                par = {h % 2, k % 2, l % 2}
                if len(par) == 1 and n not in seen:
                    seen[n] = (h, k, l)
    return [seen[n] for n in sorted(seen)]


def ring_radii_px(cfg: Config):
    """Radii (in pixels) of the gold rings from Bragg's law: 2*theta = 2 asin(lambda / 2d),
    r = D tan(2 theta).  Returns [(hkl, radius_px)] for 2 theta < 90 degrees."""
    out = []
    for hkl in fcc_reflections():
        d = A_GOLD_M / math.sqrt(sum(v * v for v in hkl))
        s = cfg.wavelength_m / (2.0 * d)
        if s >= 1.0:
            continue
        tth = 2.0 * math.asin(s)
        if tth >= 0.5 * math.pi * 0.999:
            continue
        out.append((hkl, cfg.distance_m * math.tan(tth) / cfg.pixel_m))
    return out


def _rho_px(cfg: Config) -> np.ndarray:
    """Distance of every pixel centre (j + 1/2, i + 1/2) from the beam centre, in pixels."""
    x = (np.arange(cfg.width, dtype=np.float64) + 0.5) - cfg.center_x_px
    y = (np.arange(cfg.height, dtype=np.float64) + 0.5) - cfg.center_y_px
    return np.sqrt(x[None, :] ** 2 + y[:, None] ** 2)


def rings_on_image(cfg: Config):
    """The reflections whose ring comes within 5 sigma of the detector area."""
    xs = np.array([0.0, cfg.width]) - cfg.center_x_px
    ys = np.array([0.0, cfg.height]) - cfg.center_y_px
    rmax = float(np.sqrt(max(xs ** 2) + max(ys ** 2)))
    dx = 0.0 if xs[0] <= 0.0 <= xs[1] else float(min(abs(xs)))
    dy = 0.0 if ys[0] <= 0.0 <= ys[1] else float(min(abs(ys)))
    rmin = math.hypot(dx, dy)
    return [(hkl, r) for hkl, r in ring_radii_px(cfg) if rmin - 5 * RING_SIGMA_PX <= r <= rmax + 5 * RING_SIGMA_PX]


def ideal_image(cfg: Config, ring_scale: float = 1.0) -> np.ndarray:
    """Noise-free frame: background + equal-intensity Gaussian rings (PAPER.md:50 'the intensity of all
    rings is the same').  float64, shape (H, W)."""
    rho = _rho_px(cfg)
    img = np.full(rho.shape, BACKGROUND, dtype=np.float64)
    for _, r in rings_on_image(cfg):
        # only touch the annulus where the Gaussian is non-negligible
        sel = np.abs(rho - r) < 8.0 * RING_SIGMA_PX
        img[sel] += (RING_PEAK * ring_scale) * np.exp(-((rho[sel] - r) ** 2) / (2.0 * RING_SIGMA_PX ** 2))
    return img


def _rng(offset: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(BASE_SEED + offset))


@dataclass
class Frame:
    """Inputs of one ai_integrate1d call; absent corrections are None."""
    image: np.ndarray
    dark: np.ndarray | None = None
    flat: np.ndarray | None = None
    solidangle: np.ndarray | None = None
    polarization: np.ndarray | None = None
    mask: np.ndarray | None = None
    meta: dict = field(default_factory=dict)


def correction_arrays(cfg: Config):
    """dark ~ Poisson(5), flat ~ U(0.9, 1.1), solid angle cos^3(2 theta), polarisation factor 0.99, mask of 4 % random
    pixels plus two horizontal and two vertical 10-pixel gap stripes (BASELINE.json configs[2]).  Generator-only
    formulas (the method takes these as plain input arrays)."""
    k = cfg.seed_index
    H, W = cfg.height, cfg.width
    dark = _rng(100 * k + 3).poisson(5.0, size=(H, W)).astype(np.float32)
    flat = _rng(100 * k + 2).uniform(0.9, 1.1, size=(H, W)).astype(np.float32)
    x = ((np.arange(W, dtype=np.float64) + 0.5) - cfg.center_x_px) * cfg.pixel_m
    y = ((np.arange(H, dtype=np.float64) + 0.5) - cfg.center_y_px) * cfg.pixel_m
    r = np.sqrt(x[None, :] ** 2 + y[:, None] ** 2)
    tth = np.arctan(r / cfg.distance_m)
    chi = np.arctan2(y[:, None], x[None, :])
    solid = np.cos(tth) ** 3
    f = 0.99
    pol = 0.5 * (1.0 + np.cos(tth) ** 2 - f * np.cos(2.0 * chi) * np.sin(tth) ** 2)
    mask = (_rng(100 * k + 1).random(size=(H, W)) < 0.04).astype(np.uint8)
    for a in (H // 3 - 4, (2 * H) // 3 - 5):        # 678 and 1360 for H = 2048
        mask[a:a + 10, :] = 1
    for a in (W // 3 - 4, (2 * W) // 3 - 5):
        mask[:, a:a + 10] = 1
    return dark, flat, solid.astype(np.float32), pol.astype(np.float32), mask


def make_frame(cfg: Config, frame_index: int = 0, *, noise: bool = True) -> Frame:
    """One seeded frame of `cfg` (frame_index only matters for multi-frame configs)."""
    k = cfg.seed_index
    if cfg.nframes > 1:
        rng = _rng(1000 * k + frame_index)
        scale = float(rng.uniform(0.5, 2.0))     # per-frame ring intensity (BASELINE.json configs[3])
    else:
        rng = _rng(k if frame_index == 0 else 1000 * k + frame_index)
        scale = 1.0
    ideal = ideal_image(cfg, scale)
    fr = Frame(image=None, meta={"scale": scale})
    if cfg.corrections:
        dark, flat, solid, pol, mask = correction_arrays(cfg)
        ideal = ideal * flat.astype(np.float64) * solid.astype(np.float64) * pol.astype(np.float64) + 5.0
        fr.dark, fr.flat, fr.solidangle, fr.polarization, fr.mask = dark, flat, solid, pol, mask
    raw = rng.poisson(ideal) if noise else ideal
    fr.image = np.ascontiguousarray(raw.astype(cfg.dtype))
    return fr


def make_frames(cfg: Config, nframes: int, *, start: int = 0) -> np.ndarray:
    """Stack of `nframes` raw frames, frame-major (as a detector streams them): shape (F, H, W)."""
    out = np.empty((nframes, cfg.height, cfg.width), dtype=cfg.dtype)
    base = ideal_image(cfg, 1.0) - BACKGROUND        # ring part at scale 1
    for f in range(nframes):
        rng = _rng(1000 * cfg.seed_index + start + f)
        scale = float(rng.uniform(0.5, 2.0)) if cfg.nframes > 1 else 1.0
        out[f] = rng.poisson(BACKGROUND + scale * base).astype(cfg.dtype)
    return out


def scaled(cfg: Config, **kw) -> Config:
    return replace(cfg, **kw)
