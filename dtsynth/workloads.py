"""Seeded synthetic workloads standing in for the paper's ZTF data.

The five configurations follow BASELINE.json `configs` (CFG 1-5) with the readings listed in
DESIGN.md ("Readings" A13, A20 and "Input recipe").  Every array is a pure function of the
config's seed (see rng.py), so the CPU oracle and the CUDA path regenerate the same inputs
independently, and any sub-range (orbit block, single exposure, single pixel) can be produced on
its own.

This module holds NO arithmetic of the tracking method: no mean motion, no Kepler equation, no
orbit geometry, no projection of an orbit.  Where building a scene needs the forward chain
(tangent points that track an orbit, the pixel an injected source falls on) the caller passes a
`project_fn`; tests pass the oracle's, bench/smoke pass the library's `dt_project`.  The only
geometry here is spherical bookkeeping of the *pointing* (ecliptic lon/lat of a field centre ->
RA/Dec), which is survey metadata, not the method.

Two variants per config, as the paper itself distinguishes:
  * diffuse  (literal): candidates drawn over the whole config box, pointings as the config says;
  * focused  (`focused(cfg)`): `n_guides` seeded guide orbits; exposure j points at the apparent
    position of guide j mod G (from project_fn) plus a dither, and a fraction `focus_fraction` of
    the candidates are a guide's elements plus a small seeded perturbation -- "a narrow orbit family
    against images chosen along its track".  This is what exercises the gather/stack stage.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace
from typing import Callable, Optional, Tuple

import numpy as np

from . import rng

# ---- constants, shared AS NUMBERS by oracle and library (reading A1) -------------------
GAUSS_K = 0.01720209895                      # rad/day; GM_sun = k^2 AU^3/d^2
GM_SUN = 2.959122082855911025e-4             # AU^3 / day^2
C_AU_PER_DAY = 173.14463267424033            # 299792.458 km/s * 86400 s / 149597870.7 km
OBLIQUITY = 0.40909262775014904              # 23.439281 deg in rad
PIXEL_SCALE = 9.696273622190719e-07          # 0.2 arcsec in rad
DEG = math.pi / 180.0


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    n_exp: int
    span_days: float
    width: int
    height: int
    n_orbits: int
    a_range: Tuple[float, float]
    e_range: Tuple[float, float]
    i_range_deg: Tuple[float, float]
    tangent_mode: str            # "track" | "opposition" | "band" | "guides"
    tangent_half_deg: float
    variance_mode: int           # 0: per-exposure scalar, 1: fp32 plane (scalar broadcast)
    var_range: Tuple[float, float]
    n_injected: int
    amp_range: Tuple[float, float]
    grid: Optional[Tuple[int, int, int]] = None    # CFG 1 only: (na, ne, ni) half-open grid
    injected_node: Optional[Tuple[int, int, int]] = None
    # focused variant
    n_guides: int = 0
    focus_fraction: float = 0.0
    focus_spread: Tuple[float, float, float, float, float, float] = (0.0,) * 6  # half-widths

    @property
    def pairs(self) -> int:
        return self.n_orbits * self.n_exp

    @property
    def plane_pixels(self) -> int:
        return self.width * self.height

    def image_bytes(self) -> int:
        return self.n_exp * self.plane_pixels * 4 * (2 if self.variance_mode == 1 else 1)


CONFIGS = {
    # CFG 1 (A20): 50 x 10 x 20 half-open grid, node (25, 5, 5) = index 5105 is the injected orbit
    "tiny": Config("tiny", 0, 64, 30.0, 256, 256, 10_000, (2.2, 3.2), (0.0, 0.2), (0.0, 20.0),
                   "track", 0.0, 1, (1.0, 1.0), 1, (0.5, 0.5), grid=(50, 10, 20),
                   injected_node=(25, 5, 5)),
    "small_mba": Config("small_mba", 1, 500, 365.25, 2048, 2048, 1_000_000, (2.1, 3.3), (0.0, 0.3),
                        (0.0, 25.0), "opposition", 2.0, 0, (0.8, 1.2), 100, (0.3, 0.3)),
    "lsst": Config("lsst", 2, 2000, 1095.75, 4096, 4096, 10_000_000, (2.1, 3.3), (0.0, 0.3),
                   (0.0, 25.0), "opposition", 2.0, 1, (0.8, 1.2), 1000, (0.2, 0.5)),
    "neo": Config("neo", 3, 500, 730.5, 2048, 2048, 100_000_000, (0.8, 3.0), (0.0, 0.9),
                  (0.0, 60.0), "opposition", 2.0, 0, (0.8, 1.2), 500, (0.3, 0.3)),
    "tno": Config("tno", 4, 1000, 3652.5, 4096, 4096, 100_000_000, (30.0, 50.0), (0.0, 0.3),
                  (0.0, 30.0), "band", 5.0, 1, (0.8, 1.2), 1000, (0.1, 0.3)),
}

# (n_guides, fraction, half-widths (da AU, de, di, dOmega, domega, dM0 rad)) of the focused
# families: sized so that a family member stays within a fraction of its guide's footprint.
_FOCUS = {
    "tiny": (1, 0.5, (2e-5, 2e-5, 5e-5, 1e-5, 1e-5, 1e-5)),
    "small_mba": (16, 0.5, (2e-5, 2e-5, 5e-5, 1e-4, 1e-4, 1e-4)),
    "lsst": (16, 0.5, (2e-5, 2e-5, 5e-5, 1e-4, 1e-4, 1e-4)),
    "neo": (16, 0.5, (5e-6, 5e-6, 2e-5, 3e-5, 3e-5, 3e-5)),
    "tno": (4, 0.5, (2e-2, 2e-4, 2e-4, 4e-4, 4e-4, 4e-4)),
}


def scaled(cfg: Config, **kw) -> Config:
    """A reduced copy of a config (fewer orbits / exposures / smaller planes) for parity tests."""
    return replace(cfg, **kw)


def focused(cfg: Config, n_guides: Optional[int] = None, fraction: Optional[float] = None,
            spread=None) -> Config:
    """The focused variant of a config (see module docstring)."""
    g, f, s = _FOCUS[cfg.name.split("+")[0]]
    return replace(cfg, name=cfg.name + "+focused", tangent_mode="guides",
                   n_guides=g if n_guides is None else n_guides,
                   focus_fraction=f if fraction is None else fraction,
                   focus_spread=tuple(s if spread is None else spread),
                   grid=None, injected_node=None)


# ---- exposure metadata ----------------------------------------------------------------------------
def exposure_times(cfg: Config) -> np.ndarray:
    u = rng.uniform_np(cfg.seed, rng.STREAM_TIME, np.arange(cfg.n_exp))
    return np.sort(u * cfg.span_days)


def observer_ecliptic(t: np.ndarray) -> np.ndarray:
    """Circular 1 AU ecliptic orbit, longitude k*t (CFG 1; used for all configs)."""
    lon = GAUSS_K * np.asarray(t, dtype=np.float64)
    return np.stack([np.cos(lon), np.sin(lon), np.zeros_like(lon)], axis=-1)


def variance_scalars(cfg: Config) -> np.ndarray:
    lo, hi = cfg.var_range
    if lo == hi:
        return np.full(cfg.n_exp, lo, dtype=np.float64)
    u = rng.uniform_np(cfg.seed, rng.STREAM_VAR, np.arange(cfg.n_exp))
    return lo + (hi - lo) * u


def _ecl_to_radec(lon, lat):
    v = np.stack([np.cos(lat) * np.cos(lon), np.cos(lat) * np.sin(lon), np.sin(lat)], axis=-1)
    ce, se = math.cos(OBLIQUITY), math.sin(OBLIQUITY)
    x, y, z = v[..., 0], v[..., 1] * ce - v[..., 2] * se, v[..., 1] * se + v[..., 2] * ce
    return np.mod(np.arctan2(y, x), 2.0 * math.pi), np.arcsin(np.clip(z, -1.0, 1.0))


def tangent_points(cfg: Config, t: np.ndarray, tracked_radec: Optional[np.ndarray] = None):
    """(ra0, dec0) per exposure.  'track'/'guides' need tracked_radec[N][2]: the apparent (ra, dec)
    of the orbit exposure j follows, at t_j (from a project_fn)."""
    j = np.arange(cfg.n_exp)
    if cfg.tangent_mode in ("track", "guides"):
        if tracked_radec is None:
            raise ValueError("config %r needs tracked_radec (pass a project_fn)" % cfg.name)
        dx = (rng.uniform_np(cfg.seed, rng.STREAM_DITHER_X, j) - 0.5) * (cfg.width / 2.0)
        dy = (rng.uniform_np(cfg.seed, rng.STREAM_DITHER_Y, j) - 0.5) * (cfg.height / 2.0)
        ra, dec = tracked_radec[:, 0], tracked_radec[:, 1]
        return np.mod(ra + dx * PIXEL_SCALE / np.cos(dec), 2.0 * math.pi), dec + dy * PIXEL_SCALE
    h = cfg.tangent_half_deg * DEG
    if cfg.tangent_mode == "opposition":
        lon = GAUSS_K * t + (2.0 * rng.uniform_np(cfg.seed, rng.STREAM_TAN_LON, j) - 1.0) * h
    elif cfg.tangent_mode == "band":
        lon = 2.0 * math.pi * rng.uniform_np(cfg.seed, rng.STREAM_TAN_LON, j)
    else:
        raise ValueError(cfg.tangent_mode)
    lat = (2.0 * rng.uniform_np(cfg.seed, rng.STREAM_TAN_LAT, j) - 1.0) * h
    return _ecl_to_radec(lon, lat)


# ---- candidate orbits -------------------------------------------------------------------------------
_GUIDE_BASE = 1 << 40      # guide orbits are drawn at indices no candidate array reaches


def _box_draw(cfg: Config, k: np.ndarray) -> np.ndarray:
    """(a, e, i, Omega, omega, M0) drawn uniformly over the config box at counter indices k."""
    two_pi = 2.0 * math.pi
    out = np.empty((k.size, 6), dtype=np.float64)
    ua = rng.uniform_np(cfg.seed, rng.STREAM_A, k)
    ue = rng.uniform_np(cfg.seed, rng.STREAM_E, k)
    ui = rng.uniform_np(cfg.seed, rng.STREAM_I, k)
    out[:, 0] = cfg.a_range[0] + (cfg.a_range[1] - cfg.a_range[0]) * ua
    out[:, 1] = cfg.e_range[0] + (cfg.e_range[1] - cfg.e_range[0]) * ue
    out[:, 2] = (cfg.i_range_deg[0] + (cfg.i_range_deg[1] - cfg.i_range_deg[0]) * ui) * DEG
    out[:, 3] = two_pi * rng.uniform_np(cfg.seed, rng.STREAM_NODE, k)
    out[:, 4] = two_pi * rng.uniform_np(cfg.seed, rng.STREAM_PERI, k)
    out[:, 5] = two_pi * rng.uniform_np(cfg.seed, rng.STREAM_M0, k)
    return out


def _diffuse(cfg: Config, k: np.ndarray) -> np.ndarray:
    if cfg.grid is None:
        return _box_draw(cfg, k)
    out = _box_draw(cfg, k)                       # angles Omega, omega, M0 per node
    na, ne, ni = cfg.grid
    ja, je, ji = k // (ne * ni), (k // ni) % ne, k % ni
    out[:, 0] = cfg.a_range[0] + (cfg.a_range[1] - cfg.a_range[0]) / na * ja
    out[:, 1] = cfg.e_range[0] + (cfg.e_range[1] - cfg.e_range[0]) / ne * je
    out[:, 2] = (cfg.i_range_deg[0] + (cfg.i_range_deg[1] - cfg.i_range_deg[0]) / ni * ji) * DEG
    return out


def guide_elements(cfg: Config) -> np.ndarray:
    """Orbits the pointings follow: the injected node (CFG 1 'track') or n_guides seeded draws."""
    if cfg.tangent_mode == "track":
        return _diffuse(cfg, injected_index(cfg)[:1])
    if cfg.tangent_mode == "guides":
        return _box_draw(cfg, _GUIDE_BASE + np.arange(cfg.n_guides, dtype=np.int64))
    return np.zeros((0, 6))


def focus_mask(cfg: Config, k: np.ndarray) -> np.ndarray:
    """True where candidate k belongs to a focused family (pure function of seed and k)."""
    if cfg.focus_fraction <= 0.0:
        return np.zeros(k.shape, dtype=bool)
    return rng.uniform_np(cfg.seed, rng.STREAM_PLACE, 2 * k) < cfg.focus_fraction


def elements(cfg: Config, lo: int = 0, hi: Optional[int] = None) -> np.ndarray:
    """Candidate orbits [hi-lo][6] = (a AU, e, i, Omega, omega, M0) in rad."""
    hi = cfg.n_orbits if hi is None else hi
    k = np.arange(lo, hi, dtype=np.int64)
    out = _diffuse(cfg, k)
    sel = focus_mask(cfg, k)
    if sel.any():
        ks = k[sel]
        guides = guide_elements(cfg)
        g = np.minimum((rng.uniform_np(cfg.seed, rng.STREAM_PLACE, 2 * ks + 1) * cfg.n_guides)
                       .astype(np.int64), cfg.n_guides - 1)
        fam = guides[g].copy()
        for col in range(6):
            u = rng.uniform_np(cfg.seed, rng.STREAM_PLACE + 1 + col, ks)
            fam[:, col] += (2.0 * u - 1.0) * cfg.focus_spread[col]
        fam[:, 1] = np.clip(fam[:, 1], 0.0, 0.99)
        fam[:, 2] = np.abs(fam[:, 2])
        out[sel] = fam
    return out


def injected_index(cfg: Config) -> np.ndarray:
    """Indices (into the candidate array) of the orbits that carry an injected source."""
    if cfg.injected_node is not None:
        na, ne, ni = cfg.grid
        ja, je, ji = cfg.injected_node
        return np.array([(ja * ne + je) * ni + ji], dtype=np.int64)
    n = min(cfg.n_injected, cfg.n_orbits)
    if cfg.focus_fraction <= 0.0:
        return np.arange(n, dtype=np.int64)          # literal: the first n_injected candidates
    # focused: the first n_injected family members (they are the ones that cross exposures)
    found = np.zeros(0, dtype=np.int64)
    lo = 0
    while found.size < n and lo < cfg.n_orbits:
        hi = min(cfg.n_orbits, lo + max(1024, int(4 * n / cfg.focus_fraction)))
        k = np.arange(lo, hi, dtype=np.int64)
        found = np.concatenate([found, k[focus_mask(cfg, k)]])
        lo = hi
    return found[:n]


def injected_amplitudes(cfg: Config) -> np.ndarray:
    n = injected_index(cfg).size
    lo, hi = cfg.amp_range
    u = rng.uniform_np(cfg.seed, rng.STREAM_AMP, np.arange(n))
    return lo + (hi - lo) * u


# ---- images ----------------------------------------------------------------------------------------
def noise_values_np(cfg: Config, j: int, pixel_index) -> np.ndarray:
    """fp32 noise values N(0, v_j) (quantised, see rng.py) at flat pixel indices of exposure j."""
    z = rng.normal_np(cfg.seed, rng.STREAM_NOISE_BASE + j, rng.STREAM_NOISE_BASE2 + j, pixel_index)
    return (z * math.sqrt(float(variance_scalars(cfg)[j]))).astype(np.float32)


def noise_plane_np(cfg: Config, j: int) -> np.ndarray:
    return noise_values_np(cfg, j, np.arange(cfg.plane_pixels)).reshape(cfg.height, cfg.width)


def noise_plane_t(cfg: Config, j: int, device="cpu"):
    """torch version (CPU or CUDA) of noise_plane_np: same bits (see rng.py)."""
    import torch

    k = torch.arange(cfg.plane_pixels, dtype=torch.int64, device=device)
    z = rng.normal_t(cfg.seed, rng.STREAM_NOISE_BASE + j, rng.STREAM_NOISE_BASE2 + j, k)
    z = z * math.sqrt(float(variance_scalars(cfg)[j]))
    return z.to(torch.float32).reshape(cfg.height, cfg.width)


def variance_plane_np(cfg: Config, j: int) -> np.ndarray:
    """fp32 variance plane = the exposure's scalar variance broadcast (A13)."""
    return np.full((cfg.height, cfg.width), variance_scalars(cfg)[j], dtype=np.float32)


# ---- scene ------------------------------------------------------------------------------------------
@dataclass
class Scene:
    cfg: Config
    t0: float
    t: np.ndarray            # [N] days
    obs_ecl: np.ndarray      # [N][3] AU, heliocentric ecliptic
    ra0: np.ndarray          # [N] rad
    dec0: np.ndarray         # [N] rad
    var_scalar: np.ndarray   # [N]
    inj_index: np.ndarray    # [n_inj] candidate indices carrying a source
    inj_amp: np.ndarray      # [n_inj] amplitude in units of sigma_j
    inj_pix: Optional[np.ndarray] = None     # [n_inj][N][2] (ix, iy) or (-1, -1); from project_fn

    # constants travel with the scene so both sides read the same numbers
    pixel_scale: float = PIXEL_SCALE
    gm: float = GM_SUN
    c: float = C_AU_PER_DAY
    obliquity: float = OBLIQUITY

    def elements(self, lo: int = 0, hi: Optional[int] = None) -> np.ndarray:
        return elements(self.cfg, lo, hi)

    def injection_list(self, j: int):
        """(flat pixel index, added value) pairs for exposure j."""
        if self.inj_pix is None or self.inj_index.size == 0:
            return np.zeros(0, np.int64), np.zeros(0, np.float32)
        ix, iy = self.inj_pix[:, j, 0], self.inj_pix[:, j, 1]
        ok = ix >= 0
        add = (self.inj_amp[ok] * math.sqrt(float(self.var_scalar[j]))).astype(np.float32)
        return (iy[ok].astype(np.int64) * self.cfg.width + ix[ok].astype(np.int64)), add

    def flux_plane_np(self, j: int) -> np.ndarray:
        p = noise_plane_np(self.cfg, j)
        idx, add = self.injection_list(j)
        if idx.size:
            np.add.at(p.reshape(-1), idx, add)   # fp32 adds, in list order
        return p

    def flux_plane_t(self, j: int, device="cpu"):
        import torch

        p = noise_plane_t(self.cfg, j, device)
        idx, add = self.injection_list(j)
        if idx.size:
            flat = p.reshape(-1)
            uniq, first = np.unique(idx, return_index=True)
            if uniq.size == idx.size:            # no pixel hit twice: one vectorised fp32 add
                flat[torch.as_tensor(idx, device=flat.device)] += torch.as_tensor(add, device=flat.device)
            else:                                # sequential fp32 adds, same order as numpy path
                for k in range(idx.size):
                    flat[int(idx[k])] += float(add[k])
        return p

    def flux_values_np(self, j: int, pixel_index) -> np.ndarray:
        """Flux at selected flat pixel indices of exposure j without building the plane."""
        pixel_index = np.asarray(pixel_index, dtype=np.int64)
        v = noise_values_np(self.cfg, j, pixel_index)
        idx, add = self.injection_list(j)
        for k in range(idx.size):
            v[pixel_index == idx[k]] += add[k]
        return v

    def var_plane_np(self, j: int) -> np.ndarray:
        return variance_plane_np(self.cfg, j)


ProjectFn = Callable[["Scene", np.ndarray, float], Tuple[np.ndarray, np.ndarray]]


def build_scene(cfg: Config, project_fn: Optional[ProjectFn] = None, t0: float = 0.0,
                inject: bool = True) -> Scene:
    """Assemble exposure metadata; with a project_fn also tangent tracking and source injection.

    project_fn(scene, elements[n][6], t0) -> (radec[n][N][2], pix[n][N][2] int, (-1,-1) = culled).
    """
    t = exposure_times(cfg)
    obs = observer_ecliptic(t)
    scene = Scene(cfg, t0, t, obs, np.zeros(cfg.n_exp), np.zeros(cfg.n_exp), variance_scalars(cfg),
                  injected_index(cfg), injected_amplitudes(cfg))
    if cfg.tangent_mode in ("track", "guides"):
        if project_fn is None:
            raise ValueError("config %r needs a project_fn" % cfg.name)
        guides = guide_elements(cfg)
        radec, _ = project_fn(scene, guides, t0)            # tangent-independent sky positions
        j = np.arange(cfg.n_exp)
        scene.ra0, scene.dec0 = tangent_points(cfg, t, np.asarray(radec)[j % guides.shape[0], j])
    else:
        scene.ra0, scene.dec0 = tangent_points(cfg, t)
    if inject and project_fn is not None and scene.inj_index.size:
        inj_el = np.concatenate([elements(cfg, int(k), int(k) + 1) for k in scene.inj_index]) \
            if scene.inj_index.size < 4096 else elements(cfg)[scene.inj_index]
        _, pix = project_fn(scene, inj_el, t0)
        scene.inj_pix = np.asarray(pix, dtype=np.int32)
    return scene
