"""Seeded synthetic workloads C1..C5 (BASELINE.json `configs`, recipe in SURVEY.md section 8(d)
and DESIGN.md "Input recipe").

The paper's own inputs (an 850M-particle cosmological run and its 1M/10M/100M subsets, the
small/medium/large sets of Table 2, the Millennium II snapshot: PAPER.md:138, :171, :184) are
not available; these generators stand in for them with the same SoA layout
and a comparable spread of screen footprints.

This module produces INPUTS only (particle arrays, colour tables, camera, parameters).  It
contains none of the renderer's arithmetic and is imported by both the oracle-side and the
CUDA-side tests and by bench.py.  Everything is a pure function of (config, n, seed): the
arrays are generated in chunks on a thread pool and are bit-identical however they are
chunked.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, field
from typing import Callable, Dict, List, Optional

import numpy as np

from . import rng

ADDITIVE = 0
ABSORB = 1

# stream ids (per-particle streams < 100, per-halo streams >= 100)
_S_NX, _S_NY, _S_NZ = 0, 2, 4          # normals use two streams each
_S_BX, _S_BY, _S_BZ = 6, 7, 8          # background position
_S_R = 10                               # log-normal smoothing length (10, 11)
_S_I, _S_COL, _S_TYPE = 12, 13, 14
_S_RAD, _S_CT, _S_PHI = 15, 16, 17     # NFW radius, cos(theta), phi
_H_CX, _H_CY, _H_CZ, _H_SCALE = 100, 101, 102, 103
_H_MASS = 104
_G_A, _G_B, _G_T = 110, 113, 116       # segment end points (3 streams each), position on segment

_NFW_C = 5.0                            # truncation radius in units of r_s
_CHUNK = 1 << 20


@dataclass
class Camera:
    eye: tuple
    lookat: tuple
    up: tuple
    fov_deg: float
    width: int
    height: int


@dataclass
class Workload:
    name: str
    n: int
    seed: int
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    r: np.ndarray
    I: np.ndarray
    colval: np.ndarray
    type: Optional[np.ndarray]           # uint8 or None
    cameras: List[Camera]
    lut_e: np.ndarray                    # (n_types, n_entries, 3) float32
    lut_a: Optional[np.ndarray]          # same shape, absorb mode only
    brightness: List[float]
    abs_brightness: List[float]
    mode: int
    support_f: float = 3.0
    z_near: float = 0.01
    notes: Dict[str, object] = field(default_factory=dict)
    vec: Optional[np.ndarray] = None     # (n, 3) float32: vector colouring, replaces colval + tables

    @property
    def camera(self) -> Camera:
        return self.cameras[0]

    @property
    def bytes_per_particle(self) -> int:
        return 24 + (1 if self.type is not None else 0)

    def subsample(self, stride: int, offset: int = 0) -> "Workload":
        """Every `stride`-th particle (a strided subsample keeps the footprint mix)."""
        sl = slice(offset, None, stride)
        t = None if self.type is None else np.ascontiguousarray(self.type[sl])
        arr = [np.ascontiguousarray(a[sl]) for a in (self.x, self.y, self.z, self.r, self.I, self.colval)]
        return Workload(self.name + f"/stride{stride}", len(arr[0]), self.seed, *arr, t, self.cameras,
                        self.lut_e, self.lut_a, list(self.brightness), list(self.abs_brightness),
                        self.mode, self.support_f, self.z_near, dict(self.notes),
                        None if self.vec is None else np.ascontiguousarray(self.vec[sl]))

    def checksums(self) -> Dict[str, int]:
        out = {}
        for k in ("x", "y", "z", "r", "I", "colval", "type"):
            a = getattr(self, k)
            if a is not None:
                v = a.view(np.uint8 if a.dtype == np.uint8 else np.uint32)
                out[k] = int(np.bitwise_xor.reduce(v.astype(np.uint64) * np.uint64(0x9E3779B1) +
                                                   np.arange(v.size, dtype=np.uint64)))
        return out


# ----------------------------------------------------------------------------------------------
# colour tables (inputs, "colour look-up table or palette ... external file")
# ----------------------------------------------------------------------------------------------
def lut_hot(n_entries: int = 256) -> np.ndarray:
    v = np.linspace(0.0, 1.0, n_entries)
    t = np.stack([np.clip(3 * v, 0, 1), np.clip(3 * v - 1, 0, 1), np.clip(3 * v - 2, 0, 1)], axis=1)
    return t.astype(np.float32)


def lut_hot_swapped(n_entries: int = 256) -> np.ndarray:
    return np.ascontiguousarray(lut_hot(n_entries)[:, ::-1])


def lut_absorb(n_entries: int = 256) -> np.ndarray:
    v = np.linspace(0.0, 1.0, n_entries)
    return ((0.2 + 0.8 * v)[:, None] * np.array([1.0, 0.8, 0.6])[None, :]).astype(np.float32)


# ----------------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------------
def _n_threads() -> int:
    return max(1, min(32, os.cpu_count() or 1))


def _run_chunks(n: int, fill: Callable[[int, int], None]) -> None:
    bounds = [(s, min(s + _CHUNK, n)) for s in range(0, n, _CHUNK)]
    if len(bounds) <= 1:
        for s, e in bounds:
            fill(s, e)
        return
    with ThreadPoolExecutor(_n_threads()) as ex:
        list(ex.map(lambda b: fill(*b), bounds))


def _nfw_m(x):
    return np.log1p(x) - x / (1.0 + x)


_NFW_K = 8192
_NFW_X = _NFW_C * (np.arange(_NFW_K + 1) / _NFW_K) ** 2
_NFW_M = _nfw_m(_NFW_X)


def _nfw_radius(u: np.ndarray) -> np.ndarray:
    """x = rad / r_s with enclosed-mass CDF m(x)/m(c) (tabulated inverse, x in [0, c])."""
    return np.interp(u * _NFW_M[-1], _NFW_M, _NFW_X)


def _alloc(n: int, with_type: bool):
    a = {k: np.empty(n, np.float32) for k in ("x", "y", "z", "r", "I", "colval")}
    a["type"] = np.empty(n, np.uint8) if with_type else None
    return a


def _fill_common(a, seed, idx, s, e, with_type):
    a["I"][s:e] = (0.5 + 0.5 * rng.uniform(seed, _S_I, idx)).astype(np.float32)
    a["colval"][s:e] = rng.uniform(seed, _S_COL, idx).astype(np.float32)
    if with_type:
        a["type"][s:e] = (rng.uniform(seed, _S_TYPE, idx) >= 0.5).astype(np.uint8)


def _lognormal_r(seed, idx, median, sigma_ln):
    return median * np.exp(sigma_ln * rng.normal(seed, _S_R, idx))


def _iso_dir(seed, idx):
    ct = 2.0 * rng.uniform(seed, _S_CT, idx) - 1.0
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * np.pi * rng.uniform(seed, _S_PHI, idx)
    return st * np.cos(ph), st * np.sin(ph), ct


def _halo_uniform(seed, stream, n_halos, lo, hi):
    return lo + (hi - lo) * rng.uniform(seed, stream, rng.index_range(0, n_halos))


def _halo_loguniform(seed, stream, n_halos, lo, hi):
    return lo * (hi / lo) ** rng.uniform(seed, stream, rng.index_range(0, n_halos))


def _default_camera(w, h):
    return Camera((0.5, 0.5, -1.5), (0.5, 0.5, 0.5), (0.0, 1.0, 0.0), 30.0, w, h)


# brightness literals: written by oracle/calibrate_brightness.py (frame-mean of raw S = 1,
# closed-form flux of each visible splat).  Keyed by config name.
_BRIGHTNESS = {
    "C1": 1.0,
    "C2": 1.0,
    "C3": 1.0,
    "C4": 1.0,
    "C5": 1.0,
}
try:  # the calibration table lives beside this file so the script can rewrite it
    from .brightness_table import BRIGHTNESS as _TABLE
    _BRIGHTNESS.update(_TABLE)
except ImportError:  # pragma: no cover - table not generated yet
    pass


def _brightness_for(name: str, n: int, n_full: int) -> float:
    # amplitude per particle is independent of n, so the frame mean scales like n: keep mean S ~ 1
    return float(_BRIGHTNESS[name]) * (n_full / float(n))


# ----------------------------------------------------------------------------------------------
# C1: 8 Gaussian halos + 20 % uniform, log-normal r
# ----------------------------------------------------------------------------------------------
def make_c1(n: int = 100_000, seed: int = 1004130201, width: int = 256, height: int = 256) -> Workload:
    n_halos = 8
    n_h = (n * 8) // 10
    cx = _halo_uniform(seed, _H_CX, n_halos, 0.2, 0.8)
    cy = _halo_uniform(seed, _H_CY, n_halos, 0.2, 0.8)
    cz = _halo_uniform(seed, _H_CZ, n_halos, 0.2, 0.8)
    sg = _halo_loguniform(seed, _H_SCALE, n_halos, 0.02, 0.1)
    a = _alloc(n, False)

    def fill(s, e):
        idx = rng.index_range(s, e)
        halo = np.minimum((idx * np.uint64(n_halos)) // np.uint64(max(n_h, 1)), n_halos - 1).astype(np.int64)
        is_h = idx < np.uint64(n_h)
        hx = cx[halo] + sg[halo] * rng.normal(seed, _S_NX, idx)
        hy = cy[halo] + sg[halo] * rng.normal(seed, _S_NY, idx)
        hz = cz[halo] + sg[halo] * rng.normal(seed, _S_NZ, idx)
        a["x"][s:e] = np.where(is_h, hx, rng.uniform(seed, _S_BX, idx)).astype(np.float32)
        a["y"][s:e] = np.where(is_h, hy, rng.uniform(seed, _S_BY, idx)).astype(np.float32)
        a["z"][s:e] = np.where(is_h, hz, rng.uniform(seed, _S_BZ, idx)).astype(np.float32)
        a["r"][s:e] = _lognormal_r(seed, idx, 0.005, 0.5).astype(np.float32)
        _fill_common(a, seed, idx, s, e, False)

    _run_chunks(n, fill)
    b = _brightness_for("C1", n, 100_000)
    return Workload("C1", n, seed, a["x"], a["y"], a["z"], a["r"], a["I"], a["colval"], None,
                    [_default_camera(width, height)], lut_hot()[None], None, [b], [b], ADDITIVE)


# ----------------------------------------------------------------------------------------------
# C2 / C4: NFW halos + 10 % uniform, r from the local analytic density
# ----------------------------------------------------------------------------------------------
def _nfw_fill(a, seed, s, e, n, n_h, n_halos, cx, cy, cz, rs, halo_of, count_of, r_rule):
    idx = rng.index_range(s, e)
    is_h = idx < np.uint64(n_h)
    halo = halo_of(idx)
    xr = _nfw_radius(rng.uniform(seed, _S_RAD, idx))
    dx, dy, dz = _iso_dir(seed, idx)
    rad = xr * rs[halo]
    a["x"][s:e] = np.where(is_h, cx[halo] + rad * dx, rng.uniform(seed, _S_BX, idx)).astype(np.float32)
    a["y"][s:e] = np.where(is_h, cy[halo] + rad * dy, rng.uniform(seed, _S_BY, idx)).astype(np.float32)
    a["z"][s:e] = np.where(is_h, cz[halo] + rad * dz, rng.uniform(seed, _S_BZ, idx)).astype(np.float32)
    a["r"][s:e] = r_rule(idx, is_h, halo, xr).astype(np.float32)


def _density_r(k, n, rs, count_of):
    """r = clip(k * delta^(-1/3)), delta = analytic NFW number density / mean box density (n)."""
    lo, hi = 1e-4 * k / 0.01, 0.05 * k / 0.01
    mc = _nfw_m(_NFW_C)

    def rule(idx, is_h, halo, xr):
        xf = np.maximum(xr, 1e-3)
        dens = count_of[halo] / (4.0 * np.pi * rs[halo] ** 3 * mc) / (xf * (1.0 + xf) ** 2)
        delta = np.where(is_h, dens / float(n), 0.1)
        return np.clip(k * delta ** (-1.0 / 3.0), lo, hi)

    return rule


def make_c2(n: int = 16_000_000, seed: int = 1004130202, width: int = 1024, height: int = 1024,
            n_halos: int = 512, name: str = "C2") -> Workload:
    n_h = (n * 9) // 10
    cx = _halo_uniform(seed, _H_CX, n_halos, 0.1, 0.9)
    cy = _halo_uniform(seed, _H_CY, n_halos, 0.1, 0.9)
    cz = _halo_uniform(seed, _H_CZ, n_halos, 0.1, 0.9)
    rs = _halo_loguniform(seed, _H_SCALE, n_halos, 0.005, 0.05)
    count_of = np.full(n_halos, n_h / float(n_halos))
    a = _alloc(n, False)

    def halo_of(idx):
        return np.minimum((idx * np.uint64(n_halos)) // np.uint64(max(n_h, 1)), n_halos - 1).astype(np.int64)

    rule = _density_r(0.01, n, rs, count_of)

    def fill(s, e):
        _nfw_fill(a, seed, s, e, n, n_h, n_halos, cx, cy, cz, rs, halo_of, count_of, rule)
        _fill_common(a, seed, rng.index_range(s, e), s, e, False)

    _run_chunks(n, fill)
    b = _brightness_for(name, n, 16_000_000)
    return Workload(name, n, seed, a["x"], a["y"], a["z"], a["r"], a["I"], a["colval"], None,
                    [_default_camera(width, height)], lut_hot()[None], None, [b], [b], ADDITIVE)


def make_c4(n: int = 16_000_000, seed: int = 1004130202, width: int = 1024, height: int = 1024,
            n_halos: int = 512) -> Workload:
    w = make_c2(n, seed, width, height, n_halos, name="C4")
    w.cameras = [Camera((0.5, 0.5, 0.3), (0.5, 0.5, 0.5), (0.0, 1.0, 0.0), 60.0, width, height)]
    w.lut_a = lut_absorb()[None]
    w.mode = ABSORB
    return w


# ----------------------------------------------------------------------------------------------
# C3: NFW halos strung along filaments, heavy-tailed log-normal r, two particle types
# ----------------------------------------------------------------------------------------------
def make_c3(n: int = 100_000_000, seed: int = 1004130203, width: int = 2048, height: int = 2048,
            n_halos: int = 4096, n_segments: int = 256, r_median: float = 0.005) -> Workload:
    seg = rng.index_range(0, n_segments)
    ends_a = [rng.uniform(seed, _G_A + k, seg) for k in range(3)]
    ends_b = [rng.uniform(seed, _G_B + k, seg) for k in range(3)]
    hh = np.arange(n_halos)
    t = rng.uniform(seed, _G_T, rng.index_range(0, n_halos))
    sidx = hh % n_segments
    cx, cy, cz = [ends_a[k][sidx] + t * (ends_b[k][sidx] - ends_a[k][sidx]) for k in range(3)]
    rs = _halo_loguniform(seed, _H_SCALE, n_halos, 0.005, 0.05)
    count_of = np.full(n_halos, n / float(n_halos))
    a = _alloc(n, True)

    def halo_of(idx):
        return np.minimum((idx * np.uint64(n_halos)) // np.uint64(max(n, 1)), n_halos - 1).astype(np.int64)

    def rule(idx, is_h, halo, xr):
        return _lognormal_r(seed, idx, r_median, 1.0)

    def fill(s, e):
        _nfw_fill(a, seed, s, e, n, n, n_halos, cx, cy, cz, rs, halo_of, count_of, rule)
        _fill_common(a, seed, rng.index_range(s, e), s, e, True)

    _run_chunks(n, fill)
    b = _brightness_for("C3", n, 100_000_000)
    lut = np.stack([lut_hot(), lut_hot_swapped()])
    return Workload("C3", n, seed, a["x"], a["y"], a["z"], a["r"], a["I"], a["colval"], a["type"],
                    [_default_camera(width, height)], lut, None, [b, 0.5 * b], [b, 0.5 * b], ADDITIVE)


# ----------------------------------------------------------------------------------------------
# C5: power-law halo mass function + 10 % uniform, 8-camera orbit
# ----------------------------------------------------------------------------------------------
def make_c5(n: int = 400_000_000, seed: int = 1004130205, width: int = 4096, height: int = 4096,
            n_halos: int = 65536) -> Workload:
    hidx = rng.index_range(0, n_halos)
    u = rng.uniform(seed, _H_MASS, hidx)
    mass = (1.0 - u * (1.0 - (1e5) ** (-0.9))) ** (-1.0 / 0.9)
    wfrac = 0.9 * mass / mass.sum()
    n_h = (n * 9) // 10
    cum = np.floor(np.cumsum(wfrac) / 0.9 * n_h + 0.5).astype(np.int64)
    cum[-1] = n_h
    starts = np.concatenate([[0], cum[:-1]])
    count_of = np.maximum(cum - starts, 0).astype(np.float64)
    rvir = (3.0 * wfrac / (4.0 * np.pi * 200.0)) ** (1.0 / 3.0)
    rs = rvir / _NFW_C
    cx = _halo_uniform(seed, _H_CX, n_halos, 0.05, 0.95)
    cy = _halo_uniform(seed, _H_CY, n_halos, 0.05, 0.95)
    cz = _halo_uniform(seed, _H_CZ, n_halos, 0.05, 0.95)
    a = _alloc(n, False)
    k = 0.01 * (1.6e7 / n) ** (1.0 / 3.0)

    def halo_of(idx):
        return np.minimum(np.searchsorted(cum, idx.astype(np.int64), side="right"), n_halos - 1)

    rule = _density_r(k, n, rs, np.maximum(count_of, 1.0))

    def fill(s, e):
        _nfw_fill(a, seed, s, e, n, n_h, n_halos, cx, cy, cz, rs, halo_of, count_of, rule)
        _fill_common(a, seed, rng.index_range(s, e), s, e, False)

    _run_chunks(n, fill)
    cams = []
    for j in range(8):
        th = np.deg2rad(45.0 * j)
        eye = (0.5 + 2.0 * np.sin(th), 0.5, 0.5 - 2.0 * np.cos(th))
        cams.append(Camera(tuple(float(v) for v in eye), (0.5, 0.5, 0.5), (0.0, 1.0, 0.0), 30.0, width, height))
    b = _brightness_for("C5", n, 400_000_000)
    return Workload("C5", n, seed, a["x"], a["y"], a["z"], a["r"], a["I"], a["colval"], None,
                    cams, lut_hot()[None], None, [b], [b], ADDITIVE)


MAKERS = {"C1": make_c1, "C2": make_c2, "C3": make_c3, "C4": make_c4, "C5": make_c5}
FULL_N = {"C1": 100_000, "C2": 16_000_000, "C3": 100_000_000, "C4": 16_000_000, "C5": 400_000_000}


def make(name: str, n: Optional[int] = None, **kw) -> Workload:
    """Build config `name`; `n` below the full size gives a scaled-down copy of the same
    generator (same halos, fewer particles each, brightness rescaled to keep mean S ~ 1)."""
    return MAKERS[name](n if n is not None else FULL_N[name], **kw)
