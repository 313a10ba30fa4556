"""Python face of the CPU oracle (TEST INFRASTRUCTURE, not the product).

Builds oracle/splotch_oracle.c with gcc on first use and wraps its entry points with numpy
arrays.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs import this package; nothing under paper_1004_1302_b200/ does, and this package imports
nothing from there.  See the header of splotch_oracle.c for what each function follows in the
paper and how it is pinned.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "splotch_oracle.c")
# ORACLE_SANITIZE=1 builds a second library with AddressSanitizer + UndefinedBehaviorSanitizer;
# run the pins under it with
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 ORACLE_SANITIZE=1 \
#       python -m pytest tests/test_oracle_pins.py tests/test_oracle_canonical.py -q
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") == "1"
_LIB = os.path.join(_HERE, "libsplotch_oracle_asan.so" if _SANITIZE else "libsplotch_oracle.so")
_lib = None

ADDITIVE, ABSORB = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle.  -ffp-contract=off keeps the canonical fp32 sequence unfused."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"] if _SANITIZE else ["-O2"]
        cmd = ["gcc", *opt, "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared",
               "-fPIC", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_depth_order.restype = C.c_int64
    return _lib


def _p(a: Optional[np.ndarray], t):
    return None if a is None else a.ctypes.data_as(C.POINTER(t))


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def cam_array(camera) -> np.ndarray:
    """eye(3), lookat(3), up(3), fov_deg as the float32 values the C ABI receives."""
    return np.array(list(camera.eye) + list(camera.lookat) + list(camera.up) + [camera.fov_deg], np.float32)


def camera_basis(camera) -> Tuple[np.ndarray, np.ndarray, np.ndarray, float]:
    right, upv, fwd = (np.zeros(3) for _ in range(3))
    F = C.c_double(0)
    rc = _load().orc_camera_basis(_p(cam_array(camera), C.c_float), C.c_int32(camera.width), C.c_int32(camera.height),
                                  _p(right, C.c_double), _p(upv, C.c_double), _p(fwd, C.c_double), C.byref(F))
    if rc:
        raise ValueError(f"orc_camera_basis: {rc}")
    return right, upv, fwd, F.value


def _particles(w):
    x, y, z, r, I, cv = (_f32(getattr(w, k)) for k in ("x", "y", "z", "r", "I", "colval"))
    t = None if w.type is None else np.ascontiguousarray(w.type, dtype=np.uint8)
    return x, y, z, r, I, cv, t


def project_f32(w, camera=None):
    """Canonical fp32 projector: dict of sx, sy, ss, R (f32), zkey (u32), bbox (n,4 i32), visible (u8)."""
    camera = camera or w.camera
    x, y, z, r, I, cv, t = _particles(w)
    n = len(x)
    out = dict(sx=np.zeros(n, np.float32), sy=np.zeros(n, np.float32), ss=np.zeros(n, np.float32),
               R=np.zeros(n, np.float32), zkey=np.zeros(n, np.uint32), bbox=np.zeros((n, 4), np.int32),
               visible=np.zeros(n, np.uint8))
    n_types = int(w.lut_e.shape[0])
    rc = _load().orc_project_f32(C.c_int64(n), _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float),
                                 _p(r, C.c_float), _p(I, C.c_float), _p(cv, C.c_float), _p(t, C.c_uint8),
                                 C.c_int32(n_types), _p(cam_array(camera), C.c_float),
                                 C.c_int32(camera.width), C.c_int32(camera.height),
                                 C.c_float(w.support_f), C.c_float(w.z_near),
                                 _p(out["sx"], C.c_float), _p(out["sy"], C.c_float), _p(out["ss"], C.c_float),
                                 _p(out["R"], C.c_float), _p(out["zkey"], C.c_uint32), _p(out["bbox"], C.c_int32),
                                 _p(out["visible"], C.c_uint8))
    if rc:
        raise ValueError(f"orc_project_f32: {rc}")
    return out


def depth_order(zkey: np.ndarray, visible: np.ndarray) -> np.ndarray:
    """Visible particle indices by ascending (zkey, index): nearest first (R11)."""
    n = len(zkey)
    order = np.zeros(max(n, 1), np.int64)
    V = _load().orc_depth_order(C.c_int64(n), _p(np.ascontiguousarray(zkey, np.uint32), C.c_uint32),
                                _p(np.ascontiguousarray(visible, np.uint8), C.c_uint8), _p(order, C.c_int64))
    if V < 0:
        raise MemoryError("orc_depth_order")
    return order[:V].copy()


def bins(bbox: np.ndarray, visible: np.ndarray, width: int, height: int, shift: int = 4,
         order: Optional[np.ndarray] = None, with_members: bool = True):
    """Canonical binner (B-rules).  Returns counts (T,) u32, offsets (T+1,) u64, members (D,) u32."""
    lib = _load()
    n = len(visible)
    bs = 1 << shift
    T = ((width + bs - 1) >> shift) * ((height + bs - 1) >> shift)
    counts = np.zeros(T, np.uint32)
    offsets = np.zeros(T + 1, np.uint64)
    bb = np.ascontiguousarray(bbox, np.int32)
    vis = np.ascontiguousarray(visible, np.uint8)
    od = None if order is None else np.ascontiguousarray(order, np.int64)
    n_od = 0 if od is None else len(od)
    args = (C.c_int64(n), _p(bb, C.c_int32), _p(vis, C.c_uint8), _p(od, C.c_int64), C.c_int64(n_od),
            C.c_int32(shift), C.c_int32(width), C.c_int32(height), _p(counts, C.c_uint32), _p(offsets, C.c_uint64))
    rc = lib.orc_bins(*args, None)
    if rc:
        raise ValueError(f"orc_bins: {rc}")
    members = None
    if with_members:
        members = np.zeros(max(int(offsets[-1]), 1), np.uint32)
        rc = lib.orc_bins(*args, _p(members, C.c_uint32))
        if rc:
            raise ValueError(f"orc_bins: {rc}")
        members = members[: int(offsets[-1])]
    return counts, offsets, members


def _lut_args(w):
    lut_e = _f32(w.lut_e)
    lut_a = None if w.lut_a is None else _f32(w.lut_a)
    n_types, n_entries = int(lut_e.shape[0]), int(lut_e.shape[1])
    br = np.zeros(4, np.float32)
    ab = np.zeros(4, np.float32)
    br[: len(w.brightness)] = w.brightness
    ab[: len(w.abs_brightness)] = w.abs_brightness
    return lut_e, lut_a, n_entries, n_types, br, ab


def splat_table(w, camera=None, mode: Optional[int] = None):
    """Stage 1 in double: (table (n, 11): sx, sy, sigma_s, R, tau0, E rgb, A rgb; ok (n,) u8)."""
    camera = camera or w.camera
    mode = w.mode if mode is None else mode
    x, y, z, r, I, cv, t = _particles(w)
    n = len(x)
    lut_e, lut_a, n_entries, n_types, br, ab = _lut_args(w)
    table = np.zeros((max(n, 1), 11), np.float64)
    ok = np.zeros(max(n, 1), np.uint8)
    rc = _load().orc_splat_table(C.c_int64(n), _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float),
                                 _p(r, C.c_float), _p(I, C.c_float), _p(cv, C.c_float), _p(t, C.c_uint8),
                                 _p(cam_array(camera), C.c_float), C.c_int32(camera.width), C.c_int32(camera.height),
                                 _p(lut_e, C.c_float), _p(lut_a, C.c_float), C.c_int32(n_entries), C.c_int32(n_types),
                                 _p(br, C.c_float), _p(ab, C.c_float), C.c_int32(mode), C.c_float(w.support_f),
                                 C.c_float(w.z_near), _p(table, C.c_double), _p(ok, C.c_uint8))
    if rc:
        raise ValueError(f"orc_splat_table: {rc}")
    return table[:n], ok[:n]


def render_table(table: np.ndarray, seq: np.ndarray, mode: int, roi: Sequence[int], raw: bool = False) -> np.ndarray:
    """Stage 2 on an explicit splat table and visiting sequence (nearest first in absorb mode)."""
    roi_a = np.array(roi, np.int32)
    rw, rh = int(roi_a[2] - roi_a[0]), int(roi_a[3] - roi_a[1])
    out = np.zeros((rh, rw, 3), np.float64)
    tb = np.ascontiguousarray(table, np.float64)
    sq = np.ascontiguousarray(seq, np.int64)
    rc = _load().orc_render_table(_p(tb, C.c_double), _p(sq, C.c_int64), C.c_int64(len(sq)), C.c_int32(mode),
                                  C.c_int32(1 if raw else 0), _p(roi_a, C.c_int32), _p(out, C.c_double), None)
    if rc:
        raise ValueError(f"orc_render_table: {rc}")
    return out


def render(w, camera=None, mode: Optional[int] = None, roi: Optional[Sequence[int]] = None,
           raw: bool = False, return_threads: bool = False):
    """The whole path.  roi = (x0, y0, x1, y1) pixel rectangle (default: full frame).
    Returns float64 (rows, cols, 3), row 0 = top."""
    camera = camera or w.camera
    mode = w.mode if mode is None else mode
    x, y, z, r, I, cv, t = _particles(w)
    n = len(x)
    lut_e, lut_a, n_entries, n_types, br, ab = _lut_args(w)
    if roi is None:
        roi = (0, 0, camera.width, camera.height)
    roi_a = np.array(roi, np.int32)
    rw, rh = int(roi_a[2] - roi_a[0]), int(roi_a[3] - roi_a[1])
    out = np.zeros((rh, rw, 3), np.float64)
    nth = C.c_int32(0)
    rc = _load().orc_render(C.c_int64(n), _p(x, C.c_float), _p(y, C.c_float), _p(z, C.c_float), _p(r, C.c_float),
                            _p(I, C.c_float), _p(cv, C.c_float), _p(t, C.c_uint8), _p(cam_array(camera), C.c_float),
                            C.c_int32(camera.width), C.c_int32(camera.height), _p(lut_e, C.c_float),
                            _p(lut_a, C.c_float), C.c_int32(n_entries), C.c_int32(n_types), _p(br, C.c_float),
                            _p(ab, C.c_float), C.c_int32(mode), C.c_float(w.support_f), C.c_float(w.z_near),
                            C.c_int32(1 if raw else 0), _p(roi_a, C.c_int32), _p(out, C.c_double), C.byref(nth))
    if rc:
        raise ValueError(f"orc_render: {rc}")
    return (out, int(nth.value)) if return_threads else out


def render_vector(w, camera=None, mode: Optional[int] = None, roi: Optional[Sequence[int]] = None, raw: bool = False):
    """Vector colouring ("the three components of the vectors can be mapped to the three components of
    E and A"; reading R19): E_p = brightness[type] * v_p, A_p = abs_brightness[type] * v_p with v_p = w.vec[p] used as
    given; a particle with a non-finite component is culled.  Stage 1 is the pinned splat table evaluated with colour
    tables that are identically one (so that its E / A columns hold the brightness of the particle's type), scaled here
    by the vector in float64; stage 2 is render_table."""
    camera = camera or w.camera
    mode = w.mode if mode is None else mode
    vec = np.asarray(w.vec, np.float64)
    ones = np.ones((int(w.lut_e.shape[0]), 2, 3), np.float32)
    import copy
    w1 = copy.copy(w)
    w1.lut_e, w1.lut_a = ones, ones
    w1.colval = np.zeros(len(vec), np.float32)
    table, ok = splat_table(w1, camera, mode)
    fin = np.isfinite(vec).all(axis=1)
    table = table.copy()
    table[:, 5:8] *= np.where(fin[:, None], vec, 0.0)
    table[:, 8:11] *= np.where(fin[:, None], vec, 0.0)
    ok = ok.astype(bool) & fin
    if mode == 0:
        seq = np.nonzero(ok)[0]
    else:
        p = project_f32(w1, camera)
        seq = depth_order(p["zkey"], (p["visible"].astype(bool) & fin).astype(np.uint8))
    if roi is None:
        roi = (0, 0, camera.width, camera.height)
    return render_table(table, seq, mode, roi, raw)


def normalize_field(values, log_scale: bool = False):
    """Stage (b) of the paper's pipeline, "process data (e.g. for normalization)", reading R17
    of DESIGN.md, written out in float64: f = identity or log10; lo / hi = min / max of f over the values where f
    is defined and finite; out = clamp((f - lo) / (hi - lo), 0, 1), NaN where f is undefined, 0 when hi == lo.
    Returns (out, (lo, hi)); (lo, hi) = (0, 0) when no value is in the domain."""
    v = np.asarray(values, np.float64)
    ok = np.isfinite(v)
    if log_scale:
        ok &= v > 0
    f = np.full(v.shape, np.nan)
    f[ok] = np.log10(v[ok]) if log_scale else v[ok]
    if not ok.any():
        return f, (0.0, 0.0)
    lo, hi = float(f[ok].min()), float(f[ok].max())
    out = np.full(v.shape, np.nan)
    out[ok] = 0.0 if hi == lo else np.clip((f[ok] - lo) / (hi - lo), 0.0, 1.0)
    return out, (lo, hi)


def tonemap_rgb8(values, gamma: float = 1.0):
    """Reading R18: 8-bit code rint(255 * clamp(x, 0, 1)^(1/gamma)), NaN -> 0.  The integer is decided in fp32
    (the kernel's precision): clamp, power and the product by 255 are float32 operations, rint is round-half-even."""
    x = np.asarray(values, np.float32)
    y = np.where(np.isnan(x), np.float32(0), np.clip(x, np.float32(0), np.float32(1))).astype(np.float32)
    if gamma != 1.0:
        y = np.power(y, np.float32(1.0) / np.float32(gamma), dtype=np.float32)
    return np.rint(np.float32(255.0) * y).astype(np.uint8)


def max_threads() -> int:
    return int(_load().orc_max_threads())
