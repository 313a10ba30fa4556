"""Small hand-made workloads for the pins (inputs only; no rendering arithmetic here)."""
import numpy as np

from workloads import ADDITIVE, Camera, Workload


def const_lut(rgb=(1.0, 1.0, 1.0), n_entries=2, n_types=1):
    return np.tile(np.asarray(rgb, np.float32)[None, None, :], (n_types, n_entries, 1)).copy()


def mk(points, camera, lut_e=None, lut_a=None, brightness=(1.0,), abs_brightness=None, mode=ADDITIVE,
       support_f=3.0, z_near=0.01, types=None):
    """points: rows of (x, y, z, r, I, colval)."""
    p = np.asarray(points, np.float64).reshape(-1, 6)
    cols = [np.ascontiguousarray(p[:, k], np.float32) for k in range(6)]
    lut_e = const_lut() if lut_e is None else np.asarray(lut_e, np.float32)
    if lut_e.ndim == 2:
        lut_e = lut_e[None]
    if lut_a is not None:
        lut_a = np.asarray(lut_a, np.float32)
        if lut_a.ndim == 2:
            lut_a = lut_a[None]
    t = None if types is None else np.asarray(types, np.uint8)
    ab = list(brightness if abs_brightness is None else abs_brightness)
    return Workload("hand", len(p), 0, *cols, t, [camera], lut_e, lut_a, list(brightness), ab, mode,
                    support_f, z_near)


def cam(eye=(0.0, 0.0, -10.0), lookat=(0.0, 0.0, 0.0), up=(0.0, 1.0, 0.0), fov=20.0, w=64, h=64):
    return Camera(tuple(eye), tuple(lookat), tuple(up), float(fov), int(w), int(h))
