"""Writes workloads/brightness_table.py: the brightness literal of every config.

SURVEY.md 8(d): "brightness chosen by the harness so that the frame-mean of raw S (channel
average) is 1.0, from the closed-form flux sum of P3".  The flux of a visible splat is
a_c pi sigma_s^2 (1 - exp(-f^2)) (pin P2); the part of it that lands inside the frame is
estimated by the fraction of the splat's bounding square that overlaps the frame.  This is an
INPUT calibration (it only has to put S at order one), so the estimate need not be exact.

Calls only oracle/ and workloads/ (never the CUDA path).  Run once:
    python -m oracle.calibrate_brightness            # C1, C2, C3, C4, C5
The big configs are calibrated on a strided subsample of the full-size arrays.
"""
from __future__ import annotations

import os
import sys

import numpy as np

import oracle
import workloads
from workloads import configs as cfg

STRIDE = {"C1": 1, "C2": 4, "C3": 16, "C4": 4, "C5": 32}


def frame_mean_S(w, cam) -> float:
    """Closed-form frame mean of raw S (channel average) at the workload's current brightness."""
    tab, ok = oracle.splat_table(w, cam, mode=workloads.ADDITIVE)
    t = tab[ok > 0]
    sx, sy, sg, R, tau0 = (t[:, k] for k in range(5))
    E = t[:, 5:8].mean(axis=1)
    flux = E * tau0 * np.pi * sg ** 2 * (1.0 - np.exp(-w.support_f ** 2))
    W, H = cam.width, cam.height
    ox = np.clip(np.minimum(sx + R, W) - np.maximum(sx - R, 0.0), 0.0, None)
    oy = np.clip(np.minimum(sy + R, H) - np.maximum(sy - R, 0.0), 0.0, None)
    frac = (ox * oy) / np.maximum(4.0 * R * R, 1e-300)
    return float(np.sum(flux * frac) / (W * H))


def main(names):
    table = {}
    for name in names:
        cfg._BRIGHTNESS[name] = 1.0
        w = workloads.make(name)
        stride = STRIDE[name]
        ws = w.subsample(stride) if stride > 1 else w
        del w
        m = frame_mean_S(ws, ws.cameras[0]) * stride
        table[name] = 1.0 / m
        print(f"{name}: n={workloads.FULL_N[name]} stride={stride} frame-mean S at brightness 1 = {m:.6g} "
              f"-> brightness {table[name]:.6g}", flush=True)
    path = os.path.join(os.path.dirname(os.path.abspath(cfg.__file__)), "brightness_table.py")
    old = {}
    if os.path.exists(path):
        ns = {}
        exec(open(path).read(), ns)
        old = ns.get("BRIGHTNESS", {})
    old.update(table)
    with open(path, "w") as f:
        f.write('"""Written by oracle/calibrate_brightness.py (closed-form frame-mean of raw S = 1 at full size)."""\n')
        f.write("BRIGHTNESS = {\n")
        for k in sorted(old):
            f.write(f"    {k!r}: {float(np.float32(old[k]))!r},\n")
        f.write("}\n")


if __name__ == "__main__":
    main(sys.argv[1:] or ["C1", "C2", "C3", "C4", "C5"])
