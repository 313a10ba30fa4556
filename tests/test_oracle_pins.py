"""Pins of the CPU oracle against what the paper and the mathematics fix.

The paper (arxiv 1004.1302) prints no worked numerical example and no pixel value, so the pins
are closed forms, invariants, special cases and brute force:
  * true 3-D ray integration of the Gaussian density of PAPER.md:69 (P1, camera conventions)
  * closed-form flux of a truncated Gaussian splat and energy conservation (P2, P3)
  * permutation and scale invariance (P4, P10)
  * RK4 integration of the transfer equation, Eq. (1) (P5, P6)
  * absorb == additive when A == E; front-to-back == back-to-front (P7, P8)
  * image orientation, culling, look-up table nodes, tie order (P9, P11, P12)
None of these reuses an oracle routine to produce its expected value.
"""
import numpy as np
import pytest

import oracle
from workloads import ABSORB, ADDITIVE

from helpers import cam, const_lut, mk

SQRT_PI = np.sqrt(np.pi)


def _basis(c):
    """Right-handed pinhole basis of DESIGN.md R1/R2, restated independently of the oracle."""
    eye, look, up = (np.array(v, np.float32).astype(np.float64) for v in (c.eye, c.lookat, c.up))
    fwd = look - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, up)
    right /= np.linalg.norm(right)
    upv = np.cross(right, fwd)
    F = 0.5 * c.width / np.tan(np.deg2rad(float(np.float32(c.fov_deg))) / 2)
    return eye, right, upv, fwd, F


# ------------------------------------------------------------------------------------------------
# P1 + conventions: the image of ONE particle equals the numerically integrated column density of
# rho = I exp(-|x - p|^2 / r^2) along the true 3-D ray through each pixel centre.
# A narrow field of view makes the paraxial reading R3 exact to ~2e-4.
# ------------------------------------------------------------------------------------------------
def test_p1_true_ray_integration_single_particle():
    c = cam(eye=(0, 0, -200.0), fov=0.5, w=33, h=33)
    w = mk([(0.10, -0.05, 0.30, 0.12, 0.7, 0.0)], c, lut_e=const_lut((1.0, 0.5, 0.25)), support_f=3.0)
    img = oracle.render(w, raw=True)
    eye, right, upv, fwd, F = _basis(c)
    p = np.array([w.x[0], w.y[0], w.z[0]], np.float64)
    r, I = float(w.r[0]), float(w.I[0])
    tab, ok = oracle.splat_table(w)
    assert ok[0] == 1
    sxo, syo, sgo, Ro = tab[0, :4]
    n_cov = 0
    for j in range(c.height):
        for i in range(c.width):
            d = fwd * F + right * (i + 0.5 - c.width / 2) + upv * (c.height / 2 - (j + 0.5))
            d /= np.linalg.norm(d)
            tc = np.dot(p - eye, d)
            t = np.linspace(tc - 9 * r, tc + 9 * r, 4001)
            pts = eye[None, :] + t[:, None] * d[None, :]
            rho = I * np.exp(-np.sum((pts - p) ** 2, axis=1) / r ** 2)
            tau = float(np.sum(rho[1:] + rho[:-1]) * 0.5 * (t[1] - t[0]))
            b = np.linalg.norm((p - eye) - tc * d)           # true impact parameter
            dd = np.hypot(i + 0.5 - sxo, j + 0.5 - syo)
            if abs(dd - Ro) < 0.05:                          # rim pixels: either answer is legal here
                continue
            if b <= 3.0 * r:
                n_cov += 1
                np.testing.assert_allclose(img[j, i], tau * np.array([1.0, 0.5, 0.25]), rtol=5e-4, atol=0)
            else:
                assert np.all(img[j, i] == 0.0)
    assert n_cov > 100


# ------------------------------------------------------------------------------------------------
# P2: flux of one splat fully inside the frame:
#     sum_pixels S_c = a_c pi sigma_s^2 (1 - exp(-f^2)),  a_c = E_c I r sqrt(pi)
# (integral of the truncated 2-D Gaussian; grid sampling error 2 exp(-pi^2 sigma_s^2) + rim term).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("f,tol", [(3.0, 3e-4), (5.0, 1e-9)])
@pytest.mark.parametrize("off", [(0.0, 0.0), (0.013, -0.007), (0.0041, 0.0093)])
def test_p2_flux_closed_form(f, tol, off):
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=96, h=96)
    w = mk([(off[0], off[1], 0.0, 0.1, 0.8, 0.0)], c, lut_e=const_lut((0.9, 0.6, 0.3)), support_f=f)
    S = oracle.render(w, raw=True)
    F = 48.0 / np.tan(np.deg2rad(10.0))
    sigma_s = F * float(w.r[0]) / 10.0
    assert sigma_s > 2.0
    a = np.array([0.9, 0.6, 0.3], np.float32).astype(np.float64) * float(w.I[0]) * float(w.r[0]) * SQRT_PI
    expect = a * np.pi * sigma_s ** 2 * (1.0 - np.exp(-f * f))
    np.testing.assert_allclose(S.sum(axis=(0, 1)), expect, rtol=tol)


# P3: energy conservation for many splats inside the frame
def test_p3_energy_conservation_many_splats():
    rs = np.random.RandomState(7)
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=128, h=128)
    F = 64.0 / np.tan(np.deg2rad(10.0))
    n = 200
    z = rs.uniform(-1.0, 1.0, n)
    zc = z + 10.0
    sig_s = rs.uniform(2.0, 6.0, n)
    r = sig_s * zc / F
    # keep the whole disc (f = 3) inside the frame
    half = (64.0 - 3.0 * sig_s - 1.0) * zc / F
    x = rs.uniform(-1, 1, n) * half
    y = rs.uniform(-1, 1, n) * half
    I = rs.uniform(0.5, 1.0, n)
    cv = rs.uniform(0, 1, n)
    lut = np.array([[0.2, 0.5, 0.9], [1.0, 0.3, 0.1]], np.float32)
    w = mk(np.stack([x, y, z, r, I, cv], 1), c, lut_e=lut, brightness=(0.7,))
    S = oracle.render(w, raw=True)
    cvf = w.colval.astype(np.float64)
    E = np.float64(np.float32(0.7)) * ((1 - cvf)[:, None] * lut[0].astype(np.float64) + cvf[:, None] * lut[1].astype(np.float64))
    sig = F * w.r.astype(np.float64) / (w.z.astype(np.float64) + 10.0)
    a = E * (w.I.astype(np.float64) * w.r.astype(np.float64) * SQRT_PI)[:, None]
    expect = (a * (np.pi * sig ** 2 * (1 - np.exp(-9.0)))[:, None]).sum(axis=0)
    np.testing.assert_allclose(S.sum(axis=(0, 1)), expect, rtol=3e-4)


# P4: the additive image does not depend on the particle order
def test_p4_permutation_invariance():
    import workloads
    w = workloads.make("C1", 5000, width=64, height=64)
    S = oracle.render(w, raw=True)
    perm = np.random.RandomState(3).permutation(w.n)
    w2 = mk(np.stack([w.x[perm], w.y[perm], w.z[perm], w.r[perm], w.I[perm], w.colval[perm]], 1), w.camera,
            lut_e=w.lut_e, brightness=w.brightness)
    S2 = oracle.render(w2, raw=True)
    np.testing.assert_allclose(S2, S, rtol=1e-12, atol=1e-300)
    assert S.max() > 0


# ------------------------------------------------------------------------------------------------
# brute force: RK4 integration of Eq. (1) along depth, for every pixel of a tiny image,
# density of particle p along the ray = I_p exp(-d^2/sigma_s^2) exp(-(s - z_p)^2 / r_p^2) [d <= R]
# ------------------------------------------------------------------------------------------------
def _ode_image(w, c, E, A, n_steps=6000):
    eye, right, upv, fwd, F = _basis(c)
    P = np.stack([w.x, w.y, w.z], 1).astype(np.float64) - eye[None]
    zc = P @ fwd
    sx = c.width / 2 + F * (P @ right) / zc
    sy = c.height / 2 - F * (P @ upv) / zc
    sg = F * w.r.astype(np.float64) / zc
    R = w.support_f * sg
    rr = w.r.astype(np.float64)
    jj, ii = np.meshgrid(np.arange(c.height) + 0.5, np.arange(c.width) + 0.5, indexing="ij")
    d2 = (ii[None] - sx[:, None, None]) ** 2 + (jj[None] - sy[:, None, None]) ** 2
    amp = w.I.astype(np.float64)[:, None, None] * np.exp(-d2 / sg[:, None, None] ** 2) * (d2 <= (R ** 2)[:, None, None])
    s_far, s_near = (zc + 7 * rr).max(), (zc - 7 * rr).min()
    h = (s_far - s_near) / n_steps            # step of the propagation coordinate (far -> near)

    def rhs(s, Iv):                            # Iv: (H, W, 3)
        out = np.zeros_like(Iv)
        for p in range(len(zc)):
            rho = amp[p] * np.exp(-((s - zc[p]) ** 2) / rr[p] ** 2)
            out += (E[p][None, None, :] - A[p][None, None, :] * Iv) * rho[:, :, None]
        return out

    Iv = np.zeros((c.height, c.width, 3))
    s = s_far
    for _ in range(n_steps):
        k1 = rhs(s, Iv)
        k2 = rhs(s - h / 2, Iv + h * k1 / 2)
        k3 = rhs(s - h / 2, Iv + h * k2 / 2)
        k4 = rhs(s - h, Iv + h * k3)
        Iv = Iv + h * (k1 + 2 * k2 + 2 * k3 + k4) / 6
        s -= h
    return Iv


_LUT2E = np.array([[0.2, 0.5, 0.9], [1.0, 0.3, 0.1]], np.float32)
_LUT2A = np.array([[1.5, 0.1, 0.6], [0.05, 0.9, 2.0]], np.float32)


def _lerp(lut, cv):
    cv = np.asarray(cv, np.float32).astype(np.float64)
    return (1 - cv)[:, None] * lut[0].astype(np.float64) + cv[:, None] * lut[1].astype(np.float64)


def test_p5_rk4_additive_overlapping():
    c = cam(eye=(0, 0, -10.0), fov=6.0, w=8, h=8)
    pts = [(0.00, 0.00, 0.00, 0.10, 2.0, 0.0), (0.05, -0.04, 0.05, 0.16, 1.2, 0.5),
           (-0.08, 0.06, -0.08, 0.12, 3.0, 1.0), (0.10, 0.10, 0.02, 0.05, 4.0, 0.25),
           (-0.12, -0.10, 0.20, 0.20, 0.9, 0.75)]
    w = mk(pts, c, lut_e=_LUT2E, brightness=(1.3,))
    E = np.float64(np.float32(1.3)) * _lerp(_LUT2E, w.colval)
    ref = _ode_image(w, c, E, E)
    out = oracle.render(w)                      # 1 - exp(-S)
    assert out.max() > 0.2
    np.testing.assert_allclose(out, ref, rtol=1e-7, atol=1e-9)


def _disjoint_points():
    # separated in depth by more than 6 (r_p + r_q) so that the slab reading R10 is exact
    return [(0.00, 0.00, -3.0, 0.10, 2.0, 0.0), (0.05, -0.04, 0.0, 0.16, 1.2, 0.5),
            (-0.08, 0.06, 3.0, 0.12, 3.0, 1.0), (0.02, 0.03, 6.0, 0.20, 1.5, 0.25)]


def test_p6_rk4_absorb_disjoint_and_order_matters():
    c = cam(eye=(0, 0, -12.0), fov=6.0, w=8, h=8)
    w = mk(_disjoint_points(), c, lut_e=_LUT2E, lut_a=_LUT2A, brightness=(1.3,), abs_brightness=(0.8,), mode=ABSORB)
    E = np.float64(np.float32(1.3)) * _lerp(_LUT2E, w.colval)
    A = np.float64(np.float32(0.8)) * _lerp(_LUT2A, w.colval)
    ref = _ode_image(w, c, E, A, n_steps=12000)
    out = oracle.render(w)
    assert out.max() > 0.2
    np.testing.assert_allclose(out, ref, rtol=2e-7, atol=1e-9)
    # reversing the depth order (mirror the particles through the lookat plane) changes the image
    pts2 = [(x, y, 3.0 - z, r, I, cv) for (x, y, z, r, I, cv) in _disjoint_points()]
    w2 = mk(pts2, c, lut_e=_LUT2E, lut_a=_LUT2A, brightness=(1.3,), abs_brightness=(0.8,), mode=ABSORB)
    out2 = oracle.render(w2)
    assert np.abs(out2 - out).max() > 1e-2


def test_p7_absorb_with_a_equal_e_is_additive():
    import workloads
    w = workloads.make("C1", 3000, width=48, height=48)
    w.brightness = [w.brightness[0] * 3.0]
    add = oracle.render(w, mode=ADDITIVE)
    w.lut_a = w.lut_e.copy()
    w.abs_brightness = list(w.brightness)
    ab = oracle.render(w, mode=ABSORB)
    assert add.max() > 0.5
    np.testing.assert_allclose(ab, add, rtol=1e-11, atol=1e-14)


def test_p8_front_to_back_equals_back_to_front():
    """The (C, T) recurrence nearest-first, written out here, equals the oracle's far-to-near form."""
    import workloads
    w = workloads.make("C4", 2000, width=32, height=32)
    c = w.camera
    out = oracle.render(w)
    tab, ok = oracle.splat_table(w)
    pr = oracle.project_f32(w)
    vis = ok.astype(bool)
    key = pr["zkey"].astype(np.int64).copy()
    # particles the canonical box test dropped but the double table kept need a key too
    order = [p for p in np.lexsort((np.arange(w.n), key)) if vis[p] and pr["visible"][p]]
    missing = [p for p in range(w.n) if vis[p] and not pr["visible"][p]]
    Cimg = np.zeros((c.height, c.width, 3))
    Timg = np.ones((c.height, c.width, 3))
    jj, ii = np.meshgrid(np.arange(c.height) + 0.5, np.arange(c.width) + 0.5, indexing="ij")
    for p in order:
        sx, sy, sg, R, tau0 = tab[p, :5]
        d2 = (ii - sx) ** 2 + (jj - sy) ** 2
        tau = np.where(d2 <= R * R, tau0 * np.exp(-d2 / sg ** 2), 0.0)[:, :, None]
        u = tab[p, 8:11][None, None, :] * tau
        phi = np.where(u > 0, -np.expm1(-u) / np.where(u > 0, u, 1.0), 1.0)
        Cimg += Timg * tab[p, 5:8][None, None, :] * tau * phi
        Timg *= np.exp(-u)
    # the few splats outside the canonical box touch no pixel centre: they cannot change the image
    for p in missing:
        sx, sy, sg, R = tab[p, :4]
        assert not np.any((ii - sx) ** 2 + (jj - sy) ** 2 <= R * R)
    assert out.max() > 0.05
    np.testing.assert_allclose(out, Cimg, rtol=1e-10, atol=1e-13)


# ------------------------------------------------------------------------------------------------
# P9: conventions R1, R2, R4, R5, R6
# ------------------------------------------------------------------------------------------------
def test_p9_orientation_and_culling():
    c = cam(eye=(0, 0, -10.0), lookat=(0, 0, 0), up=(0, 1, 0), fov=20.0, w=65, h=65)
    eye, right, upv, fwd, F = _basis(c)
    base = dict(lut_e=const_lut((1, 1, 1)))

    def centroid(pt):
        S = oracle.render(mk([pt], c, **base), raw=True)[:, :, 0]
        jj, ii = np.meshgrid(np.arange(65) + 0.5, np.arange(65) + 0.5, indexing="ij")
        return (S * ii).sum() / S.sum(), (S * jj).sum() / S.sum(), S

    cx, cy, S = centroid((0, 0, 0, 0.05, 1, 0))
    assert abs(cx - 32.5) < 1e-9 and abs(cy - 32.5) < 1e-9      # optical axis -> (W/2, H/2)
    ux, uy, _ = centroid(tuple(0.3 * upv) + (0.05, 1, 0))
    assert uy < cy - 3 and abs(ux - cx) < 1e-6                    # +up -> smaller row index
    rx, ry, _ = centroid(tuple(0.3 * right) + (0.05, 1, 0))
    assert rx > cx + 3 and abs(ry - cy) < 1e-6                    # +right (= fwd x up) -> larger column
    # expected displacement F * 0.3 / 10 pixels
    assert abs((rx - cx) - F * 0.3 / 10.0) < 1e-3
    # behind the camera, off-frame, inside the near plane, invalid fields: exactly zero
    for pt in [(0, 0, -20.0, 0.05, 1, 0), (50.0, 0, 0, 0.05, 1, 0), (0, 0, -10.0 + 0.005, 0.05, 1, 0),
               (0, 0, 0, -0.05, 1, 0), (0, 0, 0, 0.0, 1, 0), (np.nan, 0, 0, 0.05, 1, 0),
               (0, 0, 0, 0.05, np.inf, 0), (0, 0, 0, 0.05, 1, np.nan)]:
        assert np.all(oracle.render(mk([pt], c, **base), raw=True) == 0.0)
    # a splat too small to reach a pixel centre contributes nothing (R4); on a pixel centre it
    # lights exactly that pixel with its peak value a = E I r sqrt(pi)
    tiny = 1e-4
    Sz = oracle.render(mk([(0, 0, 0, tiny, 1, 0)], cam(eye=(0, 0, -10.0), fov=20.0, w=64, h=64), **base), raw=True)
    assert np.all(Sz == 0.0)                                      # W even: the axis falls between pixels
    So = oracle.render(mk([(0, 0, 0, tiny, 1, 0)], c, **base), raw=True)
    assert np.count_nonzero(So[:, :, 0]) == 1
    np.testing.assert_allclose(So[32, 32], np.float64(np.float32(tiny)) * SQRT_PI, rtol=1e-12)


def test_p9_type_out_of_range_is_culled():
    c = cam(w=16, h=16)
    w = mk([(0, 0, 0, 0.2, 1, 0), (0, 0, 0, 0.2, 1, 0)], c, lut_e=const_lut((1, 1, 1), n_types=2),
           brightness=(1.0, 2.0), types=[1, 3])
    w1 = mk([(0, 0, 0, 0.2, 1, 0)], c, lut_e=const_lut((1, 1, 1), n_types=2), brightness=(1.0, 2.0), types=[1])
    np.testing.assert_array_equal(oracle.render(w, raw=True), oracle.render(w1, raw=True))


# P10: tau is proportional to I r, so scaling every length by s and I by 1/s leaves the image unchanged
def test_p10_scale_invariance():
    c = cam(eye=(0.5, 0.25, -8.0), lookat=(0.5, 0.25, 0.0), fov=16.0, w=40, h=40)
    rs = np.random.RandomState(11)
    pts = np.stack([rs.uniform(-0.5, 1.5, 40), rs.uniform(-0.5, 1.0, 40), rs.uniform(-1, 1, 40),
                    rs.uniform(0.02, 0.2, 40), rs.uniform(0.5, 1, 40), rs.uniform(0, 1, 40)], 1)
    w = mk(pts, c, lut_e=_LUT2E, lut_a=_LUT2A, mode=ABSORB, z_near=0.01)
    s = 4.0                                                       # power of two: exact in fp32
    pts2 = np.stack([w.x * s, w.y * s, w.z * s, w.r * s, w.I / s, w.colval], 1)
    c2 = cam(eye=tuple(np.array(c.eye) * s), lookat=tuple(np.array(c.lookat) * s), fov=16.0, w=40, h=40)
    w2 = mk(pts2, c2, lut_e=_LUT2E, lut_a=_LUT2A, mode=ABSORB, z_near=0.01 * s)
    for mode in (ADDITIVE, ABSORB):
        np.testing.assert_allclose(oracle.render(w2, mode=mode), oracle.render(w, mode=mode), rtol=1e-12, atol=1e-15)


# P11: look-up table (R7)
def test_p11_lut_nodes_midpoints_clamp():
    c = cam(w=16, h=16)
    lut = np.array([[0.1, 0.2, 0.3], [0.5, 0.1, 0.9], [0.0, 1.0, 0.4], [0.7, 0.7, 0.2], [1.0, 0.0, 0.6]], np.float32)
    cvs = [0.0, 0.25, 0.5, 0.75, 1.0, 0.125, 0.875, -3.0, 7.0, 0.3]
    w = mk([(0, 0, 0, 0.1, 1, v) for v in cvs], c, lut_e=lut, brightness=(2.0,))
    tab, ok = oracle.splat_table(w)
    assert ok.all()
    E = tab[:, 5:8]
    L = lut.astype(np.float64)
    for k in range(5):
        np.testing.assert_array_equal(E[k], 2.0 * L[k])                      # nodes return table entries
    np.testing.assert_allclose(E[5], 2.0 * 0.5 * (L[0] + L[1]), rtol=1e-15)   # midpoints return averages
    np.testing.assert_allclose(E[6], 2.0 * 0.5 * (L[3] + L[4]), rtol=1e-15)
    np.testing.assert_array_equal(E[7], 2.0 * L[0])                           # clamp below / above
    np.testing.assert_array_equal(E[8], 2.0 * L[4])
    u = float(np.float32(0.3)) * 4
    np.testing.assert_allclose(E[9], 2.0 * ((2 - u) * L[1] + (u - 1) * L[2]), rtol=1e-14)
    np.testing.assert_array_equal(tab[:, 8:11], E)                            # additive: A == E


# P12: equal fp32 depth keys composite in particle-index order, lower index in front (R11)
def test_p12_tie_order_by_index():
    c = cam(eye=(0, 0, -10.0), fov=10.0, w=16, h=16)
    a = (0.0, 0.0, 0.0, 0.3, 2.0, 0.0)
    b = (0.0, 0.0, 0.0, 0.3, 2.0, 1.0)
    kw = dict(lut_e=_LUT2E, lut_a=_LUT2A, mode=ABSORB)
    o_ab = oracle.render(mk([a, b], c, **kw))
    o_ba = oracle.render(mk([b, a], c, **kw))
    assert np.abs(o_ab - o_ba).max() > 1e-2
    # expected: index 0 in front, i.e. C = C_0 + T_0 C_1 at the centre pixel region
    tab, _ = oracle.splat_table(mk([a, b], c, **kw))
    jj, ii = np.meshgrid(np.arange(16) + 0.5, np.arange(16) + 0.5, indexing="ij")
    d2 = (ii - tab[0, 0]) ** 2 + (jj - tab[0, 1]) ** 2
    tau = np.where(d2 <= tab[0, 3] ** 2, tab[0, 4] * np.exp(-d2 / tab[0, 2] ** 2), 0.0)[:, :, None]
    E0, A0, E1, A1 = (_LUT2E[0].astype(np.float64), _LUT2A[0].astype(np.float64),
                      _LUT2E[1].astype(np.float64), _LUT2A[1].astype(np.float64))

    def contrib(E, A):
        u = A * tau
        return E * tau * np.where(u > 0, -np.expm1(-u) / np.where(u > 0, u, 1), 1.0), np.exp(-u)

    c0, t0 = contrib(E0, A0)
    c1, t1 = contrib(E1, A1)
    np.testing.assert_allclose(o_ab, c0 + t0 * c1, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(o_ba, c1 + t1 * c0, rtol=1e-12, atol=1e-15)


def test_absorb_zero_absorption_channel_is_pure_emission():
    """R15: A_c = 0 gives phi = 1, i.e. the channel accumulates E tau like raw additive S."""
    c = cam(eye=(0, 0, -10.0), fov=10.0, w=16, h=16)
    pts = [(0.0, 0.0, 0.0, 0.3, 2.0, 0.0), (0.1, 0.05, 1.0, 0.2, 1.0, 1.0)]
    lut_a = np.array([[0.0, 0.4, 0.0], [0.0, 0.9, 0.0]], np.float32)
    out = oracle.render(mk(pts, c, lut_e=_LUT2E, lut_a=lut_a, mode=ABSORB))
    raw = oracle.render(mk(pts, c, lut_e=_LUT2E), raw=True)
    np.testing.assert_allclose(out[:, :, 0], raw[:, :, 0], rtol=1e-13)
    np.testing.assert_allclose(out[:, :, 2], raw[:, :, 2], rtol=1e-13)
    assert np.all(out[:, :, 1] <= raw[:, :, 1] + 1e-15) and np.abs(out[:, :, 1] - raw[:, :, 1]).max() > 1e-3


# ------------------------------------------------------------------------------------------------
# stage (b): range normalisation of a scalar field (reading R17)
# ------------------------------------------------------------------------------------------------
def test_p14_field_normalisation_closed_forms():
    """Pins by construction: an arithmetic progression maps to k/(n-1); a geometric progression maps to k/(n-1)
    under log10 (not under the identity); the map is invariant under v -> a v + b (a > 0) resp. v -> a v; undefined
    values give NaN and do not move the range; a constant field gives 0."""
    n = 11
    k = np.arange(n) / (n - 1)
    out, (lo, hi) = oracle.normalize_field(3.0 + 0.25 * np.arange(n))
    np.testing.assert_allclose(out, k, atol=1e-15)
    assert (lo, hi) == (3.0, 5.5)
    geo = 1e-3 * 10.0 ** (0.5 * np.arange(n))
    out, (lo, hi) = oracle.normalize_field(geo, log_scale=True)
    np.testing.assert_allclose(out, k, atol=1e-14)
    np.testing.assert_allclose((lo, hi), (-3.0, 2.0), atol=1e-14)
    assert np.abs(oracle.normalize_field(geo)[0][1:-1] - k[1:-1]).min() > 0.05      # the identity map is a different function
    rs = np.random.RandomState(3)
    v = rs.lognormal(0.0, 2.0, 1000)
    np.testing.assert_allclose(oracle.normalize_field(7.0 * v - 2.0)[0], oracle.normalize_field(v)[0], atol=1e-12)
    np.testing.assert_allclose(oracle.normalize_field(7.0 * v, True)[0], oracle.normalize_field(v, True)[0], atol=1e-12)
    w = v.copy()
    w[[5, 17]] = [np.nan, np.inf]
    out, rng_ = oracle.normalize_field(w)
    assert np.isnan(out[[5, 17]]).all() and np.isfinite(np.delete(out, [5, 17])).all()
    assert rng_ == oracle.normalize_field(np.delete(v, [5, 17]))[1]
    w = v.copy()
    w[[1, 2]] = [0.0, -4.0]
    out, rng_ = oracle.normalize_field(w, True)
    assert np.isnan(out[[1, 2]]).all() and out[np.argmax(w)] == 1.0 and np.nanmin(out) == 0.0
    out, rng_ = oracle.normalize_field(np.full(9, 2.5))
    assert (out == 0.0).all() and rng_ == (2.5, 2.5)
    out, rng_ = oracle.normalize_field(np.array([np.nan, -1.0]), True)
    assert np.isnan(out).all() and rng_ == (0.0, 0.0)
    assert oracle.normalize_field(np.zeros(0))[1] == (0.0, 0.0)


def test_p15_tonemap_codes():
    """Pins: the codes of k/255 are k; values below 0 / above 1 / NaN clamp to 0 / 255 / 0; halves round to even;
    gamma 2 maps (k/255)^2 back to k; the map is monotone."""
    k = np.arange(256)
    assert np.array_equal(oracle.tonemap_rgb8(k / 255.0), k)
    assert list(oracle.tonemap_rgb8([-1.0, 0.0, 1.0, 7.0, np.nan, np.inf, -np.inf])) == [0, 0, 255, 255, 0, 255, 0]
    assert list(oracle.tonemap_rgb8(np.array([0.5, 1.5, 2.5, 3.5]) / 255.0)) == [0, 2, 2, 4]
    assert np.array_equal(oracle.tonemap_rgb8((k / 255.0) ** 2, gamma=2.0), k)
    x = np.sort(np.random.RandomState(1).uniform(-0.2, 1.2, 5000))
    for g in (1.0, 2.2):
        assert (np.diff(oracle.tonemap_rgb8(x, g).astype(int)) >= 0).all()


def test_p16_vector_colouring_reduces_to_the_scalar_path():
    """PAPER.md:75 vector colouring (reading R19).  Pins: a constant vector is a constant colour table; in the additive
    raw sum channel c with per-particle v_c equals the scalar path with a table of ones and I scaled by v_c (tau is
    linear in I, O6); a particle with a non-finite component vanishes."""
    import copy
    rs = np.random.RandomState(7)
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=72, h=56)
    n = 40
    pts = np.stack([rs.uniform(-1.5, 1.5, n), rs.uniform(-1.2, 1.2, n), rs.uniform(-1, 1, n), rs.uniform(0.05, 0.4, n),
                    rs.uniform(0.5, 2.0, n), rs.uniform(0, 1, n)], 1)
    w = mk(pts, c, lut_e=const_lut((0.7, 0.4, 0.2)), brightness=(1.3,))
    ref = oracle.render(w, raw=True)
    wv = copy.copy(w)
    wv.vec = np.tile(np.array([[0.7, 0.4, 0.2]], np.float32), (n, 1))
    np.testing.assert_allclose(oracle.render_vector(wv, raw=True), ref, rtol=1e-12, atol=1e-15)
    vec = rs.uniform(0.0, 2.0, (n, 3)).astype(np.float32)
    wv.vec = vec
    got = oracle.render_vector(wv, raw=True)
    for ch in range(3):
        w1 = mk(np.column_stack([pts[:, :4], pts[:, 4] * vec[:, ch].astype(np.float64), pts[:, 5]]), c, lut_e=const_lut(),
                brightness=(1.3,))
        # I is stored as float32 in the workload: compare at float32 resolution of the product
        np.testing.assert_allclose(got[..., ch], oracle.render(w1, raw=True)[..., 0], rtol=3e-7, atol=1e-12)
    wv.vec = vec.copy()
    wv.vec[3, 1] = np.nan
    keep = np.arange(n) != 3
    w2 = mk(pts[keep], c, lut_e=const_lut(), brightness=(1.3,))
    w2.vec = vec[keep]
    np.testing.assert_allclose(oracle.render_vector(wv, raw=True), oracle.render_vector(w2, raw=True), rtol=1e-12, atol=1e-15)
    # absorb mode: A = abs_brightness * v as well; with equal brightness this is the additive image (P7)
    wa = mk(pts, c, lut_e=const_lut(), lut_a=const_lut(), brightness=(1.3,), abs_brightness=(1.3,), mode=ABSORB)
    wa.vec = vec
    np.testing.assert_allclose(oracle.render_vector(wa), oracle.render_vector(wv.__class__(**{**wv.__dict__, "vec": vec})), rtol=1e-9, atol=1e-12)


# ------------------------------------------------------------------------------------------------
# P17: per-type colour tables and per-type brightness (PAPER.md:75 transfer function per particle
# property; readings R7, R14).  Two types with DIFFERENT tables and DIFFERENT brightness /
# abs_brightness.  Expected values are written by hand from the input tables: a particle at table
# node k of type t has E = brightness[t] * tabE[t][k], A = abs_brightness[t] * tabA[t][k], and its
# image is the single-splat closed form of O6 / O8 evaluated here, not by the oracle.
# ------------------------------------------------------------------------------------------------
_T2E = np.array([[[0.10, 0.20, 0.30], [0.50, 0.10, 0.90], [0.00, 1.00, 0.40]],
                 [[0.80, 0.60, 0.05], [0.25, 0.75, 0.35], [0.90, 0.15, 0.65]]], np.float32)
_T2A = np.array([[[1.50, 0.10, 0.60], [0.05, 0.90, 2.00], [0.70, 0.30, 0.20]],
                 [[0.40, 1.20, 0.15], [2.50, 0.45, 0.85], [0.12, 0.55, 1.75]]], np.float32)
_BR2, _AB2 = (1.25, 0.375), (0.5, 3.0)            # exact in binary32


def test_p17_per_type_tables_and_brightness_in_the_splat_table():
    c = cam(w=16, h=16)
    pts, types = [], []
    for t in (0, 1):
        for cv in (0.0, 0.5, 1.0, 0.25):          # three nodes and one midpoint
            pts.append((0, 0, 0, 0.1, 1, cv))
            types.append(t)
    w = mk(pts, c, lut_e=_T2E, lut_a=_T2A, brightness=_BR2, abs_brightness=_AB2, mode=ABSORB, types=types)
    tab, ok = oracle.splat_table(w)
    assert ok.all()
    LE, LA = _T2E.astype(np.float64), _T2A.astype(np.float64)
    row = 0
    for t in (0, 1):
        for k in range(3):
            np.testing.assert_array_equal(tab[row, 5:8], _BR2[t] * LE[t, k])
            np.testing.assert_array_equal(tab[row, 8:11], _AB2[t] * LA[t, k])
            row += 1
        np.testing.assert_allclose(tab[row, 5:8], _BR2[t] * 0.5 * (LE[t, 0] + LE[t, 1]), rtol=1e-15)
        np.testing.assert_allclose(tab[row, 8:11], _AB2[t] * 0.5 * (LA[t, 0] + LA[t, 1]), rtol=1e-15)
        row += 1
    # additive mode: A == E of the particle's own type and brightness
    tab0, _ = oracle.splat_table(w, mode=ADDITIVE)
    np.testing.assert_array_equal(tab0[:, 8:11], tab0[:, 5:8])
    np.testing.assert_array_equal(tab0[:, 5:8], tab[:, 5:8])


@pytest.mark.parametrize("mode", [ADDITIVE, ABSORB])
def test_p17_per_type_single_splat_image_closed_form(mode):
    """One particle per type, far apart on the screen, each at a table node of its own type: every pixel
    equals the hand-evaluated single-splat value with that type's table row and brightness."""
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=96, h=48)
    F = 48.0 / np.tan(np.deg2rad(10.0))
    #            x     y    z    r     I    colval            type, node
    pts = [(-1.0, 0.1, 0.0, 0.15, 0.8, 0.5), (1.1, -0.2, 0.5, 0.12, 1.5, 1.0)]
    types, nodes = [1, 0], [1, 2]
    w = mk(pts, c, lut_e=_T2E, lut_a=_T2A, brightness=_BR2, abs_brightness=_AB2, mode=mode, types=types)
    img = oracle.render(w, raw=True)
    jj, ii = np.meshgrid(np.arange(c.height) + 0.5, np.arange(c.width) + 0.5, indexing="ij")
    expect = np.zeros((c.height, c.width, 3))
    for p in range(2):
        x, y, z, r, I = (float(np.float32(v)) for v in pts[p][:5])
        zc = z + 10.0                              # right = fwd x up = (-1, 0, 0) for this camera (R2)
        sx, sy, sg = c.width / 2 - F * x / zc, c.height / 2 - F * y / zc, F * r / zc
        d2 = (ii - sx) ** 2 + (jj - sy) ** 2
        tau = np.where(d2 <= (3.0 * sg) ** 2, I * r * SQRT_PI * np.exp(-d2 / sg ** 2), 0.0)[:, :, None]
        E = _BR2[types[p]] * _T2E[types[p], nodes[p]].astype(np.float64)
        if mode == ADDITIVE:
            expect += E * tau
        else:
            A = _AB2[types[p]] * _T2A[types[p], nodes[p]].astype(np.float64)
            u = A * tau
            expect += E * tau * np.where(u > 0, -np.expm1(-u) / np.where(u > 0, u, 1.0), 1.0)   # discs do not overlap
    assert (expect[:, :48] > 0).any() and (expect[:, 48:] > 0).any() and np.all(expect[:, 46:50] == 0)   # disjoint discs
    np.testing.assert_allclose(img, expect, rtol=1e-11, atol=1e-15)


def test_p17_type_out_of_range_is_culled_and_in_range_types_differ():
    """R6: type >= n_types contributes exactly 0; the same particle rendered as type 0 and as type 1 differs by the
    hand-computed ratio of brightness * table entry (a `type -> 0` slip anywhere would make them equal)."""
    c = cam(w=16, h=16)
    lut = np.stack([const_lut((1.0, 0.5, 0.25))[0], const_lut((0.5, 1.0, 0.125))[0]])
    kw = dict(lut_e=lut, brightness=(1.0, 2.0))
    S0 = oracle.render(mk([(0, 0, 0, 0.2, 1, 0)], c, types=[0], **kw), raw=True)
    S1 = oracle.render(mk([(0, 0, 0, 0.2, 1, 0)], c, types=[1], **kw), raw=True)
    S3 = oracle.render(mk([(0, 0, 0, 0.2, 1, 0)], c, types=[3], **kw), raw=True)
    assert S0.max() > 0 and np.all(S3 == 0.0)
    np.testing.assert_allclose(S1[..., 0], S0[..., 0] * 1.0, rtol=1e-15)      # 2.0 * 0.5  vs 1.0 * 1.0
    np.testing.assert_allclose(S1[..., 1], S0[..., 1] * 4.0, rtol=1e-15)      # 2.0 * 1.0  vs 1.0 * 0.5
    np.testing.assert_allclose(S1[..., 2], S0[..., 2] * 1.0, rtol=1e-15)      # 2.0 * .125 vs 1.0 * 0.25


# ------------------------------------------------------------------------------------------------
# P18: the region-of-interest path of the oracle (SURVEY.md 8(c) "Oracle practicalities"): the only
# checker of the full-size images.  An off-origin, non-aligned ROI must equal (a) the hand-evaluated
# single-splat closed form a exp(-d^2/sigma_s^2) at the ROI's own pixel centres, (b) the same crop of
# the full-frame render bit for bit, in both modes, with many overlapping particles (the per-pixel
# visiting order is the same, so even the rounding is).
# ------------------------------------------------------------------------------------------------
def test_p18_roi_single_splat_closed_form_at_roi_pixels():
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=80, h=64)
    F = 40.0 / np.tan(np.deg2rad(10.0))
    x, y, z, r, I = (float(np.float32(v)) for v in (0.31, -0.17, 0.4, 0.21, 0.9))
    w = mk([(x, y, z, r, I, 0.0)], c, lut_e=const_lut((0.9, 0.6, 0.3)))
    zc = z + 10.0
    sx, sy, sg = 40.0 - F * x / zc, 32.0 - F * y / zc, F * r / zc      # right = fwd x up = (-1, 0, 0) (R2)
    a = np.array([0.9, 0.6, 0.3], np.float32).astype(np.float64) * I * r * SQRT_PI
    for roi in [(14, 21, 43, 50), (33, 33, 34, 34), (0, 33, 80, 40), (29, 0, 36, 64), (60, 5, 77, 11)]:
        x0, y0, x1, y1 = roi
        got = oracle.render(w, roi=roi, raw=True)
        assert got.shape == (y1 - y0, x1 - x0, 3)
        jj, ii = np.meshgrid(np.arange(y0, y1) + 0.5, np.arange(x0, x1) + 0.5, indexing="ij")
        d2 = (ii - sx) ** 2 + (jj - sy) ** 2
        expect = np.where(d2 <= (3.0 * sg) ** 2, np.exp(-d2 / sg ** 2), 0.0)[:, :, None] * a
        np.testing.assert_allclose(got, expect, rtol=1e-11, atol=1e-300)
    assert oracle.render(w, roi=(14, 21, 43, 50), raw=True).max() > 0.05


@pytest.mark.parametrize("mode", [ADDITIVE, ABSORB])
def test_p18_roi_equals_crop_of_full_frame(mode):
    rs = np.random.RandomState(23)
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=150, h=131)
    n = 600
    pts = np.stack([rs.uniform(-2.2, 2.2, n), rs.uniform(-2.0, 2.0, n), rs.uniform(-1, 1, n),
                    np.exp(rs.uniform(np.log(0.01), np.log(0.6), n)), rs.uniform(0.5, 1.5, n), rs.uniform(0, 1, n)], 1)
    types = rs.randint(0, 2, n)
    w = mk(pts, c, lut_e=_T2E, lut_a=_T2A, brightness=_BR2, abs_brightness=_AB2, mode=mode, types=types)
    full = oracle.render(w)
    assert full.max() > 0.1
    for roi in [(37, 21, 101, 85), (1, 1, 150, 131), (149, 130, 150, 131), (64, 64, 128, 128), (13, 90, 77, 107),
                (100, 0, 150, 3)]:
        x0, y0, x1, y1 = roi
        got = oracle.render(w, roi=roi)
        np.testing.assert_array_equal(got, full[y0:y1, x0:x1])


# ------------------------------------------------------------------------------------------------
# P19 (reading R20): negative absorption / emission / optical-depth modulation are unphysical but
# "used as given": the slab solution of Eq. (1), holds for either sign of u = A tau.
# RK4 integration of Eq. (1) with a negative A channel, a negative E channel and one negative I.
# ------------------------------------------------------------------------------------------------
def test_p19_rk4_absorb_negative_coefficients():
    c = cam(eye=(0, 0, -12.0), fov=6.0, w=8, h=8)
    pts = _disjoint_points()
    pts[2] = pts[2][:4] + (-1.5,) + pts[2][5:]                   # negative I
    lut_e = np.array([[0.2, -0.5, 0.9], [1.0, 0.3, -0.1]], np.float32)
    lut_a = np.array([[1.5, 0.1, -0.6], [-0.05, 0.9, 2.0]], np.float32)
    w = mk(pts, c, lut_e=lut_e, lut_a=lut_a, brightness=(1.3,), abs_brightness=(0.8,), mode=ABSORB)
    E = np.float64(np.float32(1.3)) * _lerp(lut_e, w.colval)
    A = np.float64(np.float32(0.8)) * _lerp(lut_a, w.colval)
    ref = _ode_image(w, c, E, A, n_steps=12000)
    out = oracle.render(w)
    assert out.max() > 0.2 and out.min() < -0.05
    np.testing.assert_allclose(out, ref, rtol=2e-7, atol=1e-9)
    # additive mode is linear in E and I: S(-I) = -S(I)
    wa = mk(pts, c, lut_e=lut_e, brightness=(1.3,))
    pts_pos = [p[:4] + (abs(p[4]),) + p[5:] for p in pts]
    Sa = oracle.render(wa, raw=True)
    only = oracle.render(mk([pts[2]], c, lut_e=lut_e, brightness=(1.3,)), raw=True)
    only_pos = oracle.render(mk([pts_pos[2]], c, lut_e=lut_e, brightness=(1.3,)), raw=True)
    np.testing.assert_allclose(only, -only_pos, rtol=1e-15)
    np.testing.assert_allclose(Sa, oracle.render(mk(pts_pos, c, lut_e=lut_e, brightness=(1.3,)), raw=True) - 2.0 * only_pos,
                               rtol=1e-12, atol=1e-15)
