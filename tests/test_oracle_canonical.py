"""Pins of the canonical fp32 projector / binner (the integers the CUDA path must match bit-exactly).

The integer definitions are north_star's, not the paper's ("Tile/bin indices and counts must be
bit-exact"); the paper only says "determining screen areas affected by individual particles"
(PAPER.md:105).  They are pinned here against (i) the same sequence evaluated with numpy float32
scalars (an independent IEEE implementation: catches contraction / double-promotion in the C
build), (ii) the double splat table, (iii) brute-force binning in Python, (iv) numpy's lexsort.
"""
import numpy as np

import oracle
import workloads
from workloads import Camera

from helpers import cam, mk


def _small(name="C1", n=4000, w=96, h=80):
    return workloads.make(name, n, width=w, height=h)


def test_projector_matches_numpy_float32_sequence():
    w = _small("C4", 3000, 96, 80)
    c = w.camera
    pr = oracle.project_f32(w)
    right, upv, fwd, F = oracle.camera_basis(c)
    f32 = np.float32
    r3, u3, f3 = right.astype(f32), upv.astype(f32), fwd.astype(f32)
    e = np.array(c.eye, f32)
    Ff, cx, cy = f32(F), f32(c.width / 2), f32(c.height / 2)
    nvis = 0
    for p in range(w.n):
        dx, dy, dz = w.x[p] - e[0], w.y[p] - e[1], w.z[p] - e[2]

        def dot(v):
            # fmaf(dz, v.z, fmaf(dy, v.y, dx * v.x)) emulated exactly in float64 (products of two
            # float32 are exact in float64; one rounding per fused step)
            t = f32(np.float64(dx) * np.float64(v[0]))
            t = f32(np.float64(dy) * np.float64(v[1]) + np.float64(t))
            return f32(np.float64(dz) * np.float64(v[2]) + np.float64(t))

        xc, yc, zc = dot(r3), dot(u3), dot(f3)
        if not (zc > f32(w.z_near)):
            assert pr["visible"][p] == 0
            continue
        q = Ff / zc
        sx = f32(np.float64(xc) * np.float64(q) + np.float64(cx))
        sy = f32(-np.float64(yc) * np.float64(q) + np.float64(cy))
        ss = w.r[p] * q
        R = f32(w.support_f) * ss
        i0 = min(max(np.ceil((sx - R) - f32(0.5)), 0), c.width)
        i1 = max(min(np.floor((sx + R) - f32(0.5)), c.width - 1), -1)
        j0 = min(max(np.ceil((sy - R) - f32(0.5)), 0), c.height)
        j1 = max(min(np.floor((sy + R) - f32(0.5)), c.height - 1), -1)
        vis = bool(i0 <= i1 and j0 <= j1 and ss > 0 and np.isfinite(R))
        assert bool(pr["visible"][p]) == vis
        if vis:
            nvis += 1
            assert pr["sx"][p] == sx and pr["sy"][p] == sy and pr["ss"][p] == ss and pr["R"][p] == R
            assert tuple(pr["bbox"][p]) == (int(i0), int(i1), int(j0), int(j1))
            assert pr["zkey"][p] == np.array([zc], f32).view(np.uint32)[0]
    assert 200 < nvis < w.n            # camera inside the volume: a real mix of culled and visible


def test_projector_agrees_with_double_table_and_box_is_tight():
    w = _small("C1", 4000)
    pr = oracle.project_f32(w)
    tab, ok = oracle.splat_table(w)
    vis = pr["visible"] > 0
    assert vis.sum() > 1000
    # fp32 screen position within a few ulp of the double one
    assert np.abs(pr["sx"][vis] - tab[vis, 0]).max() < 1e-4
    assert np.abs(pr["sy"][vis] - tab[vis, 1]).max() < 1e-4
    assert np.abs(pr["ss"][vis] / tab[vis, 2] - 1).max() < 1e-6
    # the box holds every pixel centre within R and no empty border column/row beyond rounding
    b = pr["bbox"][vis].astype(np.float64)
    sx, sy, R = tab[vis, 0], tab[vis, 1], tab[vis, 3]
    W, H = w.camera.width, w.camera.height
    eps = 1e-3
    assert np.all((b[:, 0] + 0.5 >= sx - R - eps) | (b[:, 0] == 0))
    assert np.all((b[:, 0] - 0.5 < sx - R + eps) | (b[:, 0] == 0))
    assert np.all((b[:, 1] + 0.5 <= sx + R + eps) | (b[:, 1] == W - 1))
    assert np.all((b[:, 1] + 1.5 > sx + R - eps) | (b[:, 1] == W - 1))
    assert np.all((b[:, 2] + 0.5 >= sy - R - eps) | (b[:, 2] == 0))
    assert np.all((b[:, 3] + 0.5 <= sy + R + eps) | (b[:, 3] == H - 1))
    # particles the table keeps but the box test drops touch no pixel centre
    dropped = (ok > 0) & ~vis
    for p in np.nonzero(dropped)[0][:200]:
        sxp, syp, Rp = tab[p, 0], tab[p, 1], tab[p, 3]
        ii = np.arange(W) + 0.5
        jj = np.arange(H) + 0.5
        nx = ii[(ii >= sxp - Rp + 1e-6) & (ii <= sxp + Rp - 1e-6)]
        ny = jj[(jj >= syp - Rp + 1e-6) & (jj <= syp + Rp - 1e-6)]
        assert len(nx) == 0 or len(ny) == 0


def test_depth_key_orders_like_depth_and_order_is_lexsort():
    w = _small("C4", 5000)
    pr = oracle.project_f32(w)
    vis = pr["visible"] > 0
    zc = pr["zkey"].view(np.float32)
    assert np.all(zc[vis] > w.z_near)
    order = oracle.depth_order(pr["zkey"], pr["visible"])
    idx = np.nonzero(vis)[0]
    expect = idx[np.lexsort((idx, pr["zkey"][idx]))]
    np.testing.assert_array_equal(order, expect)
    assert np.all(np.diff(zc[order].astype(np.float64)) >= 0)


def test_depth_order_ties_by_index():
    zkey = np.array([5, 3, 5, 3, 9, 3], np.uint32)
    vis = np.array([1, 1, 1, 0, 1, 1], np.uint8)
    np.testing.assert_array_equal(oracle.depth_order(zkey, vis), [1, 5, 0, 2, 4])


def _brute_bins(bbox, visible, W, H, shift, order=None):
    bs = 1 << shift
    nbx, nby = (W + bs - 1) >> shift, (H + bs - 1) >> shift
    lists = [[] for _ in range(nbx * nby)]
    seq = range(len(visible)) if order is None else order
    for p in seq:
        if not visible[p]:
            continue
        i0, i1, j0, j1 = bbox[p]
        for by in range(j0 // bs, j1 // bs + 1):
            for bx in range(i0 // bs, i1 // bs + 1):
                lists[by * nbx + bx].append(p)
    return lists


def test_bins_match_brute_force_index_order_and_depth_order():
    w = _small("C1", 3000, 100, 70)          # ragged: 100 and 70 are not multiples of 16
    pr = oracle.project_f32(w)
    for shift in (4, 6):
        counts, offsets, members = oracle.bins(pr["bbox"], pr["visible"], 100, 70, shift)
        lists = _brute_bins(pr["bbox"], pr["visible"], 100, 70, shift)
        assert len(counts) == len(lists)
        np.testing.assert_array_equal(counts, [len(l) for l in lists])
        np.testing.assert_array_equal(offsets, np.concatenate([[0], np.cumsum([len(l) for l in lists])]))
        for t, l in enumerate(lists):
            np.testing.assert_array_equal(members[int(offsets[t]):int(offsets[t + 1])], l)
    order = oracle.depth_order(pr["zkey"], pr["visible"])
    counts, offsets, members = oracle.bins(pr["bbox"], pr["visible"], 100, 70, 4, order=order)
    lists = _brute_bins(pr["bbox"], pr["visible"], 100, 70, 4, order=order)
    for t, l in enumerate(lists):
        np.testing.assert_array_equal(members[int(offsets[t]):int(offsets[t + 1])], l)
    assert offsets[-1] > 3000


def test_bins_single_splat_covers_exactly_its_box():
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=64, h=64)
    w = mk([(0.0, 0.0, 0.0, 0.2, 1.0, 0.0)], c)
    pr = oracle.project_f32(w)
    i0, i1, j0, j1 = pr["bbox"][0]
    counts, offsets, members = oracle.bins(pr["bbox"], pr["visible"], 64, 64, 4)
    grid = counts.reshape(4, 4)
    exp = np.zeros((4, 4), np.uint32)
    exp[j0 // 16:j1 // 16 + 1, i0 // 16:i1 // 16 + 1] = 1
    np.testing.assert_array_equal(grid, exp)
    # symmetric splat on the axis: the box is symmetric about the centre
    assert i0 + i1 == 63 and j0 + j1 == 63


def test_workload_generators_are_deterministic_and_chunk_invariant():
    a = workloads.make("C3", 300_000)
    b = workloads.make("C3", 300_000)
    for k in ("x", "y", "z", "r", "I", "colval", "type"):
        np.testing.assert_array_equal(getattr(a, k), getattr(b, k))
    # regenerate one slice by hand through the counter-based generator: same bytes
    from workloads import rng
    idx = rng.index_range(123_456, 123_466)
    np.testing.assert_array_equal(a.colval[123_456:123_466], rng.uniform(a.seed, 13, idx).astype(np.float32))
    assert a.type is not None and 0.45 < a.type.mean() < 0.55
    assert abs(np.median(a.r) / 0.005 - 1) < 0.02
