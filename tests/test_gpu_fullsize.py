"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (SURVEY.md 8(c) "Oracle
practicalities"; what is compared is the image of PAPER.md:69-75).

  C2  16M particles, 1024^2, additive : FULL FRAME against the oracle (ALU-only = the automatic choice, and tensor cores forced)
  C4  16M particles, 1024^2, absorb   : FULL FRAME against the oracle (multi-unit ordered merge, ~1e4 slabs per pixel)
  C3  100M particles, 2048^2, additive: 256 tiles of 16x16 pixels chosen BY RULE from the device's own 16x16 bin counts
                                        (64 fullest, 64 emptiest non-empty, 128 seeded random), all particles, in the three
                                        tensor modes; tensor-core and ALU-only images must also agree everywhere
  C5  400M particles, 4096^2, additive: the same 256-tile rule for two cameras of the orbit (0 and 3)

A full-frame double-precision oracle render of C3 / C5 takes tens of minutes to hours, so there the oracle computes the
sampled tiles one by one (every particle that can reach the tile, those pixels only).  Every test reports its worst
|delta| / tolerance (tolerance = 1e-4 max(1, |ref|), north_star) on stdout (pytest -s shows it).
"""
import copy
import json
import os
import time

import numpy as np
import pytest

import oracle
import workloads

pytestmark = [pytest.mark.gpu, pytest.mark.slow]

torch = pytest.importorskip("torch")
psutil = pytest.importorskip("psutil")

TILE = 16
_ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _report(**kw):
    """One line per case on stdout (run pytest with -s, or read the captured output of a failing case): a test writes
    nothing into the tree."""
    print("fullsize parity:", json.dumps(kw))


def _need(host_gb, dev_gb):
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    if psutil.virtual_memory().available < host_gb * 2 ** 30:
        pytest.skip(f"needs {host_gb} GB of free host memory")
    free, _ = torch.cuda.mem_get_info()
    if free < dev_gb * 2 ** 30:
        pytest.skip(f"needs {dev_gb} GB of free device memory")


def _worst(out, ref):
    err = np.abs(np.asarray(out, np.float64) - ref)
    return float((err / (1e-4 * np.maximum(1.0, np.abs(ref)))).max())


def _scene(w, cam=None):
    from paper_1004_1302_b200 import Scene
    sc = Scene(w)
    sc.reserve(cam)
    return sc


def _render(sc, tensor, cam=None, raw=True):
    sc.tensor = tensor
    img = sc.render(cam=cam, raw=raw).cpu().numpy()
    sc.tensor = None
    return img


# ---------------------------------------------------------------------------------------------------
# rule-chosen tiles from the device's own bin counts at 16x16 pixels (splotch_debug_bins, s = 4)
# ---------------------------------------------------------------------------------------------------
def _tile_counts(sc, cam):
    from paper_1004_1302_b200 import binding as B
    from paper_1004_1302_b200.scene import _camera_struct
    cs, ps = _camera_struct(cam), sc.params()
    nx, ny = (cam.width + TILE - 1) // TILE, (cam.height + TILE - 1) // TILE
    nbytes = B.splotch_debug_workspace_bytes(sc.n, cs, ps, 4, 0)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(nx * ny, dtype=torch.int32, device="cuda")
    off = torch.zeros(nx * ny + 1, dtype=torch.int64, device="cuda")
    B.splotch_debug_bins(sc.particles(), sc.n, cs, sc.colormap(), ps, sc._aligned(ws), nbytes, 4, cnt, off, None, 0)
    torch.cuda.synchronize()
    return cnt.cpu().numpy().view(np.uint32).reshape(ny, nx).astype(np.int64)


def _rule_tiles(counts, seed):
    """64 fullest, 64 emptiest non-empty, 128 seeded random tiles (distinct), as (tx, ty)."""
    ny, nx = counts.shape
    flat = counts.ravel()
    order = np.argsort(flat, kind="stable")
    nonempty = order[flat[order] > 0]
    assert len(nonempty) >= 256
    chosen = list(nonempty[-64:]) + list(nonempty[:64])
    taken = set(int(t) for t in chosen)
    rs = np.random.RandomState(seed)
    while len(chosen) < 256:
        t = int(rs.randint(0, nx * ny))
        if t not in taken:
            taken.add(t)
            chosen.append(t)
    return [(int(t) % nx, int(t) // nx) for t in chosen]


def _slice(w, s, e):
    sh = copy.copy(w)
    for k in ("x", "y", "z", "r", "I", "colval"):
        setattr(sh, k, getattr(w, k)[s:e])
    sh.type = None if w.type is None else w.type[s:e]
    sh.n = e - s
    return sh


def _oracle_tiles(w, cam, tiles):
    """Raw additive S of the oracle on every tile: stage 1 (oracle.splat_table) in chunks, keeping only splats whose
    disc (+1 pixel of slack) reaches a chosen tile; stage 2 (oracle.render_table) per tile on the splats that reach it."""
    nx, ny = (cam.width + TILE - 1) // TILE, (cam.height + TILE - 1) // TILE
    mark = np.zeros((ny + 1, nx + 1), np.int64)
    for tx, ty in tiles:
        mark[ty + 1, tx + 1] = 1
    sat = mark.cumsum(0).cumsum(1)                       # summed-area table of chosen tiles
    kept = []
    step = 25_000_000
    for s in range(0, w.n, step):
        tab, ok = oracle.splat_table(_slice(w, s, min(s + step, w.n)), cam, workloads.ADDITIVE)
        lo_x, hi_x = tab[:, 0] - tab[:, 3] - 1.0, tab[:, 0] + tab[:, 3] + 1.0
        lo_y, hi_y = tab[:, 1] - tab[:, 3] - 1.0, tab[:, 1] + tab[:, 3] + 1.0
        on = ok.astype(bool) & (hi_x >= 0) & (lo_x <= cam.width) & (hi_y >= 0) & (lo_y <= cam.height)
        tx0 = np.clip(np.floor(lo_x / TILE), 0, nx - 1).astype(np.int64)
        tx1 = np.clip(np.floor(hi_x / TILE), 0, nx - 1).astype(np.int64)
        ty0 = np.clip(np.floor(lo_y / TILE), 0, ny - 1).astype(np.int64)
        ty1 = np.clip(np.floor(hi_y / TILE), 0, ny - 1).astype(np.int64)
        hits = sat[ty1 + 1, tx1 + 1] - sat[ty0, tx1 + 1] - sat[ty1 + 1, tx0] + sat[ty0, tx0]
        kept.append(tab[on & (hits > 0)])
        del tab, ok
    table = np.ascontiguousarray(np.concatenate(kept))
    del kept
    lo_x, hi_x = table[:, 0] - table[:, 3] - 1.0, table[:, 0] + table[:, 3] + 1.0
    lo_y, hi_y = table[:, 1] - table[:, 3] - 1.0, table[:, 1] + table[:, 3] + 1.0
    out = {}
    for tx, ty in tiles:
        x0, y0 = tx * TILE, ty * TILE
        x1, y1 = min(x0 + TILE, cam.width), min(y0 + TILE, cam.height)
        sel = np.nonzero((hi_x >= x0) & (lo_x <= x1) & (hi_y >= y0) & (lo_y <= y1))[0]
        out[(tx, ty)] = oracle.render_table(table[sel], np.arange(len(sel)), workloads.ADDITIVE, (x0, y0, x1, y1), raw=True)
    return out, len(table)


def _check_tiles(name, images, ref_tiles, cam):
    worst = {}
    for mode, img in images.items():
        wm = 0.0
        for (tx, ty), ref in ref_tiles.items():
            x0, y0 = tx * TILE, ty * TILE
            wm = max(wm, _worst(img[y0:y0 + ref.shape[0], x0:x0 + ref.shape[1]], ref))
        worst[str(mode)] = wm
    return worst


# ---------------------------------------------------------------------------------------------------
# C2, C4: full frame
# ---------------------------------------------------------------------------------------------------
def test_c2_full_size_full_frame():
    _need(16, 12)
    t0 = time.time()
    w = workloads.make("C2")
    sc = _scene(w)
    vis, pairs, updates = sc.stats()
    assert w.n == 16_000_000 and updates > 5e10
    images = {m: _render(sc, m) for m in (None, False, True)}
    ref = oracle.render(w, raw=True)
    assert 0.8 < ref.mean() < 1.25 and ref.shape == (1024, 1024, 3)
    worst = {str(m): _worst(img, ref) for m, img in images.items()}
    mapped = _render(sc, None, raw=False)
    worst["mapped"] = _worst(mapped, -np.expm1(-ref))
    _report(config="C2", n=w.n, pixels_checked=1024 * 1024, updates=int(updates), worst_over_tol=worst, seconds=round(time.time() - t0, 1))
    assert max(worst.values()) <= 1.0, worst


def test_c4_full_size_full_frame_absorb():
    _need(16, 16)
    t0 = time.time()
    w = workloads.make("C4")
    sc = _scene(w)
    vis, pairs, updates = sc.stats()
    assert w.n == 16_000_000 and w.mode == workloads.ABSORB and updates > 5e10
    img = sc.render().cpu().numpy()
    img2 = sc.render().cpu().numpy()
    assert np.array_equal(img, img2)                       # ordered merge: a repeat call is bit-identical
    ref = oracle.render(w)
    assert ref.max() > 0.3 and ref.shape == (1024, 1024, 3)
    worst = _worst(img, ref)
    _report(config="C4", n=w.n, pixels_checked=1024 * 1024, updates=int(updates), worst_over_tol=worst,
            seconds=round(time.time() - t0, 1))
    assert worst <= 1.0, worst


# ---------------------------------------------------------------------------------------------------
# C3: 256 rule-chosen tiles, three tensor modes, tensor vs ALU everywhere
# ---------------------------------------------------------------------------------------------------
def test_c3_full_size_rule_tiles_and_both_rasterisers():
    _need(40, 24)
    t0 = time.time()
    w = workloads.make("C3")
    cam = w.camera
    sc = _scene(w)
    vis, pairs, updates = sc.stats()
    assert w.n == 100_000_000 and vis > 0.9 * w.n and pairs > 5 * vis and updates > 1e12
    images = {m: _render(sc, m) for m in (True, False, None)}          # None = what bench.py times
    # the split between tensor cores and ALUs is exact up to the order of the partial sums
    np.testing.assert_allclose(images[True], images[False], rtol=4e-5, atol=1e-5)
    np.testing.assert_allclose(images[None], images[False], rtol=4e-5, atol=1e-5)
    assert 0.8 < float(images[None].mean()) < 1.25                      # brightness is calibrated to a frame mean of 1
    tiles = _rule_tiles(_tile_counts(sc, cam), seed=1004130203)
    del sc
    torch.cuda.empty_cache()
    ref_tiles, n_kept = _oracle_tiles(w, cam, tiles)
    worst = _check_tiles("C3", images, ref_tiles, cam)
    _report(config="C3", n=w.n, tiles=len(tiles), pixels_checked=len(tiles) * TILE * TILE, splats_reaching_tiles=n_kept,
            updates=int(updates), worst_over_tol=worst, seconds=round(time.time() - t0, 1))
    assert max(worst.values()) <= 1.0, worst


def test_c3_mapped_image_is_the_map_of_the_raw_sum():
    _need(16, 24)
    w = workloads.make("C3")
    sc = _scene(w)
    raw = _render(sc, None)
    mapped = _render(sc, None, raw=False)
    np.testing.assert_allclose(mapped, -np.expm1(-raw.astype(np.float64)), rtol=0, atol=2e-5)   # 1 - exp(-S), slope <= 1


# ---------------------------------------------------------------------------------------------------
# C5: two cameras of the orbit, 256 rule-chosen tiles each
# ---------------------------------------------------------------------------------------------------
def test_c5_full_size_rule_tiles_two_cameras():
    _need(48, 60)
    t0 = time.time()
    w = workloads.make("C5")
    assert w.n == 400_000_000 and len(w.cameras) == 8
    from paper_1004_1302_b200 import Scene
    sc = Scene(w)
    for ci in (0, 3):
        cam = w.cameras[ci]
        sc.reserve(cam)
        images = {None: _render(sc, None, cam)}
        if ci == 0:
            images[True] = _render(sc, True, cam)
        tiles = _rule_tiles(_tile_counts(sc, cam), seed=1004130205 + ci)
        ref_tiles, n_kept = _oracle_tiles(w, cam, tiles)
        worst = _check_tiles("C5", images, ref_tiles, cam)
        _report(config="C5", camera=ci, n=w.n, tiles=len(tiles), pixels_checked=len(tiles) * TILE * TILE,
                splats_reaching_tiles=n_kept, worst_over_tol=worst, seconds=round(time.time() - t0, 1))
        assert max(worst.values()) <= 1.0, (ci, worst)
