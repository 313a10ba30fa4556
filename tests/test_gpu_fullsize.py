"""GPU parity at BASELINE.json's full size, in the launch configuration bench.py times (C3: 100M particles,
2048x2048, additive mode).  A full-frame double-precision oracle render of C3 takes tens of minutes, so the
oracle computes sampled rectangles of the image one by one (all particles, those pixels only), and properties
that hold at any size cover the rest: the tensor-core and the ALU-only rasteriser must agree everywhere, and
the statistics of the two front-end passes must agree with each other.
"""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
psutil = pytest.importorskip("psutil")

# pixel rectangles (x0, y0, x1, y1): image centre (densest overlap), a filament region, the sparse top-left corner
ROIS = [(960, 1016, 1216, 1032), (300, 1500, 556, 1516), (0, 0, 256, 16)]


@pytest.fixture(scope="module")
def c3():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    if psutil.virtual_memory().available < 48 * 2 ** 30:
        pytest.skip("the oracle's double table of 1e8 splats needs ~15 GB of host memory")
    free, _ = torch.cuda.mem_get_info()
    if free < 24 * 2 ** 30:
        pytest.skip("needs 24 GB of free device memory")
    from paper_1004_1302_b200 import Scene
    w = workloads.make("C3")
    sc = Scene(w)
    vis, pairs, updates = sc.stats()
    sc.reserve(max_pairs=pairs + 1024)
    return w, sc, (vis, pairs, updates)


def _within(out, ref):
    err = np.abs(np.asarray(out, np.float64) - ref)
    return float((err / (1e-4 * np.maximum(1.0, np.abs(ref)))).max())


def test_c3_full_size_sampled_pixels_and_both_rasterisers(c3):
    w, sc, (vis, pairs, updates) = c3
    assert w.n == 100_000_000 and vis > 0.9 * w.n and pairs > 5 * vis and updates > 1e12
    images = {}
    for tensor in (True, False):
        sc.tensor = tensor
        images[tensor] = sc.render(raw=True).cpu().numpy()
    sc.tensor = None
    images[None] = sc.render(raw=True).cpu().numpy()          # what bench.py times
    # the split between tensor cores and ALUs is exact up to the order of the partial sums
    np.testing.assert_allclose(images[True], images[False], rtol=4e-5, atol=1e-5)
    np.testing.assert_allclose(images[None], images[False], rtol=4e-5, atol=1e-5)
    assert 0.8 < float(images[None].mean()) < 1.25             # brightness is calibrated to a frame mean of 1
    for roi in ROIS:
        ref = oracle.render(w, raw=True, roi=roi)
        x0, y0, x1, y1 = roi
        for tensor, img in images.items():
            worst = _within(img[y0:y1, x0:x1], ref)
            assert worst <= 1.0, f"C3 full size, roi {roi}, tensor={tensor}: worst |delta| / tol = {worst:.3f}"
    # the mapped image of the default path: 1 - exp(-S), slope <= 1
    mapped = sc.render(raw=False).cpu().numpy()
    np.testing.assert_allclose(mapped, -np.expm1(-images[None].astype(np.float64)), rtol=0, atol=2e-5)
