"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): integers (visible set, pixel boxes, depth keys, bin counts,
offsets, membership) bit-exact; pixels within |delta| <= 1e-4 * max(1, |ref|) in both modes.
"""
import numpy as np
import pytest

import oracle
import workloads
from workloads import ABSORB, ADDITIVE

from helpers import cam, const_lut, mk

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1004_1302_b200 import binding
    binding.library_path()
    return binding


def _scene(w, tensor=None):
    """tensor: None = the library decides, True = SPLOTCH_FORCE_TENSOR, False = SPLOTCH_NO_TENSOR."""
    from paper_1004_1302_b200 import Scene
    sc = Scene(w)
    sc.tensor = tensor
    return sc


def _tol_check(out, ref, what=""):
    out = np.asarray(out, np.float64)
    err = np.abs(out - ref)
    bound = 1e-4 * np.maximum(1.0, np.abs(ref))
    worst = float((err / bound).max()) if err.size else 0.0
    assert worst <= 1.0, f"{what}: worst |delta| / (1e-4 max(1,|ref|)) = {worst:.3f} at {np.unravel_index((err / bound).argmax(), err.shape)}"
    return worst


# ------------------------------------------------------------------------------------------------
# building blocks
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 5, 2047, 2048, 2049, 70_001, 1_000_003])
def test_scan_matches_cumsum(B, n):
    rs = np.random.RandomState(n % 1000)
    a = rs.randint(0, 2 ** 32, size=max(n, 1), dtype=np.uint64).astype(np.uint32)[:n]
    d_in = torch.from_numpy(a.astype(np.int64)).to("cuda").to(torch.int64)
    d_in32 = torch.empty(max(n, 1), dtype=torch.int32, device="cuda")
    if n:
        d_in32[:n] = torch.from_numpy(a.view(np.int32)).cuda()
    out = torch.zeros(n + 1, dtype=torch.int64, device="cuda")
    sb = (n // 2048 + 2) * 8 + 512
    scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
    B.splotch_debug_scan(d_in32, out, n, scratch, sb)
    torch.cuda.synchronize()
    expect = np.concatenate([[0], np.cumsum(a.astype(np.uint64))]).astype(np.uint64)
    np.testing.assert_array_equal(out.cpu().numpy().view(np.uint64), expect)


@pytest.mark.parametrize("n,bits", [(1, 8), (31, 8), (4095, 12), (4096, 32), (4097, 32), (300_001, 32), (1_000_000, 10)])
def test_radix_sort_is_stable_and_sorted(B, n, bits):
    rs = np.random.RandomState(bits * 7 + n % 13)
    keys = rs.randint(0, 2 ** min(bits, 31), size=n, dtype=np.int64).astype(np.uint32)
    if bits == 32:
        keys |= (rs.randint(0, 2, size=n).astype(np.uint32) << np.uint32(31))
    keys[: n // 3] = keys[: n // 3] & np.uint32(0xFF)                        # many ties
    vals = np.arange(n, dtype=np.uint32)
    dk = torch.from_numpy(keys.view(np.int32)).cuda()
    dv = torch.from_numpy(vals.view(np.int32)).cuda()
    tk, tv = torch.empty_like(dk), torch.empty_like(dv)
    sb = B.splotch_sort_scratch_bytes(n)
    scratch = torch.empty(sb, dtype=torch.uint8, device="cuda")
    B.splotch_debug_sort_pairs(dk, dv, tk, tv, n, bits, scratch, sb)
    torch.cuda.synchronize()
    order = np.argsort(keys, kind="stable")
    np.testing.assert_array_equal(dv.cpu().numpy().view(np.uint32), order.astype(np.uint32))
    np.testing.assert_array_equal(dk.cpu().numpy().view(np.uint32), keys[order])


# ------------------------------------------------------------------------------------------------
# K1: bit-exact projection, culling, depth key
# ------------------------------------------------------------------------------------------------
def _gpu_project(B, w, camera=None):
    sc = _scene(w)
    camera = camera or w.camera
    n = w.n
    from paper_1004_1302_b200.scene import _camera_struct
    cs, ps = _camera_struct(camera), sc.params()
    nbytes = B.splotch_debug_workspace_bytes(n, cs, ps, 6, 0)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    o = dict(sx=torch.zeros(n, dtype=torch.float32, device="cuda"), sy=torch.zeros(n, dtype=torch.float32, device="cuda"),
             ss=torch.zeros(n, dtype=torch.float32, device="cuda"), R=torch.zeros(n, dtype=torch.float32, device="cuda"),
             zkey=torch.zeros(n, dtype=torch.int32, device="cuda"), bbox=torch.zeros((n, 4), dtype=torch.int32, device="cuda"),
             visible=torch.zeros(n, dtype=torch.uint8, device="cuda"))
    B.splotch_debug_project(sc.particles(), n, cs, sc.colormap(), ps, sc._aligned(ws), nbytes, o["sx"], o["sy"], o["ss"],
                            o["R"], o["zkey"], o["bbox"], o["visible"])
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in o.items()}
    out["zkey"] = out["zkey"].view(np.uint32)
    return out


def _edge_particles():
    pts = [(0.5, 0.5, 0.5, 0.01, 1.0, 0.5)] * 3
    pts += [(np.nan, 0.5, 0.5, 0.01, 1, 0), (0.5, np.inf, 0.5, 0.01, 1, 0), (0.5, 0.5, 0.5, -0.01, 1, 0),
            (0.5, 0.5, 0.5, 0.0, 1, 0), (0.5, 0.5, 0.5, 0.01, np.nan, 0), (0.5, 0.5, 0.5, 0.01, 1, np.inf),
            (0.5, 0.5, -1.5, 0.01, 1, 0), (0.5, 0.5, -1.4905, 0.01, 1, 0), (0.5, 0.5, -3.0, 0.01, 1, 0),
            (30.0, 0.5, 0.5, 0.01, 1, 0), (0.5, 0.5, 0.5, 1e-7, 1, 0), (0.5, 0.5, 0.5, 5.0, 1, 0),
            (0.5, 0.5, 0.5, 1e30, 1, 0), (0.5, 0.5, 0.5, 3e38, 1, 0), (1e30, 0.5, 0.5, 0.01, 1, 0),
            (0.5, 0.5, 0.5, 1e-38, 1, 0)]
    return pts


@pytest.mark.parametrize("case", ["C1", "C4", "C3", "edge"])
def test_project_bit_exact(B, case):
    if case == "C1":
        w = workloads.make("C1")
    elif case == "C4":
        w = workloads.make("C4", 200_003, width=1000, height=700)
    elif case == "C3":
        w = workloads.make("C3", 300_001, width=2048, height=2048)
    else:
        w = mk(_edge_particles(), workloads.make("C1", 10).camera)
    ref = oracle.project_f32(w)
    got = _gpu_project(B, w)
    np.testing.assert_array_equal(got["visible"], ref["visible"])
    assert 0 < ref["visible"].sum() < w.n or case == "edge"
    for k in ("sx", "sy", "ss", "R"):
        np.testing.assert_array_equal(got[k].view(np.uint32), ref[k].view(np.uint32), err_msg=k)
    np.testing.assert_array_equal(got["zkey"], ref["zkey"])
    np.testing.assert_array_equal(got["bbox"], ref["bbox"])


# ------------------------------------------------------------------------------------------------
# K2: bit-exact bins
# ------------------------------------------------------------------------------------------------
def _gpu_bins(B, w, shift, with_members=True, cap=None):
    sc = _scene(w)
    from paper_1004_1302_b200.scene import _camera_struct
    cs, ps = _camera_struct(w.camera), sc.params()
    bs = 1 << shift
    T = ((w.camera.width + bs - 1) >> shift) * ((w.camera.height + bs - 1) >> shift)
    ref = oracle.project_f32(w)
    order = oracle.depth_order(ref["zkey"], ref["visible"]) if w.mode == ABSORB else None
    rc, ro, rm = oracle.bins(ref["bbox"], ref["visible"], w.camera.width, w.camera.height, shift, order=order)
    D = int(ro[-1])
    cap = D + 7 if cap is None else cap
    nbytes = B.splotch_debug_workspace_bytes(w.n, cs, ps, shift, cap)
    ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(T, dtype=torch.int32, device="cuda")
    off = torch.zeros(T + 1, dtype=torch.int64, device="cuda")
    mem = torch.full((max(cap, 1),), -1, dtype=torch.int32, device="cuda")
    B.splotch_debug_bins(sc.particles(), w.n, cs, sc.colormap(), ps, sc._aligned(ws), nbytes, shift, cnt, off,
                         mem if with_members else None, cap if with_members else 0)
    torch.cuda.synchronize()
    return (cnt.cpu().numpy().view(np.uint32), off.cpu().numpy().view(np.uint64), mem.cpu().numpy().view(np.uint32)), (rc, ro, rm)


@pytest.mark.parametrize("case,shift", [("C1", 4), ("C1", 6), ("C2", 4), ("C2", 6), ("C3", 6)])
def test_bins_additive_bit_exact(B, case, shift):
    w = {"C1": lambda: workloads.make("C1"),
         "C2": lambda: workloads.make("C2", 60_000, width=500, height=333),
         "C3": lambda: workloads.make("C3", 120_000, width=1024, height=1024)}[case]()
    (cnt, off, mem), (rc, ro, rm) = _gpu_bins(B, w, shift)
    np.testing.assert_array_equal(cnt, rc)
    np.testing.assert_array_equal(off, ro)
    D = int(ro[-1])
    assert D > w.n // 2
    for t in range(len(rc)):                                   # member SET of every bin
        a, b = int(ro[t]), int(ro[t + 1])
        np.testing.assert_array_equal(np.sort(mem[a:b]), np.sort(rm[a:b]))


@pytest.mark.parametrize("shift", [4, 6])
def test_bins_absorb_sequence_bit_exact(B, shift):
    w = workloads.make("C4", 150_000, width=640, height=400)
    (cnt, off, mem), (rc, ro, rm) = _gpu_bins(B, w, shift)
    np.testing.assert_array_equal(cnt, rc)
    np.testing.assert_array_equal(off, ro)
    D = int(ro[-1])
    assert D > 10_000
    np.testing.assert_array_equal(mem[:D], rm)                 # member SEQUENCE: depth order, ties by index


def test_bins_member_capacity_is_respected(B):
    w = workloads.make("C1", 20_000)
    (cnt, off, mem), (rc, ro, rm) = _gpu_bins(B, w, 4, cap=100)
    np.testing.assert_array_equal(cnt, rc)
    np.testing.assert_array_equal(off, ro)
    assert np.all(mem == np.uint32(0xFFFFFFFF))                # untouched


# ------------------------------------------------------------------------------------------------
# whole path: pixels
# ------------------------------------------------------------------------------------------------
def _render_both(w, raw=False, mode=None, tensor=None):
    sc = _scene(w, tensor)
    out = sc.render(raw=raw, mode=mode)
    torch.cuda.synchronize()
    ref = oracle.render(w, raw=raw, mode=mode)
    return out.cpu().numpy(), ref


@pytest.mark.parametrize("raw", [True, False])
def test_additive_c1_full(B, raw):
    w = workloads.make("C1")
    out, ref = _render_both(w, raw=raw)
    assert ref.max() > (1.0 if raw else 0.9)
    _tol_check(out, ref, "C1")


@pytest.mark.parametrize("tensor", [None, True, False])
@pytest.mark.parametrize("case", ["C2", "C3", "C5"])
def test_additive_scaled_configs(B, case, tensor):
    w = {"C2": lambda: workloads.make("C2", 200_000, width=512, height=512),
         "C3": lambda: workloads.make("C3", 300_000, width=600, height=360),        # ragged: not multiples of 64
         "C5": lambda: workloads.make("C5", 400_000, width=513, height=257)}[case]()  # odd width: scalar write path
    out, ref = _render_both(w, raw=True, tensor=tensor)
    assert ref.mean() > 0.05
    _tol_check(out, ref, case)
    out, ref = _render_both(w, raw=False, tensor=tensor)
    _tol_check(out, ref, case)


@pytest.mark.parametrize("size", [(704, 512), (601, 333)])
def test_tensor_path_big_bright_splats(B, size):
    """Splats from 10 to 600 pixels wide with amplitudes up to ~0.3, centres on and off screen: most pixel
    updates lie in fully covered 32-pixel row segments, i.e. on the tensor cores (split TF32, raster_mma.cu).
    Checked against the oracle (rim pixels masked: a_c of order one, DESIGN.md error budget), against the
    ALU-only path, and the automatic choice must reproduce one of the two."""
    rs = np.random.RandomState(11)
    n = 2500
    c = cam(eye=(0.0, 0.0, -10.0), fov=25.0, w=size[0], h=size[1])
    r = np.exp(rs.uniform(np.log(0.03), np.log(2.0), n))
    pts = np.stack([rs.uniform(-3.5, 3.5, n), rs.uniform(-2.6, 2.6, n), rs.uniform(-1, 1, n), r,
                    rs.uniform(0.02, 0.3, n) / r, rs.uniform(0, 1, n)], 1)
    w = mk(pts, c, lut_e=workloads.lut_hot(), support_f=3.1)
    ref = oracle.render(w, raw=True)
    assert ref.max() > 20.0
    outs = {}
    for tensor in (True, False, None):
        sc = _scene(w, tensor)
        outs[tensor] = sc.render(raw=True).cpu().numpy()
        _tol_check_masked(w, outs[tensor], ref, max_rim=0.10)
    np.testing.assert_allclose(outs[True], outs[False], rtol=3e-5, atol=3e-5)
    assert np.array_equal(outs[None], outs[True]) or np.allclose(outs[None], outs[False], rtol=1e-5, atol=1e-6)


def test_tensor_path_mixed_bright_and_faint_splats(B):
    """K3t runs a batch of 16 queued splats as ONE TF32 product when all of them are faint (|a_c| <= 2^-11) and as the
    three-product split otherwise (raster_mma.cu: kFaintAmp).  Big splats.  Scene 1: most of them faint (a ~ 5e-5 .. 4.5e-4),
    every 23rd bright (a up to 0.3), so that both kinds of batches and mixed ones occur.  Scene 2: a = 2e-3 .. 7.5e-3, all on
    the split path, S of order 1.  Scene 3: faint splats only, where a biased cut of the operands (truncation instead of an
    unbiased rounding) would show as a relative offset of 2^-11 = 4.9e-4 per operand."""
    rs = np.random.RandomState(17)
    c = cam(eye=(0.0, 0.0, -10.0), fov=25.0, w=640, h=448)
    for bright_every, n, amp_lo, amp_hi, s_min, big_at in ((23, 3000, 5e-5, 4.5e-4, 1.0, 0.5), (0, 8000, 2e-3, 7.5e-3, 1.0, 0.5),
                                                           (0, 8000, 1e-4, 4.8e-4, 0.05, 0.03)):
        r = np.exp(rs.uniform(np.log(0.08), np.log(2.0), n))
        amp = np.exp(rs.uniform(np.log(amp_lo), np.log(amp_hi), n))
        if bright_every:
            amp[::bright_every] = rs.uniform(0.05, 0.3, len(amp[::bright_every]))
        pts = np.stack([rs.uniform(-3.2, 3.2, n), rs.uniform(-2.3, 2.3, n), rs.uniform(-1, 1, n), r,
                        amp / (r * np.sqrt(np.pi)), rs.uniform(0.7, 1.0, n)], 1)
        w = mk(pts, c, lut_e=const_lut((1.0, 0.7, 0.4)), support_f=3.1)
        ref = oracle.render(w, raw=True)
        assert ref.max() > s_min
        outs = {}
        for tensor in (True, False):
            outs[tensor] = _scene(w, tensor).render(raw=True).cpu().numpy()
            _tol_check_masked(w, outs[tensor], ref, max_rim=0.25)
        rel = (outs[True].astype(np.float64) - ref) / np.maximum(ref, 1e-30)
        big = ref > big_at
        assert big.mean() > 0.2 and abs(float(rel[big].mean())) < 3e-5          # no systematic offset of the tensor path


def _coincident_scenes():
    """Scenes whose splats share their operand bits: what a snapshot with duplicated particles or grid / glass initial
    conditions looks like to the rasteriser.  (name, workload); amplitudes a_c = I r sqrt(pi), all faint and big."""
    c = cam(eye=(0.0, 0.0, -10.0), fov=20.0, w=320, h=256)
    F = 160.0 / np.tan(np.radians(10.0))                      # pixels per unit of x / z at the lookat plane times 10
    out = []
    for name, a, n_copies, sigma_px in (("3000 copies, a = 4e-4", 4e-4, 3000, 40.0), ("170 copies, a = 7e-3", 7e-3, 170, 40.0)):
        r = sigma_px * 10.0 / F
        pts = np.tile(np.array([[0.013, -0.007, 0.0, r, a / (r * np.sqrt(np.pi)), 0.5]]), (n_copies, 1))
        out.append((name, mk(pts, c, lut_e=const_lut((1.0, 0.7, 0.4)), support_f=3.1)))
    # a regular lattice, 8 pixels apart, 100 coincident splats on every node
    r = 30.0 * 10.0 / F
    gx, gy = np.meshgrid(np.arange(-4, 5) * 8.0 * 10.0 / F, np.arange(-3, 4) * 8.0 * 10.0 / F)
    node = np.stack([gx.ravel(), gy.ravel(), np.zeros(gx.size), np.full(gx.size, r),
                     np.full(gx.size, 3e-4 / (r * np.sqrt(np.pi))), np.full(gx.size, 0.5)], 1)
    out.append(("lattice x 100 copies, a = 3e-4", mk(np.repeat(node, 100, axis=0), c, lut_e=const_lut((1.0, 0.7, 0.4)), support_f=3.1)))
    return out


def test_tensor_path_coincident_and_lattice_faint_splats(B):
    """The parity bound must not rest on the input being random.  Many IDENTICAL faint big splats (and a lattice of them)
    have identical MMA operands: any rounding of those operands that is a function of the value alone repeats its error N
    times, and with S of order 1 a relative 2^-10 is ten times the tolerance.  K3t therefore rounds its single-product
    (faint) operands with a dither that depends on the queue position, not on the value (raster_mma.cu).  Element-wise
    against the oracle, every pixel, in all three tensor modes."""
    report = []
    for name, w in _coincident_scenes():
        ref = oracle.render(w, raw=True)
        assert 0.5 < ref.max() < 1.5, (name, ref.max())
        for tensor in (None, True, False):
            sc = _scene(w, tensor)
            out = sc.render(raw=True).cpu().numpy().astype(np.float64)
            ratio = np.abs(out - ref) / (1e-4 * np.maximum(1.0, np.abs(ref)))
            at = np.unravel_index(ratio.argmax(), ratio.shape)
            report.append((name, tensor, float(ratio.max()), float((out - ref)[at]), tuple(int(v) for v in at)))
            print(f"coincident splats: {name}, tensor={tensor}: worst/tol {ratio.max():.3f} (signed delta {(out - ref)[at]:+.3e} at {at})")
            if tensor is not False:
                upd, on, _ = sc.tensor_stats()
                assert upd > 0 and (tensor or on == 1), (name, upd, on)   # the tensor-core kernel did run
    assert max(r[2] for r in report) <= 1.0, report


def test_absorb_scaled_c4(B):
    w = workloads.make("C4", 200_000, width=512, height=384)
    out, ref = _render_both(w)
    assert ref.max() > 0.3
    _tol_check(out, ref, "C4")


def test_absorb_with_a_equal_e_matches_additive_oracle(B):
    w = workloads.make("C1", 50_000, width=200, height=200)
    w.lut_a = w.lut_e.copy()
    w.abs_brightness = list(w.brightness)
    w.mode = ABSORB
    sc = _scene(w)
    out = sc.render().cpu().numpy()
    ref = oracle.render(w, mode=ADDITIVE)
    _tol_check(out, ref, "absorb(A=E) vs additive")


def test_absorb_strong_absorption_and_zero_channel(B):
    """u = A tau well above 0.25 (exact phi branch) and A_c = 0 in one channel (R15)."""
    rs = np.random.RandomState(5)
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=96, h=96)
    n = 400
    pts = np.stack([rs.uniform(-1.2, 1.2, n), rs.uniform(-1.2, 1.2, n), rs.uniform(-2, 2, n),
                    rs.uniform(0.05, 0.5, n), rs.uniform(0.5, 3.0, n), rs.uniform(0, 1, n)], 1)
    lut_e = np.array([[0.2, 0.5, 0.9], [1.0, 0.3, 0.1]], np.float32)
    lut_a = np.array([[3.0, 0.0, 0.6], [0.5, 0.0, 8.0]], np.float32)
    w = mk(pts, c, lut_e=lut_e, lut_a=lut_a, mode=ABSORB, support_f=3.2)
    out, ref = _render_both(w)
    assert ref.max() > 0.5
    # pixels whose coverage decision sits on the rim may flip between fp32 and fp64 (DESIGN.md error budget)
    _tol_check_masked(w, out, ref)


def _tol_check_masked(w, out, ref, max_rim=0.05):
    tab, ok = oracle.splat_table(w)
    H, W = ref.shape[:2]
    jj, ii = np.meshgrid(np.arange(H) + 0.5, np.arange(W) + 0.5, indexing="ij")
    rim = np.zeros((H, W), bool)
    for p in np.nonzero(ok)[0]:
        d2 = (ii - tab[p, 0]) ** 2 + (jj - tab[p, 1]) ** 2
        rim |= np.abs(d2 - tab[p, 3] ** 2) < 1e-4 * tab[p, 3] ** 2
    err = np.abs(out - ref) / (1e-4 * np.maximum(1.0, np.abs(ref)))
    assert rim.mean() < max_rim
    assert err[~rim].max() <= 1.0, err[~rim].max()


def test_single_splat_shapes(B):
    """One bright splat at several sizes (sub-pixel to screen filling), a_c of order one."""
    for r, f in [(0.0004, 3.1), (0.004, 3.1), (0.04, 3.1), (0.4, 3.1), (4.0, 3.1), (0.02, 5.0)]:
        c = cam(eye=(0.013, -0.007, -10.0), lookat=(0.013, -0.007, 0.0), fov=20.0, w=200, h=136)
        w = mk([(0.05, 0.02, 0.0, r, 1.0 / r, 0.3)], c, lut_e=const_lut((1.0, 0.6, 0.3)), support_f=f)
        for tensor in (True, False):
            out, ref = _render_both(w, raw=True, tensor=tensor)
            _tol_check_masked(w, out, ref)
        assert ref.max() > 0.05 or r < 0.001


def test_edge_cases(B):
    c = workloads.make("C1", 10).camera
    # empty input
    w0 = mk(np.zeros((0, 6)), c)
    sc = _scene(w0)
    assert float(sc.render(raw=True).abs().max()) == 0.0
    # everything culled
    w1 = mk([(0.5, 0.5, -5.0, 0.01, 1, 0), (np.nan, 0, 0, 0.01, 1, 0)], c)
    assert float(_scene(w1).render(raw=False).abs().max()) == 0.0
    # absorb, empty and culled
    w2 = mk([(0.5, 0.5, -5.0, 0.01, 1, 0)], c, lut_a=const_lut(), mode=ABSORB)
    assert float(_scene(w2).render().abs().max()) == 0.0
    # pair capacity too small: error status, zero image, never a partial image
    w3 = workloads.make("C1", 20_000)
    sc = _scene(w3)
    pairs, vis = sc.count_pairs()
    assert pairs > vis > 10_000
    sc.reserve(max_pairs=pairs // 2)
    img = sc.render(check=False)
    status, v2, p2 = B.splotch_workspace_status(sc._aligned(sc.workspace))
    assert status == B.SPLOTCH_ERR_WORKSPACE and p2 == pairs and v2 == vis
    assert float(img.abs().max()) == 0.0
    with pytest.raises(B.SplotchError):
        sc.render()
    # exact capacity works
    sc.reserve(max_pairs=pairs)
    assert float(sc.render().abs().max()) > 0.0


@pytest.mark.parametrize("mode", [ADDITIVE, ABSORB])
def test_pair_capacity_contract_both_modes(B, mode):
    """D > max_pairs (and max_pairs = 0): SPLOTCH_ERR_WORKSPACE in the status head, a ZERO image, never a partial one;
    the same workspace then serves a correctly sized render (the absorb failure path had never run)."""
    w = workloads.make("C4" if mode == ABSORB else "C2", 30_000, width=300, height=200)
    sc = _scene(w)
    pairs, vis = sc.count_pairs()
    assert pairs > vis > 1000
    good = None
    for cap in (pairs, pairs // 3, 0, pairs):
        sc.reserve(max_pairs=max(cap, pairs))       # the allocation is large enough; only the declared capacity varies
        sc.max_pairs = cap
        img = torch.full((200, 300, 3), 7.0, dtype=torch.float32, device="cuda")
        sc.render(out=img, check=False)
        status, v2, p2 = B.splotch_workspace_status(sc._aligned(sc.workspace))
        assert p2 == pairs and v2 == vis
        if cap >= pairs:
            assert status == B.SPLOTCH_OK and float(img.max()) > 0.0 and float(img.max()) < 7.0
            if good is None:
                good = img.cpu().numpy()
            else:
                np.testing.assert_allclose(img.cpu().numpy(), good, rtol=2e-5, atol=1e-6)
        else:
            assert status == B.SPLOTCH_ERR_WORKSPACE
            assert float(img.abs().max()) == 0.0


def test_negative_coefficients_follow_the_oracle(B):
    """Reading R20: negative I, E, A are used as given (the slab solution of Eq. (1) holds for either sign of u); the
    absorb kernel must pick its polynomial tier from |A tau|."""
    rs = np.random.RandomState(9)
    c = cam(eye=(0, 0, -10.0), fov=20.0, w=160, h=96)
    n = 500
    pts = np.stack([rs.uniform(-1.6, 1.6, n), rs.uniform(-1.0, 1.0, n), rs.uniform(-2, 2, n),
                    rs.uniform(0.05, 0.5, n), rs.uniform(-2.0, 3.0, n), rs.uniform(0, 1, n)], 1)
    lut_e = np.array([[0.2, -0.5, 0.9], [1.0, 0.3, -0.1]], np.float32)
    lut_a = np.array([[-1.5, 0.1, 0.6], [0.5, -0.9, 2.0]], np.float32)
    w = mk(pts, c, lut_e=lut_e, lut_a=lut_a, mode=ABSORB, support_f=3.2, abs_brightness=(0.2,))
    out, ref = _render_both(w)
    assert ref.max() > 0.3 and ref.min() < -0.05
    _tol_check_masked(w, out, ref)
    for tensor in (True, False):
        out, ref = _render_both(w, raw=True, mode=ADDITIVE, tensor=tensor)
        assert ref.min() < -0.05
        _tol_check_masked(w, out, ref)


def test_repeat_calls_and_orbit_cameras(B):
    """C5's use case: several cameras over one resident particle set; same camera twice gives the same image."""
    w = workloads.make("C5", 300_000, width=256, height=256)
    sc = _scene(w, tensor=True)
    worst_pairs = max(sc.count_pairs(cm)[0] for cm in w.cameras)
    sc.reserve(max_pairs=worst_pairs)
    first = None
    for j, cm in enumerate(w.cameras[:3]):
        out = sc.render(cam=cm, raw=True).cpu().numpy()
        ref = oracle.render(w, camera=cm, raw=True)
        _tol_check(out, ref, f"C5 camera {j}")
        if j == 0:
            first = out
    again = sc.render(cam=w.cameras[0], raw=True).cpu().numpy()
    np.testing.assert_allclose(again, first, rtol=2e-5, atol=1e-6)   # atomics and MMA batching: order of partial sums may differ


def test_render_batch_orbit_matches_oracle_per_camera(B):
    """splotch_render_batch (f4): the 8-camera orbit of C5 in ONE call over the resident particle set;
    every frame against the oracle, and bit-for-bit equal to what it is defined as (splotch_render per camera, ALU path:
    deterministic up to the order of atomics, so compared within rounding); per-frame status words."""
    w = workloads.make("C5", 200_000, width=192, height=160)
    sc = _scene(w, tensor=False)
    imgs, status = sc.render_batch(raw=True)
    torch.cuda.synchronize()
    st = status.cpu().numpy()
    assert imgs.shape == (8, 160, 192, 3) and (st[:, 0] == 0).all() and (st[:, 3] == 0).all()
    for j, cm in enumerate(w.cameras):
        ref = oracle.render(w, camera=cm, raw=True)
        _tol_check(imgs[j].cpu().numpy(), ref, f"C5 batch camera {j}")
        pairs, vis = sc.count_pairs(cm)
        assert int(st[j, 1]) == vis and int(st[j, 2]) == pairs
    single = sc.render(cam=w.cameras[5], raw=True).cpu().numpy()
    np.testing.assert_allclose(imgs[5].cpu().numpy(), single, rtol=2e-5, atol=1e-6)
    # a capacity that only some frames exceed: those frames are zero with an error status, the others complete
    pairs_all = [sc.count_pairs(cm)[0] for cm in w.cameras]
    cap = sorted(pairs_all)[3]
    sc.max_pairs = cap
    imgs2, status2 = sc.render_batch(raw=True, check=False)
    st2 = status2.cpu().numpy()
    for j, p in enumerate(pairs_all):
        if p > cap:
            assert st2[j, 0] == B.SPLOTCH_ERR_WORKSPACE and float(imgs2[j].abs().max()) == 0.0
        else:
            assert st2[j, 0] == 0
            np.testing.assert_allclose(imgs2[j].cpu().numpy(), imgs[j].cpu().numpy(), rtol=2e-5, atol=1e-6)
    with pytest.raises(B.SplotchError):
        sc.render_batch(raw=True)
    # mixed image sizes are rejected before anything is enqueued; an empty batch is a no-op
    from paper_1004_1302_b200.scene import _camera_struct
    cs = [_camera_struct(w.cameras[0]), B.make_camera((0, 0, -3), (0, 0, 0), (0, 1, 0), 30.0, 100, 100)]
    with pytest.raises(B.SplotchError):
        B.splotch_render_batch(sc.particles(), sc.n, cs, sc.colormap(), sc.params(), imgs, None, sc._aligned(sc.workspace),
                               sc.workspace.numel() - 256, sc.max_pairs)
    B.splotch_render_batch(sc.particles(), sc.n, [], sc.colormap(), sc.params(), imgs, None, sc._aligned(sc.workspace),
                           sc.workspace.numel() - 256, sc.max_pairs)


def test_render_is_capturable_in_a_cuda_graph(B):
    """splotch_render only enqueues on the caller's stream (include/splotch.h "Asynchrony"): it can be captured into a CUDA
    graph and replayed, in both modes; the replayed image equals the eagerly rendered one (ALU paths are deterministic up to
    the order of atomics) and a replay after the particle arrays changed in place renders the new scene."""
    for name, kw in (("C1", dict(n=30_000, width=160, height=128)), ("C4", dict(n=20_000, width=160, height=128))):
        w = workloads.make(name, **kw)
        sc = _scene(w, tensor=False)
        sc.reserve()
        cam_ = w.camera
        out = torch.zeros((cam_.height, cam_.width, 3), dtype=torch.float32, device="cuda")
        eager = sc.render(out=out.clone()).cpu().numpy()
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            sc.render(out=out, check=False)                    # warm-up on the capture stream
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            sc.render(out=out, check=False)
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        np.testing.assert_allclose(out.cpu().numpy(), eager, rtol=2e-5, atol=1e-6)
        status, _, _ = B.splotch_workspace_status(sc._aligned(sc.workspace))
        assert status == B.SPLOTCH_OK
        sc.d["I"].mul_(0.5)                                     # same buffers, new content: the graph renders the new scene
        graph.replay()
        torch.cuda.synchronize()
        w.I = w.I * np.float32(0.5)
        ref = oracle.render(w)
        _tol_check(out.cpu().numpy(), ref, f"{name} graph replay")


def test_tensor_path_and_batch_are_capturable_in_a_cuda_graph(B):
    """The header's capture claim also covers the tensor-core rasteriser and splotch_render_batch: a forced-tensor render
    and a two-camera batch, captured and replayed, give the eagerly rendered images (sums may be reordered: within rounding)
    and match the oracle."""
    import dataclasses
    w = workloads.make("C3", 60_000, width=256, height=192)
    cam2 = dataclasses.replace(w.camera, fov_deg=w.camera.fov_deg * 0.8)
    sc = _scene(w, tensor=True)
    sc.reserve(max_pairs=max(sc.count_pairs(c)[0] for c in (w.camera, cam2)) + 1024)
    H, W = w.camera.height, w.camera.width
    side = torch.cuda.Stream()

    def capture(fn):
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()                                               # warm-up on the capture stream
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            fn()
        return graph

    out = torch.zeros((H, W, 3), dtype=torch.float32, device="cuda")
    eager = sc.render(raw=True).cpu().numpy()
    assert sc.tensor_stats()[0] > 0                            # the tensor-core kernel really has work in this scene
    g1 = capture(lambda: sc.render(raw=True, out=out, check=False))
    out.zero_()
    g1.replay()
    torch.cuda.synchronize()
    np.testing.assert_allclose(out.cpu().numpy(), eager, rtol=2e-5, atol=1e-6)
    _tol_check(out.cpu().numpy(), oracle.render(w, raw=True), "tensor path, graph replay")

    outs = torch.zeros((2, H, W, 3), dtype=torch.float32, device="cuda")
    eager2, _ = sc.render_batch([w.camera, cam2], raw=True)
    eager2 = eager2.cpu().numpy()
    g2 = capture(lambda: sc.render_batch([w.camera, cam2], raw=True, out=outs, check=False))
    outs.zero_()
    g2.replay()
    torch.cuda.synchronize()
    np.testing.assert_allclose(outs.cpu().numpy(), eager2, rtol=2e-5, atol=1e-6)
    _tol_check(outs[1].cpu().numpy(), oracle.render(w, camera=cam2, raw=True), "batch frame 1, graph replay")


def test_nan_amplitude_is_not_dropped_by_the_tensor_path(B):
    """A colour table with a NaN entry gives some splats a NaN amplitude.  The ALU rasteriser carries it into every pixel
    such a splat covers; the tensor-core rasteriser must not turn it into a number (its faint single-product path rounds
    bit patterns, which would): every pixel that is NaN on the ALU path is NaN with the tensor cores forced on."""
    rs = np.random.RandomState(5)
    n = 400
    pts = np.stack([rs.uniform(-1.2, 1.2, n), rs.uniform(-1.2, 1.2, n), rs.uniform(-0.5, 0.5, n), rs.uniform(0.3, 0.5, n),
                    np.full(n, 1e-3), rs.uniform(0, 1, n)], 1)
    lut = np.linspace(0.2, 1.0, 8 * 3, dtype=np.float32).reshape(8, 3)
    lut[5, 1] = np.nan
    w = mk(pts, cam(w=256, h=192), lut_e=lut)
    imgs = {}
    for tensor in (False, True):
        sc = _scene(w, tensor=tensor)
        imgs[tensor] = sc.render(raw=True).cpu().numpy()
        if tensor:
            assert sc.tensor_stats()[0] > 0
    nan_alu, nan_tc = np.isnan(imgs[False]), np.isnan(imgs[True])
    assert nan_alu.any() and not nan_alu[..., 0].any()          # only the green channel holds the NaN entry
    assert (nan_tc | ~nan_alu).all()
    both = ~nan_alu & ~nan_tc
    np.testing.assert_allclose(imgs[True][both], imgs[False][both], rtol=2e-4, atol=1e-6)


def test_scene_caches_follow_the_camera(B):
    """Scene.render_batch grows a workspace that was reserved for a camera with fewer pairs instead of failing, and the
    pinned output images of render_host_pipelined are re-made when width and height swap (same byte count)."""
    import dataclasses
    w = workloads.make("C5", 100_000, width=160, height=128)
    sc = _scene(w, tensor=False)
    pairs = [sc.count_pairs(c)[0] for c in w.cameras]
    small = w.cameras[int(np.argmin(pairs))]
    assert max(pairs) > min(pairs)
    sc.reserve(small, slack=1.0)
    sc.max_pairs = min(pairs)                                   # exactly what the smallest camera needs
    imgs, status = sc.render_batch(raw=True)                    # would raise without the re-reserve
    assert (status.cpu().numpy()[:, 0] == 0).all() and sc.max_pairs >= max(pairs)
    k = int(np.argmax(pairs))
    _tol_check(imgs[k].cpu().numpy(), oracle.render(w, camera=w.cameras[k], raw=True), "batch after growing the workspace")

    w2 = workloads.make("C3", 50_000, width=192, height=128)
    sc2 = _scene(w2)
    tall = dataclasses.replace(w2.camera, width=128, height=192)
    sc2.reserve(max_pairs=max(sc2.count_pairs(c)[0] for c in (w2.camera, tall)) + 1024)
    hb = sc2.host_buffers()
    a = sc2.render_host_pipelined(hb, 2)[0]
    assert tuple(a.shape) == (128, 192, 3)
    b = sc2.render_host_pipelined(hb, 2, cam=tall)[0]
    assert tuple(b.shape) == (192, 128, 3)
    _tol_check(b.numpy(), oracle.render(w2, camera=tall), "pipelined host render, transposed image shape")


def test_normalize_output_map(B):
    """splotch_normalize: out = 1 - exp(-S) (R13), the step the multi-GPU path applies after its all-reduce.  In place and
    out of place, odd lengths, a pointer that is not 16-byte aligned (scalar tail path), negative and huge S, n = 0."""
    rs = np.random.RandomState(3)
    for n, off in ((0, 0), (1, 0), (7, 1), (4099, 0), (4099, 3), (1_000_003, 1)):
        S = np.concatenate([rs.lognormal(-2.0, 3.0, max(n - 4, 0)), [0.0, -0.25, 1e-8, 200.0]])[:n].astype(np.float32)
        buf = torch.zeros(n + off + 4, dtype=torch.float32, device="cuda")
        src = buf[off:off + n]
        src.copy_(torch.from_numpy(S))
        dst = torch.full((n + off + 4,), -7.0, dtype=torch.float32, device="cuda")
        B.splotch_normalize(src, dst[off:off + n], n)                  # out of place
        B.splotch_normalize(src, src, n)                               # in place (S == out)
        torch.cuda.synchronize()
        ref = -np.expm1(-S.astype(np.float64))
        for got in (dst[off:off + n].cpu().numpy(), src.cpu().numpy()):
            np.testing.assert_allclose(got, ref, rtol=3e-6, atol=1e-7)
        assert bool((dst[:off] == -7.0).all()) and bool((dst[off + n:] == -7.0).all())     # nothing written outside [0, n)


def test_sharded_scene_on_one_gpu(B):
    """PAPER.md:95 on one device: two particle shards of C1 rendered to raw partial images by two ShardedScenes, summed (what
    the all-reduce does), mapped once with splotch_normalize; against the oracle and the unsharded render.  Then
    ShardedScene.render itself under a one-rank NCCL process group: render raw -> dist.all_reduce -> splotch_normalize,
    the exact call sequence of the N-GPU job."""
    import socket
    import torch.distributed as dist
    from paper_1004_1302_b200.multi import ShardedScene, shard_workload
    w = workloads.make("C1")
    ref = oracle.render(w)
    whole = _scene(w).render().cpu().numpy()
    parts = [ShardedScene(shard_workload(w, 2, r), "cuda:0") for r in range(2)]
    assert parts[0].scene.n + parts[1].scene.n == w.n
    total = parts[0].render(raw=True).clone()
    total += parts[1].render(raw=True)
    B.splotch_normalize(total, total, total.numel())
    torch.cuda.synchronize()
    _tol_check(total.cpu().numpy(), ref, "two shards, summed and mapped")
    np.testing.assert_allclose(total.cpu().numpy(), whole, rtol=1e-4, atol=2e-6)
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1, device_id=torch.device("cuda:0"))
    try:
        one = ShardedScene(w, "cuda:0")
        img = one.render().cpu().numpy()                      # raw render -> all_reduce over the one-rank group -> output map
        _tol_check(img, ref, "ShardedScene.render, one-rank NCCL group")
        raw = one.render(raw=True).cpu().numpy()
        _tol_check(raw, oracle.render(w, raw=True), "ShardedScene.render(raw=True)")
    finally:
        dist.destroy_process_group()


def test_stats_counts(B):
    w = workloads.make("C1")
    sc = _scene(w)
    vis, pairs, upd = sc.stats(bin_shift=4)
    ref = oracle.project_f32(w)
    _, ro, _ = oracle.bins(ref["bbox"], ref["visible"], 256, 256, 4, with_members=False)
    assert vis == int(ref["visible"].sum()) and pairs == int(ro[-1])
    tab, ok = oracle.splat_table(w)
    # U: covered pixel centres, counted independently in double for a sample of particles
    idx = np.nonzero(ref["visible"])[0][::50]
    ws = mk(np.stack([w.x[idx], w.y[idx], w.z[idx], w.r[idx], w.I[idx], w.colval[idx]], 1), w.camera, lut_e=w.lut_e,
            brightness=w.brightness)
    _, _, upd_s = _scene(ws).stats(bin_shift=4)
    jj, ii = np.meshgrid(np.arange(256) + 0.5, np.arange(256) + 0.5, indexing="ij")
    expect = sum(int(((ii - tab[p, 0]) ** 2 + (jj - tab[p, 1]) ** 2 <= tab[p, 3] ** 2).sum()) for p in idx)
    assert abs(upd_s - expect) <= max(3, expect // 20000)
    assert upd > 50 * upd_s * 0.5


def test_render_host_matches_device_render(B):
    w = workloads.make("C3", 200_000, width=320, height=320)
    sc = _scene(w)
    dev = sc.render().cpu().numpy()
    hb = sc.host_buffers()
    out_host, _ = sc.render_host(hb)
    np.testing.assert_allclose(out_host.numpy(), dev, rtol=2e-6, atol=1e-7)
    ref = oracle.render(w)
    _tol_check(out_host.numpy(), ref, "render_host")


def test_render_host_async_pipelined_frames(B):
    """splotch_render_host_async: frames streamed with two in flight (two streams, two workspaces).  Every frame must
    equal the synchronous call; changing a host array between frames changes exactly the frames enqueued afterwards; a
    frame whose pair capacity is too small reports it through the status head of its own workspace."""
    w = workloads.make("C3", 150_000, width=256, height=192)
    sc = _scene(w)
    sc.reserve()
    hb = sc.host_buffers()
    ref_host, _ = sc.render_host(hb)
    ref_host = ref_host.numpy().copy()
    outs = sc.render_host_pipelined(hb, 5)                     # frames 3 and 4 are in the two slots at the end
    for o in outs:
        np.testing.assert_allclose(o.numpy(), ref_host, rtol=2e-5, atol=1e-6)
    _tol_check(outs[0].numpy(), oracle.render(w), "pipelined host render")
    hb["I"].mul_(0.5)                                          # pinned host array changed in place: the next frames see it
    outs = sc.render_host_pipelined(hb, 2)
    w.I = w.I * np.float32(0.5)
    ref2 = oracle.render(w)
    for o in outs:
        _tol_check(o.numpy(), ref2, "pipelined host render, changed input")
    with pytest.raises(B.SplotchError):
        sc.render_host_pipelined(hb, 2, max_pairs=sc.max_pairs // 4)


# ------------------------------------------------------------------------------------------------
# stage (b): range normalisation of a scalar field on the device
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("log_scale", [False, True])
@pytest.mark.parametrize("n", [0, 1, 3, 1025, 4_000_003])
def test_field_normalisation_matches_oracle(B, n, log_scale):
    rs = np.random.RandomState(n % 97 + 1)
    v = rs.lognormal(-1.0, 2.5, n).astype(np.float32) - (0.0 if log_scale else 0.7)
    if n >= 1025:
        v[[7, 300, 1024]] = [np.nan, np.inf, -np.inf]
        v[11] = 0.0
        v[12] = -3.0
    ref, (lo, hi) = oracle.normalize_field(v, log_scale)
    buf = torch.empty(n + 1, dtype=torch.float32, device="cuda")          # +1: misaligned view exercises the scalar path
    for view in (buf[:n], buf[1:n + 1]):
        view.copy_(torch.from_numpy(v))
        rng_dev = torch.empty(2, dtype=torch.float32, device="cuda")
        out = torch.empty(n, dtype=torch.float32, device="cuda")
        B.splotch_field_range(view, n, log_scale, rng_dev)
        B.splotch_field_normalize(view, n, log_scale, rng_dev, out)
        torch.cuda.synchronize()
        got_rng = rng_dev.cpu().numpy().astype(np.float64)
        np.testing.assert_allclose(got_rng, (lo, hi), rtol=2e-6, atol=2e-6)
        got = out.cpu().numpy().astype(np.float64)
        assert np.array_equal(np.isnan(got), np.isnan(ref))
        np.testing.assert_allclose(got[~np.isnan(ref)], ref[~np.isnan(ref)], rtol=0, atol=3e-6)
        B.splotch_field_normalize(view, n, log_scale, rng_dev, view)       # in place
        torch.cuda.synchronize()
        np.testing.assert_array_equal(view.cpu().numpy(), out.cpu().numpy())


@pytest.mark.parametrize("gamma", [1.0, 2.2])
@pytest.mark.parametrize("n", [0, 5, 3 * 333 * 257])
def test_tonemap_codes_match_oracle(B, n, gamma):
    rs = np.random.RandomState(n % 89 + 2)
    v = rs.uniform(-0.1, 1.1, n).astype(np.float32)
    if n > 100:
        v[:8] = [np.nan, np.inf, -np.inf, 0.0, 1.0, 0.5 / 255, 1.5 / 255, 254.5 / 255]
        v[8:264] = np.arange(256, dtype=np.float32) / np.float32(255)
    d = torch.from_numpy(v).cuda()
    out = torch.empty(n, dtype=torch.uint8, device="cuda")
    B.splotch_tonemap_rgb8(d, n, gamma, out)
    torch.cuda.synchronize()
    got, ref = out.cpu().numpy().astype(int), oracle.tonemap_rgb8(v, gamma).astype(int)
    if gamma == 1.0:
        assert np.array_equal(got, ref)                      # bit-exact: the same fp32 operations on both sides
    else:                                                    # powf differs in the last ulp between libm and CUDA: a code may
        y = 255.0 * np.clip(np.nan_to_num(v.astype(np.float64), nan=0.0), 0, 1) ** (1.0 / gamma)   # flip only next to a half
        bad = got != ref
        assert (np.abs(got - ref) <= 1).all() and (np.abs((y[bad] % 1.0) - 0.5) < 1e-3).all() and bad.sum() <= 1e-3 * max(n, 1)


# ------------------------------------------------------------------------------------------------
# vector colouring (reading R19)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", [ADDITIVE, ABSORB])
def test_vector_colouring_matches_oracle(B, mode):
    w = workloads.make("C1", 60_000, width=300, height=212)
    rs = np.random.RandomState(21)
    w.vec = rs.uniform(0.0, 1.5, (w.n, 3)).astype(np.float32)
    w.vec[[5, 900], [0, 2]] = [np.nan, np.inf]                 # culled
    w.mode = mode
    if mode == ABSORB:
        w.lut_a = w.lut_e.copy()                               # ignored, but the absorb mode wants a table
        w.abs_brightness = [0.6 * b for b in w.brightness]
    sc = _scene(w)
    sc.d["colval"] = None                                      # colval may be NULL with vector colouring
    out = sc.render(raw=(mode == ADDITIVE)).cpu().numpy()
    ref = oracle.render_vector(w, raw=(mode == ADDITIVE))
    assert ref.max() > 0.2
    _tol_check(out, ref, f"vector colouring, mode {mode}")
    # the colour table is really ignored: a different table gives the same image
    w.lut_e = w.lut_e[:, ::-1].copy()
    out2 = _scene(w).render(raw=(mode == ADDITIVE)).cpu().numpy()
    np.testing.assert_allclose(out2, out, rtol=2e-5, atol=1e-6)
    # ... and may be absent altogether (include/splotch.h: the table pointers may be NULL with vector colouring)
    sc3 = _scene(w)
    sc3.d["colval"] = None
    sc3.d["lut_e"] = None
    sc3.d["lut_a"] = None
    out3 = sc3.render(raw=(mode == ADDITIVE)).cpu().numpy()
    np.testing.assert_allclose(out3, out, rtol=2e-5, atol=1e-6)
