"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol the header declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1004_1302_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def _declared():
    text = open(os.path.join(ROOT, "include", "splotch.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(splotch_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/splotch.h but not exported"


def test_binding_lists_every_symbol():
    from paper_1004_1302_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    for n in binding.EXPORTS:
        assert callable(getattr(binding, n)), n


def test_host_only_calls(lib):
    from paper_1004_1302_b200 import binding as B
    assert B.splotch_version() >= 100
    assert B.splotch_status_string(0) == "ok"
    assert "workspace" in B.splotch_status_string(B.SPLOTCH_ERR_WORKSPACE)
    cam = B.make_camera((0.5, 0.5, -1.5), (0.5, 0.5, 0.5), (0, 1, 0), 30.0, 2048, 2048)
    p = B.make_params([1.0], mode=B.SPLOTCH_ADDITIVE)
    small = B.splotch_workspace_bytes(1000, cam, p, 0)
    big = B.splotch_workspace_bytes(100_000_000, cam, p, 1_000_000_000)
    assert big > small > 0
    assert big >= 100_000_000 * 32 + 1_000_000_000 * 4
    pa = B.make_params([1.0], mode=B.SPLOTCH_ABSORB)
    assert B.splotch_workspace_bytes(1000, cam, pa, 1000) > B.splotch_workspace_bytes(1000, cam, p, 1000)
    assert B.splotch_sort_scratch_bytes(1 << 20) > 0


@pytest.mark.parametrize("kw", [dict(fov=0.0), dict(fov=180.0), dict(w=0), dict(w=20000), dict(eye_eq_look=True),
                                dict(up_parallel=True), dict(f=0.0), dict(mode=7), dict(znear=-1.0)])
def test_invalid_arguments_are_rejected_on_the_host(lib, kw):
    from paper_1004_1302_b200 import binding as B
    eye = (0.5, 0.5, -1.5)
    look = eye if kw.get("eye_eq_look") else (0.5, 0.5, 0.5)
    up = (0, 0, 1) if kw.get("up_parallel") else (0, 1, 0)
    cam = B.make_camera(eye, look, up, kw.get("fov", 30.0), kw.get("w", 256), 256)
    p = B.make_params([1.0], mode=kw.get("mode", 0), support_f=kw.get("f", 3.0), z_near=kw.get("znear", 0.01))
    with pytest.raises(B.SplotchError) as e:
        B.splotch_workspace_bytes(1000, cam, p, 1000)
    assert e.value.status in (B.SPLOTCH_ERR_INVALID_ARG, B.SPLOTCH_ERR_LIMIT)


def test_compute_entry_points_need_a_device(lib):
    """No CPU fallback: without a CUDA device the Scene refuses to run."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    import workloads
    from paper_1004_1302_b200 import Scene
    with pytest.raises(RuntimeError):
        Scene(workloads.make("C1", 100))


def test_bench_reference_arm_prints_one_json_line():
    """bench.py --impl reference is the CPU oracle on the box's host cores (no GPU needed): one JSON line with the
    contract's keys; under torchrun every rank but 0 exits without work."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--workload", "C1", "--steps", "1", "--warmup", "0"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env={**os.environ, "RANK": "0", "WORLD_SIZE": "1"})
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "Mparticles/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]
    assert "C1" in d["config"]["workload"]
    out1 = subprocess.run(cmd, capture_output=True, text=True, timeout=120, env={**os.environ, "RANK": "1", "WORLD_SIZE": "2"})
    assert out1.returncode == 0 and out1.stdout.strip() == ""
