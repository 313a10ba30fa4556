"""N > 1 host logic on CPU: world-size-2 gloo run of the additive sharding.

The render of each shard is the oracle's raw-S image here (the CUDA render needs a GPU); what is
under test is the product's host logic in paper_1004_1302_b200/multi.py: shard bounds, ONE
sum-reduction of the partial images, output map applied once after the reduction.
"""
import os
import socket

import numpy as np
import pytest

import oracle
import workloads
from paper_1004_1302_b200 import multi

torch = pytest.importorskip("torch")


@pytest.mark.parametrize("n,world", [(0, 2), (1, 2), (7, 3), (100, 8), (100_000_003, 8)])
def test_shard_bounds_partition_the_particles(n, world):
    b = [multi.shard_bounds(n, world, r) for r in range(world)]
    assert b[0][0] == 0 and b[-1][1] == n
    for r in range(world - 1):
        assert b[r][1] == b[r + 1][0]
    sizes = [e - s for s, e in b]
    assert max(sizes) - min(sizes) <= 1 and sum(sizes) == n
    with pytest.raises(ValueError):
        multi.shard_bounds(n, world, world)


def test_shard_workload_slices_every_array():
    w = workloads.make("C3", 1001)
    parts = [multi.shard_workload(w, 3, r) for r in range(3)]
    for k in ("x", "y", "z", "r", "I", "colval", "type"):
        np.testing.assert_array_equal(np.concatenate([getattr(p, k) for p in parts]), getattr(w, k))
    assert [p.n for p in parts] == [334, 334, 333]
    assert parts[0].brightness == w.brightness and parts[0].cameras is w.cameras


def test_shard_workload_slices_the_colour_vectors():
    """vector colouring (f3) + particle sharding (e): every rank must see ITS particles' vectors."""
    w = workloads.make("C1", 1001)
    w.vec = np.random.RandomState(0).uniform(0, 1, (w.n, 3)).astype(np.float32)
    parts = [multi.shard_workload(w, 3, r) for r in range(3)]
    np.testing.assert_array_equal(np.concatenate([p.vec for p in parts]), w.vec)
    assert [len(p.vec) for p in parts] == [334, 334, 333] and w.vec.shape == (1001, 3)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q, vec=False):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.make("C1", 20_000, width=96, height=64)
        if vec:
            w.vec = np.random.RandomState(5).uniform(0, 1, (w.n, 3)).astype(np.float32)
        sh = multi.shard_workload(w, world, rank)
        render = oracle.render_vector if vec else oracle.render
        partial = torch.from_numpy(render(sh, raw=True))                 # this rank's raw S (double)
        calls = {"reduce": 0, "map": 0}

        def all_reduce(t):
            calls["reduce"] += 1
            dist.all_reduce(t, op=dist.ReduceOp.SUM)

        def output_map(t):
            calls["map"] += 1
            t.copy_(-torch.expm1(-t))

        img = multi.combine_partials(partial, all_reduce, output_map)
        raw = multi.combine_partials(torch.from_numpy(render(sh, raw=True)), all_reduce, None)
        q.put((rank, img.numpy().copy(), raw.numpy().copy(), dict(calls)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("vec", [False, True])
def test_two_rank_gloo_sharded_render_equals_single_render(vec):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, vec)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=300) for _ in procs]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    w = workloads.make("C1", 20_000, width=96, height=64)
    if vec:
        w.vec = np.random.RandomState(5).uniform(0, 1, (w.n, 3)).astype(np.float32)
        ref, ref_raw = oracle.render_vector(w), oracle.render_vector(w, raw=True)
    else:
        ref, ref_raw = oracle.render(w), oracle.render(w, raw=True)
    assert ref.max() > 0.3
    for rank, img, raw, calls in got:
        assert calls == {"reduce": 2, "map": 1}
        np.testing.assert_allclose(raw, ref_raw, rtol=1e-12, atol=1e-15)      # order-independent sum
        np.testing.assert_allclose(img, ref, rtol=1e-12, atol=1e-15)          # map AFTER the reduction
    np.testing.assert_array_equal(got[0][1], got[1][1])                       # every rank holds the image


def test_sharding_refuses_absorb_mode():
    w = workloads.make("C4", 100, width=32, height=32)
    with pytest.raises((ValueError, RuntimeError)):
        multi.ShardedScene(w, "cuda:0")


def test_bench_spawn_command_is_the_drivers_launch_line():
    """`python bench.py --gpus N` outside torchrun re-executes itself as one rank per GPU with the rendezvous on 127.0.0.1:
    the command it builds is the launch line the driver uses, with the user's arguments passed through."""
    import importlib.util
    import os
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "2", "--warmup", "3"])
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"]
    assert "--nnodes=1" in cmd and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and int(cmd[cmd.index("--master-port") + 1]) > 0
    k = cmd.index(os.path.join(root, "bench.py"))
    assert cmd[k + 1:] == ["--gpus", "4", "--steps", "2", "--warmup", "3"]
