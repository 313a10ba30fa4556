#!/usr/bin/env python
"""bench.py -- the Splotch render hot path on B200: Mparticles/s and roofline fractions.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--r-median X] [--impl ours|reference]

A "step" is one pass of the whole hot path (transform/cull/colour -> bin -> rasterise -> output
map) over the resident synthetic particle set of the workload.  The default workload is C3, the
100M-particle additive config BASELINE.json's north_star quotes its target on.  For C5 a step is the
whole 8-camera orbit (one splotch_render_batch).  --r-median X renders C3's geometry with another median
smoothing length (the footprint sweep of SURVEY.md 8(d): where the path becomes HBM-bound).  One JSON
line is printed on stdout (rank 0); everything else goes to stderr.

N > 1 (torchrun, one rank per GPU): additive mode shards by particles exactly like the paper's
MPI layer: every rank renders its own particle set into a raw-S partial image,
one NCCL all-reduce sums the partial images, then the output map is applied.  Weak scaling:
every rank holds a full-size particle set generated from its own seed.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "Mparticles/s rendered and achieved HBM GB/s fraction on one B200"
SM_COUNT_NOMINAL = 148
LANES_PER_SM = 128
L2_BYTES = 126 * 1000 * 1000                 # B200 L2 (B200_PROFILING.md)
ALGO_LANE_OPS_PER_UPDATE = {0: 5.0, 1: 17.0}   # 1 mul + 3 FMA + 1 test; absorb adds 3 exp + ~9 ops


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)),
                        bf16_tflops=float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", 1379.5))), source="measured")
        except Exception:  # pragma: no cover
            pass
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, bf16_tflops=1379.5, source="fallback")


def read_traffic(workload: str, kernel: str):
    """dram read + write bytes per launch of `kernel` from the committed ncu summary (profiles/traffic.csv)."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    import csv
    for row in csv.DictReader(open(path)):
        if row["workload"] == workload and row["kernel"] == kernel:
            return float(row["dram_bytes_read"]) + float(row["dram_bytes_write"])
    return None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def make_workload(name: str, n, rank: int, r_median=None):
    import workloads
    kw = {}
    if r_median is not None:
        if name != "C3":
            raise SystemExit("--r-median applies to C3's geometry only")
        kw["r_median"] = float(r_median)
    if rank > 0:
        kw["seed"] = {"C1": 1004130201, "C2": 1004130202, "C3": 1004130203, "C4": 1004130202, "C5": 1004130205}[name] + 1000 * rank
    t = time.time()
    w = workloads.make(name, n, **kw)
    log(f"[bench] rank {rank}: generated {name} n={w.n} in {time.time() - t:.1f}s")
    return w


def oracle_sample(w, target_seconds: float):
    """Bounded sample of the workload for the CPU oracle: a strided subsample at full resolution,
    stride chosen from a short calibration run so that one render takes about target_seconds."""
    import oracle
    cores = oracle.max_threads()
    probe = w.subsample(4096)
    t = time.time()
    oracle.render(probe)
    dt = max(time.time() - t, 1e-3)
    per_particle = dt / probe.n
    stride = int(np.ceil(per_particle * w.n / target_seconds))
    stride = max(1, min(stride, 4096))
    return w.subsample(stride), stride, cores


def run_reference(args):
    """--impl reference: the CPU oracle (as it stands) on a bounded sample of the same workload."""
    import oracle
    w = make_workload(args.workload, args.n, 0, args.r_median)
    budget = 150.0 / max(1, args.steps + args.warmup)
    ws, stride, cores = oracle_sample(w, min(25.0, budget))
    for _ in range(args.warmup):
        oracle.render(ws)
    t = time.time()
    for _ in range(args.steps):
        oracle.render(ws)
    dt = (time.time() - t) / max(1, args.steps)
    val = ws.n / dt / 1e6
    cam = w.camera
    line = dict(impl="reference", metric=METRIC, value=val, unit="Mparticles/s", n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=dt * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic",
                config=dict(workload=f"{w.name}: {w.n} particles, {cam.width}x{cam.height}, "
                                     f"{'absorb' if w.mode else 'additive'} mode", sample=f"1-in-{stride} strided subsample"),
                cpu_baseline=dict(value=val, unit="Mparticles/s", cores=cores, kind="oracle",
                                  sample=f"1-in-{stride} particle-strided subsample ({ws.n} particles) at full resolution"),
                e2e=dict(value=val, unit="Mparticles/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line), flush=True)


def spawn_command(n_gpus: int, argv, port: int = 0):
    """The torchrun command line that `python bench.py --gpus N <argv>` re-executes itself under: the driver's own launch
    line (one rank per GPU, rendezvous on 127.0.0.1).  port 0 = pick a free one."""
    if not port:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__), *argv]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--n", type=int, default=None, help="particle count (default: the config's full size)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--force-tensor", action="store_true", help="additive mode: SPLOTCH_FORCE_TENSOR")
    ap.add_argument("--no-tensor", action="store_true", help="additive mode: SPLOTCH_NO_TENSOR (everything on the FP32 ALUs)")
    ap.add_argument("--r-median", type=float, default=None,
                    help="C3 only: median smoothing length (default 0.005 = the config); the footprint sweep uses 0.0015 / 0.0005 / 0.00015")
    ap.add_argument("--single-frame", action="store_true", help="C5: time camera 0 only instead of the 8-camera orbit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args)
        return 0

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` outside torchrun: start the N ranks ourselves (one process per GPU), so that the
        # plain command and the driver's torchrun command run the same job.  Rank 0 of the child job prints the line.
        import subprocess
        import torch
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: this node has {torch.cuda.device_count()} CUDA device(s)")
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")                  # the communicator log (rings / NVLS) goes to stderr
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        return subprocess.call(spawn_command(args.gpus, sys.argv[1:]), env=env)
    if args.gpus != world:
        log(f"[bench] --gpus {args.gpus} but WORLD_SIZE={world}: the launcher decides; running {world} rank(s)")

    import torch
    import torch.distributed as dist
    from paper_1004_1302_b200 import Scene, binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    peaks = read_peaks()
    w = make_workload(args.workload, args.n, rank, args.r_median)
    if world > 1 and w.mode != 0:
        raise SystemExit("multi-GPU sharding is defined for the additive mode only (DESIGN.md 'Multi-GPU')")
    cams = list(w.cameras) if (len(w.cameras) > 1 and not args.single_frame) else [w.camera]
    n_frames = len(cams)                                   # C5: the 8-camera orbit is ONE step
    cam = cams[0]
    if world > 1:
        from paper_1004_1302_b200.multi import ShardedScene
        sharded = ShardedScene(w, dev)                     # every rank: its own particle set (weak scaling) + one all-reduce
        sc = sharded.scene
    else:
        sc = Scene(w, dev)
    sc.tensor = False if args.no_tensor else True if args.force_tensor else None
    per_cam = [sc.stats(c) for c in cams]                  # (visible, pairs, updates) per camera
    vis, pairs = per_cam[0][0], max(p for _, p, _ in per_cam)
    updates = float(np.mean([u for _, _, u in per_cam]))   # per frame
    if w.mode == 0:
        ts = [sc.tensor_stats(c) for c in cams]
        upd_tensor, tensor_on, tensor_share = float(np.mean([t[0] for t in ts])), ts[0][1], float(np.mean([t[2] for t in ts]))
    else:
        upd_tensor, tensor_on, tensor_share = 0, 0, 0.0
    sc.reserve(cam, max_pairs=pairs + 1024)
    log(f"[bench] rank {rank}: visible {vis}, pairs {pairs}, pixel updates U {updates:.4g} per frame, frames per step {n_frames}, "
        f"workspace {sc.workspace.numel() / 2**30:.2f} GiB")
    out = torch.empty((n_frames, cam.height, cam.width, 3), dtype=torch.float32, device=dev)

    def step():
        if world > 1:                              # one collective reduction of the partial images, then the output map
            sharded.render(cam, out=out[0], check=False)
        elif n_frames > 1:
            sc.render_batch(cams, out=out, check=False)
        else:
            sc.render(cam, out=out[0], check=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        step()
    barrier()
    status, _, _ = B.splotch_workspace_status(sc._aligned(sc.workspace))
    assert status == B.SPLOTCH_OK, "workspace too small"

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    launches0 = B.splotch_launch_count()
    B.splotch_profile_enable(True)
    # L2: a step streams the particle arrays and the workspace (splat records + pair list).  When that is at least twice
    # the 126 MB L2 nothing of one step survives into the next and no flush is needed; a smaller scene (C1) gets a 256 MB
    # fill between steps, outside the per-step event pairs, and its step time is the sum of the pairs.
    touched = w.n * 24 + sc.workspace.numel()
    need_flush = touched < 2 * L2_BYTES
    flushbuf = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if need_flush else None
    l2_note = (f"{touched / 1e6:.0f} MB touched per step < 2 x L2: 256 MB fill between steps, outside the timed event pairs" if need_flush else
               f"inputs + workspace ({touched / 1e9:.2f} GB per step) exceed the 126 MB L2 many times over; no flush needed")
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    barrier()
    for k in range(args.steps):
        if need_flush:
            flushbuf.fill_(k & 255)
        ev0[k].record()
        step()
        ev1[k].record()                            # one event pair per step: median and best beside the mean
    barrier()
    per_step = [ev0[k].elapsed_time(ev1[k]) for k in range(args.steps)]
    ms_total = sum(per_step) if need_flush else ev0[0].elapsed_time(ev1[-1])
    stage_ms, prof_calls = B.splotch_profile_read()
    B.splotch_profile_enable(False)
    launches = B.splotch_launch_count() - launches0
    clocks = sampler.stop()
    ms_step = ms_total / max(1, args.steps)
    if world > 1:
        t = torch.tensor([ms_step], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step = float(t.item())
        tl = torch.tensor([launches], dtype=torch.int64, device=dev)
        dist.all_reduce(tl)
        launches = int(tl.item())
    total_particles = w.n * world * n_frames       # every frame renders all N input particles
    value = total_particles / (ms_step * 1e-3) / 1e6
    ms_frame = ms_step / n_frames

    # ---- rooflines of the rasteriser (K3): plain FP32 ALU kernel, and in the additive mode the tensor-core kernel ----
    tensor_ms, alu_ms = stage_ms[3], stage_ms[4]
    raster_ms = tensor_ms + alu_ms
    tensor_used = w.mode == 0 and tensor_ms > 0.05
    sm_count = torch.cuda.get_device_properties(local_rank).multi_processor_count
    alu_peak = sm_count * LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12          # Tlane-op/s
    c_ops = ALGO_LANE_OPS_PER_UPDATE[w.mode]
    upd_alu = updates - (upd_tensor if tensor_used else 0)
    alu_kernel = "raster_additive_kernel" if w.mode == 0 else "raster_absorb_kernel"
    alu_achieved = upd_alu * c_ops / (alu_ms * 1e-3) / 1e12 if alu_ms > 0 else 0.0
    alu_roof = dict(bound="alu", kernel=alu_kernel, achieved=alu_achieved, peak=alu_peak, unit="Tlane-op/s",
                    frac=alu_achieved / alu_peak if alu_peak else None, traffic=read_traffic(w.name, alu_kernel),
                    kernel_ms=alu_ms, kernel_share_of_step=alu_ms / ms_frame if ms_frame else None,
                    updates_per_launch=upd_alu, algorithmic_lane_ops_per_update=c_ops,
                    peak_source=f"{sm_count} SMs x {LANES_PER_SM} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz ({peaks['source']} clock)")
    tensor_roof = None
    if tensor_used:
        tf32_peak = 0.5 * peaks["bf16_tflops"]                                     # guide: TF32 dense = half of BF16
        t_achieved = 2.0 * 3.0 * upd_tensor / (tensor_ms * 1e-3) / 1e12            # one multiply-add per channel per update
        tensor_roof = dict(bound="tensor", kernel="raster_additive_mma_kernel", achieved=t_achieved, peak=tf32_peak,
                           unit="TFLOP/s", frac=t_achieved / tf32_peak, traffic=read_traffic(w.name, "raster_additive_mma_kernel"),
                           kernel_ms=tensor_ms, kernel_share_of_step=tensor_ms / ms_frame, updates_per_launch=upd_tensor,
                           algorithmic_flops_per_update=6.0,
                           # 128/96 padded accumulator rows x the TF32 products per term: 1 for a batch of faint splats
                           # (|a_c| <= 2^-7: every splat of C1..C5), 3 (split operands) for a batch with a brighter one
                           executed_over_algorithmic="1.33 (faint batches) .. 4.0 (three-product split)",
                           peak_source=f"0.5 x sustained dense BF16 cuBLAS throughput ({peaks['source']}) = TF32 dense")
    # the dominant kernel by time is the headline roofline; the whole rasteriser is also quoted in ALU terms
    roofline = alu_roof if (not tensor_used or alu_ms >= tensor_ms) else tensor_roof
    eq = updates * c_ops / (raster_ms * 1e-3) / 1e12 if raster_ms > 0 else 0.0
    raster_equiv = dict(unit="Tlane-op/s", achieved=eq, peak=alu_peak, frac=eq / alu_peak if alu_peak else None,
                        raster_ms=raster_ms, updates=updates, updates_on_tensor_cores=upd_tensor if tensor_used else 0,
                        tensor_share_estimate=tensor_share, tensor_cores_used=bool(tensor_used),
                        note="all K3 updates x algorithmic lane-ops / (tensor + ALU kernel time): what an ALU-only "
                             "rasteriser would have to sustain to match")
    algo_bytes = w.n * w.bytes_per_particle + cam.width * cam.height * 12       # per frame
    hbm_gbs = algo_bytes / (ms_frame * 1e-3) / 1e9
    hbm = dict(algorithmic_bytes_per_step=algo_bytes, achieved_gbs=hbm_gbs, frac_of_measured=hbm_gbs / peaks["hbm_gbs"],
               frac_of_nominal_8TBs=hbm_gbs / 8000.0, peak_gbs=peaks["hbm_gbs"], peak_source=peaks["source"])

    # front end (K1 and the lists) against the HBM roofline by the bytes these kernels themselves must move
    rec_bytes = 48 if w.mode else 32
    k1_bytes = w.n * (w.bytes_per_particle + rec_bytes + 4 + (4 if w.mode else 0))    # inputs read; record, packed bin box (, depth key) written
    list_bytes = w.n * 4 + per_cam[0][1] * 4                                          # packed bin boxes read, pair list written (additive)
    frontend = dict(project_ms=stage_ms[0], project_bytes=k1_bytes,
                    project_frac_of_hbm=k1_bytes / (stage_ms[0] * 1e-3) / 1e9 / peaks["hbm_gbs"] if stage_ms[0] > 0 else None,
                    lists_ms=stage_ms[2], lists_bytes=list_bytes if w.mode == 0 else None,
                    lists_frac_of_hbm=(list_bytes / (stage_ms[2] * 1e-3) / 1e9 / peaks["hbm_gbs"]) if (w.mode == 0 and stage_ms[2] > 0) else None,
                    frontend_share_of_frame=(stage_ms[0] + stage_ms[1] + stage_ms[2]) / ms_frame if ms_frame else None)

    # ---- end to end through the C ABI with host buffers: every frame copies its inputs H2D and its image D2H ----
    e2e = None
    if not args.no_e2e and world == 1:
        hb = sc.host_buffers()
        out_host = torch.empty((cam.height, cam.width, 3), dtype=torch.float32).pin_memory()
        sc.workspace = None
        torch.cuda.empty_cache()
        mp = pairs + 1024
        # (a) one call at a time: splotch_render_host (copies, render, copy back, synchronise)
        _, hws = sc.render_host(hb, cam, out_host=out_host, max_pairs=mp)
        n_serial = max(1, min(args.steps, 3))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_serial):
            sc.render_host(hb, cam, out_host=out_host, max_pairs=mp, workspace=hws)
        dt_serial = (time.perf_counter() - t0) / n_serial
        del hws
        torch.cuda.empty_cache()
        # (b) a stream of frames, two in flight (splotch_render_host_async on two streams / workspaces): the copies of
        #     frame k + 1 run on the copy engines while frame k is rasterised; every frame still moves all its bytes
        free, _ = torch.cuda.mem_get_info()
        need = 2 * B.splotch_workspace_bytes_host(w.n, B.make_camera(cam.eye, cam.lookat, cam.up, cam.fov_deg, cam.width, cam.height),
                                                  B.make_colormap(hb["lut_e"], hb["lut_a"], sc.n_entries, sc.n_types), sc.params(), mp)
        dt_pipe, n_pipe = None, 0
        if free > need + (2 << 30):
            sc.render_host_pipelined(hb, 2, cam, max_pairs=mp)                       # warm-up: allocates the two slots
            n_pipe = max(4, min(2 * args.steps, 10))
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sc.render_host_pipelined(hb, n_pipe, cam, max_pairs=mp)
            dt_pipe = (time.perf_counter() - t0) / n_pipe
            sc._pipe = None
            torch.cuda.empty_cache()
        dt = dt_pipe if dt_pipe is not None else dt_serial
        e2e = dict(value=w.n / dt / 1e6, unit="Mparticles/s", h2d_bytes_per_step=sc.h2d_bytes(),
                   d2h_bytes_per_step=cam.width * cam.height * 12, ms_per_step=dt * 1e3, steps=n_pipe if dt_pipe is not None else n_serial,
                   call=("splotch_render_host_async, two frames in flight on two streams (pinned host buffers; every frame "
                         "copies its inputs H2D and its image D2H inside the timed region)") if dt_pipe is not None else
                        "splotch_render_host (pinned host buffers; copies inside the timed call)",
                   serial=dict(value=w.n / dt_serial / 1e6, ms_per_step=dt_serial * 1e3, steps=n_serial,
                               call="splotch_render_host, one synchronous call at a time (latency of one frame)"),
                   frames_per_step=1, note="per frame (camera 0)" if n_frames > 1 else None)
    elif world > 1:
        e2e = dict(value=None, unit="Mparticles/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0,
                   note="end-to-end host-buffer path is measured at N=1")

    # ---- CPU baseline: the oracle on a bounded sample, rank 0 at N=1 only; best and median of 3 ----
    cpu = None
    if not args.no_cpu_baseline and world == 1 and rank == 0:
        import oracle
        ws_, stride, cores = oracle_sample(w, 7.0)
        times = []
        for _ in range(3):
            t0 = time.time()
            oracle.render(ws_)
            times.append(time.time() - t0)
        best, med = min(times), float(np.median(times))
        cpu = dict(value=ws_.n / best / 1e6, unit="Mparticles/s", cores=cores, kind="oracle", seconds=best,
                   median_value=ws_.n / med / 1e6, runs=3,
                   sample=f"1-in-{stride} particle-strided subsample ({ws_.n} particles) of {w.name} at full resolution "
                          f"(subsample measurement; best of 3, median beside it)")

    if rank == 0:
        wl = f"{w.name}: {w.n} particles/GPU, {cam.width}x{cam.height}, {'absorb' if w.mode else 'additive'} mode, f={w.support_f}"
        if args.r_median is not None:
            wl += f", median r {args.r_median} (footprint sweep; the config has 0.005)"
        if n_frames > 1:
            wl += f", orbit of {n_frames} cameras per step (splotch_render_batch)"
        line = dict(metric=METRIC, value=value, unit="Mparticles/s", n_gpus=world, steps=args.steps, warmup=args.warmup,
                    ms_per_step=ms_step, ms_per_step_median=float(np.median(per_step)), ms_per_step_best=float(min(per_step)),
                    higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                    data="synthetic",
                    config=dict(workload=wl,
                                parallelism=f"particle shards x{world} + all-reduce of raw S" if world > 1 else "single GPU",
                                l2=l2_note,
                                seed=w.seed, visible=vis, pairs=pairs, pixel_updates=updates, updates_per_particle=updates / w.n,
                                frames_per_step=n_frames, ms_per_frame=ms_frame,
                                pixels_per_s=cam.width * cam.height / (ms_frame * 1e-3),
                                updates_per_s=updates * world / (ms_frame * 1e-3)),
                    clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline,
                    roofline_alu=alu_roof, roofline_tensor=tensor_roof, raster_alu_equivalent=raster_equiv, hbm_roofline=hbm,
                    frontend=frontend,
                    stage_ms=dict(zip(["project_count", "offsets", "lists", "raster_tensor", "raster_alu", "output_map"], stage_ms)),
                    cpu_baseline=cpu)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
