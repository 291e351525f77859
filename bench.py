#!/usr/bin/env python
"""bench.py -- PVG render FPS at 1920x1280 on B200 (BASELINE.json metric), with roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (preprocess, depth sort, scan + duplicate, onesweep
sort, tile ranges, blend) over one frame (camera, t) of the workload: BASELINE.json config 3,
3M Gaussians, 1920x1280, 50 timestamps in [0,1]. The scene (the model theta) is resident in HBM
like network weights; the per-step input is (camera, t). N > 1: frames are sharded over ranks,
no data-path collective, weak scaling.

Prints ONE JSON line on rank 0. `--impl reference` times the CPU oracle (test infrastructure,
never tuned) on the host cores for the same metric/config and prints the same line shape.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "render_fps_1920x1280"
UNIT = "frames/s"
CONFIG_NAMES = {0: "cfg0_tiny_4096g_128x96", 1: "cfg1_mid_200kg_960x640", 2: "cfg2_urban_1Mg_1920x1280",
                3: "cfg3_timesweep_3Mg_1920x1280_50t", 4: "cfg4_stress_6Mg_5cams"}
# issue slots per (pixel, list entry) evaluation of the blend
SLOTS_REJECT, SLOTS_ACCEPT_EXTRA = 11, 6


def base_config(args, n_gaussians: int, frames, world_size: int) -> dict:
    """`config` of the JSON line: what is rendered. Identical in both arms (ours / reference) by construction; what is
    specific to an arm's run goes into `run_details`."""
    c0 = frames[0][0]
    return {"workload": CONFIG_NAMES[args.config], "n_gaussians": int(n_gaussians), "resolution": f"{c0.width}x{c0.height}",
            "frames": "one (camera, t) per step, round-robin over the sweep",
            "l2_policy": f"inputs larger than L2: the model, {n_gaussians * 256 / 1e6:.0f} MB, is read every frame (126 MB L2)",
            "parallelism": f"frames sharded over {world_size} rank(s), no collective"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--n", type=int, default=None, help="override the point count (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-pipelined", action="store_true")
    ap.add_argument("--presort", type=int, default=1)
    ap.add_argument("--block-bins", type=int, default=1)
    ap.add_argument("--split", default="frames", choices=["frames", "band"],
                    help="frames (default, the contract's line): every rank renders its own frames, no collective; "
                         "band: all ranks render tile-row bands of the SAME frame + one all-gather (strong scaling)")
    ap.add_argument("--bands", type=int, default=0,
                    help="with --split band on ONE GPU: time the bands of a K-way split one after another and "
                         "report the slowest band per frame (what one of K GPUs would compute; no collective)")
    ap.add_argument("--lazy-chunks", type=int, default=-1, help="PVG_OPT_LAZY_CHUNKS (-1: the library default)")
    ap.add_argument("--no-legs", action="store_true", help="skip the complete_lists / parked / sustained legs")
    ap.add_argument("--sustained-seconds", type=float, default=2.5)
    ap.add_argument("--selftest-spawn", action="store_true",
                    help="CPU self-test of the --gpus N launch path: the ranks rendezvous over gloo, take the max of a "
                         "dummy time and rank 0 prints a line with n_gpus (no CUDA work)")
    ap.add_argument("--event-stride", type=int, default=5,
                    help="record per-kernel CUDA events on every k-th timed frame (each record costs ~2 us of stream time)")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel: str, workload: str):
    """dram bytes per launch from the committed ncu --set full capture, if one exists."""
    try:
        with open(os.path.join(ROOT, "profiles", "roofline_traffic.json")) as f:
            d = json.load(f)
        return d.get(workload, {}).get(kernel)
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("timestamp,index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None
        self.t0 = self.t1 = None

    def mark_start(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.12)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        import datetime
        rows = []
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 10:
                continue
            try:
                ts = datetime.datetime.strptime(parts[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                rows.append((ts, float(parts[2]), float(parts[3]), parts[5:10]))
            except Exception:
                continue
        sel = [r for r in rows if self.t0 is not None and self.t0 - 0.05 <= r[0] <= self.t1 + 0.05] or rows
        if sel:
            out["sm_mhz"] = statistics.median(r[1] for r in sel)
            out["sm_max_mhz"] = max(r[2] for r in sel)
            names = ["active_mask", "hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            seen = set()
            for r in sel:
                for nm, v in zip(names[1:], r[3][1:]):
                    if v.lower().startswith("active"):
                        seen.add(nm)
            out["reasons"] = sorted(seen)
            out["samples"] = len(sel)
        try:
            os.unlink(self.f.name)
        except Exception:
            pass
        return out


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------------
def oracle_frame_time(wl, cam, t, sample_tiles: int = 0, seed: int = 0):
    """Times the CPU oracle (as it stands) on ONE WHOLE frame: Oracle-P on all N Gaussians + Oracle-R (binned) on
    every tile. Nothing is sampled or extrapolated. Returns (seconds, detail dict)."""
    import oracle
    tiles_total = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    t0 = time.perf_counter()
    _, rec = oracle.preprocess_scene(wl.scene, cam, t)
    t1 = time.perf_counter()
    oracle.render(rec, cam.width, cam.height, bg=cam.bg, mode="binned")
    t2 = time.perf_counter()
    return t2 - t0, dict(preprocess_s=t1 - t0, tiles_s=t2 - t1, tiles=int(tiles_total), tiles_total=int(tiles_total))


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only. Every step is ONE WHOLE FRAME
    (Oracle-P on all N Gaussians + Oracle-R binned on every tile): nothing is sampled or extrapolated, so the figure
    agrees with the `cpu_baseline` the GPU arm measures on the same box (3 s per config-3 frame on 16 cores: the default
    50 + 3 steps take under three minutes)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from workloads import make_config
    if "WORLD_SIZE" in os.environ:
        # torchrun exports OMP_NUM_THREADS=1 to its workers; the oracle is timed on all the host cores it may use
        oracle.set_threads(len(os.sched_getaffinity(0)))
    wl = make_config(args.config, args.n)
    frames = list(wl.frames())
    times = []
    det = None
    for s in range(args.warmup + args.steps):
        cam, t = frames[s % len(frames)]
        sec, det = oracle_frame_time(wl, cam, float(np.float32(t)), 0, seed=s)
        if s >= args.warmup:
            times.append(sec)
    sec = float(np.mean(times))
    fps = 1.0 / sec
    line = {"impl": "reference", "metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": base_config(args, wl.scene.n, frames, args.gpus),
            "cpu_baseline": {"value": fps, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": (f"every step one whole frame: Oracle-P on all {wl.scene.n} Gaussians + Oracle-R (binned) "
                                        f"on all {det['tiles_total']} tiles; no sampling, no extrapolation")},
            "e2e": {"value": fps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a torchrun environment: start the N ranks here (one process per GPU, the
    launch line the driver uses) and pass their output through; rank 0 prints the one JSON line."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_selftest_spawn(args):
    """The plumbing of an N-rank run without CUDA: gloo rendezvous, barrier, max over ranks, one line from rank 0."""
    from paper_2311_18561_b200 import dist
    rank, local_rank, ws = dist.init("gloo")
    frames = [("cam", k / 49.0) for k in range(50)]
    sched = dist.frame_schedule(rank, ws, args.steps, frames)
    dist.barrier()
    elapsed = dist.max_over_ranks(1e-3 * (rank + 1))
    total = dist.sum_over_ranks(len(sched))
    dist.barrier()
    if rank == 0:
        print(json.dumps({"selftest": "spawn", "n_gpus": ws, "steps": args.steps, "frames_total": int(total),
                          "elapsed_max_s": elapsed}), flush=True)
    dist.shutdown()


# ------------------------------------------------------------------------------------------
def algorithmic_bytes(agg, K, N, S, Msum, Mbsum, chunks, lazy):
    """Algorithmic HBM bytes over the K sampled frames, per (kernel, stage)."""
    alg = {("preprocess", "preprocess"): K * (64.0 * N + 80.0 * N + 192.0 * S),
           ("scan_counts", "duplicate"): K * 12.0 * N,   # 8 B sorted key (or 4 B visit + 4 B count) + 4 B offset
           # block-entry path (blockbin.cuh): 13 B entries (u8 block, u32 Gaussian, u64 mask)
           ("bin_expand", "duplicate"): 13.0 * Mbsum + K * 16.0 * S,
           ("tile_grid", "ranges"): K * 16.0 * N,
           ("bin_pass", "sort"): 25.0 * Mbsum,
           ("bin_emit", "sort"): 12.0 * Mbsum + K * 16.0 * S,   # fused expand + split: 16 B per survivor read, (u32 g, u64 mask) written
           ("bin_write", "sort"): 12.0 * Mbsum + 4.0 * Msum + 256.0 * chunks,
           ("duplicate", "duplicate"): (6.0 if any(k[0] == "compact_pass_last" for k in agg) else 12.0) * Msum,
           ("compact_pass", "sort"): 12.0 * Msum * (agg.get(("compact_pass", "sort"), [0, K])[1] / K),
           ("compact_pass_last", "sort"): 10.0 * Msum,
           ("onesweep_histogram", "sort"): 8.0 * Msum,
           ("onesweep_histogram", "depth_sort"): K * 8.0 * N,
           ("tile_ranges", "ranges"): 8.0 * Msum}
    if lazy:
        # deferred records: preprocess reads the 64 B model + 1 B flag and writes tile info, count and depth key (28 B)
        alg[("preprocess", "preprocess")] = K * 93.0 * N
        # lazy lists: bin_emit forms the first 1/8 of the entries and bin_write the first chunks of every block -- what
        # they move depends on where the tiles saturate, so no algorithmic-byte figure is claimed for them
        alg.pop(("bin_emit", "sort"), None)
        alg.pop(("bin_write", "sort"), None)
    if ("depth_select", "depth_sort") in agg:
        # front-first depth order (PVG_OPT_LAZY_DEPTH): the selection reads the n depth pairs (8 B) and writes the few
        # pairs in front; the front's passes and scan (front_sort_scan, or onesweep_pass + scan_counts for a large
        # front) move some ten thousand pairs -- latency, no byte figure claimed
        alg[("depth_select", "depth_sort")] = agg[("depth_select", "depth_sort")][1] * 8.0 * N
        alg.pop(("scan_counts", "duplicate"), None)
    for key in (("onesweep_pass", "sort"), ("onesweep_pass", "depth_sort")):
        if key == ("onesweep_pass", "depth_sort") and ("depth_select", "depth_sort") in agg:
            continue
        if key in agg:
            per_frame = agg[key][1] / K
            # depth sort (9 + 9 + 9 + 4 bits): pass 0 reads the n keys (8 B; the value of pair i is i) and writes the S
            # surviving pairs (12 B), passes 1 and 2 move the S pairs, the top-digit pass is the identity and not launched
            alg[key] = 24.0 * Msum * per_frame if key[1] == "sort" else K * (8.0 * N + 60.0 * S)
    return alg


def timed_frames(pvg, torch, dist, scene, sched, cams, out_by_cam, local_rank, dev, stride, on_start=None, on_end=None):
    """K frames, inputs resident in HBM, device-timed with CUDA events on the current stream, barrier + synchronize on
    both sides, max over ranks. Per-kernel CUDA-event records on every stride-th frame."""
    scene.set_option(pvg.OPT_EVENT_STRIDE, stride)
    scene.set_option(pvg.OPT_KERNEL_EVENTS, 2)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    Ms, Mbs, parked = [], [], []
    dist.barrier(local_rank)
    torch.cuda.synchronize()
    if on_start:
        on_start()
    e0.record()
    for cam, t in sched:
        scene.render(cams[id(cam)], t, out_by_cam[id(cam)])
        fs = scene.frame_stats()
        Ms.append(fs["M"])
        Mbs.append(fs["block_entries"])
    e1.record()
    torch.cuda.synchronize()
    if on_end:
        on_end()
    dist.barrier(local_rank)
    elapsed_s = dist.max_over_ranks(e0.elapsed_time(e1) / 1e3, dev)
    krecs = scene.kernel_times_ms()
    scene.set_option(pvg.OPT_EVENT_STRIDE, 1)
    scene.set_option(pvg.OPT_KERNEL_EVENTS, 0)
    return dict(elapsed_s=elapsed_s, krecs=krecs, Ms=Ms, Mbs=Mbs, parked=scene.frame_stats()["parked_tiles"])


def count_pairs(pvg, scene, sched, cams, out_by_cam):
    """Blend work (pairs evaluated / contributing) of the same frames, counted in an untimed pass."""
    scene.set_option(pvg.OPT_COUNT_PAIRS, 1)
    ev = co = 0
    for cam, t in sched:
        scene.render(cams[id(cam)], t, out_by_cam[id(cam)])
        a, b = scene.blend_counters()
        ev += a
        co += b
    scene.set_option(pvg.OPT_COUNT_PAIRS, 0)
    return ev, co


def kernel_table(run, stride, N, S, lazy, hbm_peak, alu_peak, pairs=None):
    """Per-kernel aggregation of one timed loop: times, shares, achieved GB/s or thread-instructions/s, and per-stage
    ms and Gaussians/s (north_star: 'frames/sec and Gaussians/sec per stage')."""
    Kall = len(run["Ms"])
    sampled = list(range(0, Kall, stride))
    K = len(sampled)
    Msum, Mbsum = float(sum(run["Ms"][i] for i in sampled)), float(sum(run["Mbs"][i] for i in sampled))
    chunks = Mbsum / 512 + K * 150
    agg = {}
    for name, stage, ms in run["krecs"]:
        a = agg.setdefault((name, stage), [0.0, 0])
        a[0] += ms
        a[1] += 1
    alg = algorithmic_bytes(agg, K, N, S, Msum, Mbsum, chunks, lazy)
    frame_ms = run["elapsed_s"] * 1e3 / Kall
    kernels = {}
    for (name, stage), (ms, cnt) in agg.items():
        d = {"launches": cnt, "ms_total": ms, "ms_avg": ms / cnt, "ms_per_frame": ms / K, "share": (ms / K) / frame_ms}
        b = alg.get((name, stage))
        if b:
            d["GBps"] = b / (ms * 1e-3) / 1e9
            d["hbm_frac"] = d["GBps"] / hbm_peak
            d["algorithmic_bytes_per_launch"] = b / cnt
        kernels[f"{stage}/{name}"] = d
    bl = agg.get(("blend", "blend"))
    if bl and pairs:
        ev, co = pairs
        slots = (SLOTS_REJECT * ev + SLOTS_ACCEPT_EXTRA * co) * K / Kall   # pairs were counted on all frames
        k = kernels["blend/blend"]
        k["pairs_eval_per_frame"] = ev / Kall
        k["pairs_contrib_per_frame"] = co / Kall
        k["Tinstr_per_s"] = slots / (bl[0] * 1e-3) / 1e12
        k["alu_frac"] = k["Tinstr_per_s"] / alu_peak
    stage_ms, stage_gps = {}, {}
    for (name, stage), (ms, cnt) in agg.items():
        stage_ms[stage] = stage_ms.get(stage, 0.0) + ms / K
    for stage, ms in stage_ms.items():
        stage_gps[stage] = N / (ms * 1e-3) if ms > 0 else None
    return dict(kernels=kernels, agg=agg, alg=alg, stage_ms=stage_ms, stage_gaussians_per_s=stage_gps, K=K, Kall=Kall,
                Msum=Msum, Mbsum=Mbsum, launches_per_frame=len(run["krecs"]) / K)


def run_ours(args):
    import torch
    import paper_2311_18561_b200 as pvg
    from paper_2311_18561_b200 import build as pvg_build, dist
    from workloads import make_config

    rank, local_rank, ws = dist.init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the render path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        pvg_build.build()
    dist.barrier(local_rank)

    wl = make_config(args.config, args.n)
    frames = list(wl.frames())
    sched = dist.frame_schedule(rank, ws, args.steps, frames)
    warm = dist.frame_schedule(rank, ws, max(args.warmup, 3), frames)
    scene = pvg.Scene.from_workload_scene(wl.scene)
    scene.set_option(pvg.OPT_PRESORT_DEPTH, args.presort)
    scene.set_option(pvg.OPT_BLOCK_BINS, args.block_bins)
    if args.lazy_chunks >= 0:
        scene.set_option(pvg.OPT_LAZY_CHUNKS, args.lazy_chunks)
    cams = {id(c): pvg.camera_struct(c) for c, _ in frames}

    def outs(c):
        return (torch.empty((3, c.height, c.width), device=dev), torch.empty((c.height, c.width), device=dev),
                torch.empty((c.height, c.width), device=dev))

    out_by_cam = {k: outs(c) for k, c in {id(c): c for c, _ in frames}.items()}

    def warm_up(sc):
        for cam, t in warm:
            sc.render(cams[id(cam)], t, out_by_cam[id(cam)])
        torch.cuda.synchronize()

    # ---- warm-up (also sizes the workspace)
    warm_up(scene)

    # ---- the ALU / issue peak of this device, measured: FFMA only, FFMA + LOP3, packed FFMA2
    calib = {}
    for mode, name in ((0, "ffma"), (1, "ffma_lop3"), (2, "ffma2")):
        rate, sms = pvg.calibrate_fp32(mode)
        calib[name] = rate / 1e12
    calib["sms"] = sms

    # ---- timed region: K frames, inputs resident in HBM, device-timed, max over ranks
    sampler = ClockSampler(physical_gpu_index(local_rank)) if rank == 0 else None
    time.sleep(0.3 if sampler else 0.0)
    stride = max(1, min(args.event_stride, len(sched)))
    main = timed_frames(pvg, torch, dist, scene, sched, cams, out_by_cam, local_rank, dev, stride,
                        on_start=sampler.mark_start if sampler else None, on_end=sampler.mark_end if sampler else None)
    clocks = sampler.stop() if sampler else None
    elapsed_s = main["elapsed_s"]
    total_frames = args.steps * ws
    fps = total_frames / elapsed_s
    pairs = count_pairs(pvg, scene, sched, cams, out_by_cam)

    # ---- two frames in flight: the same K frames through the scene and a fork of it (shared model), on two streams
    handles = [scene, scene.fork()]
    lanes = [torch.cuda.Stream(), torch.cuda.Stream()]
    out2 = [out_by_cam, {k: outs(c) for k, c in {id(c): c for c, _ in frames}.items()}]
    cur = torch.cuda.current_stream()

    def in_flight(seq):
        for i, (cam, t) in enumerate(seq):
            with torch.cuda.stream(lanes[i % 2]):
                handles[i % 2].render(cams[id(cam)], t, out2[i % 2][id(cam)])

    pipelined = None
    if not args.no_pipelined:
        in_flight(warm[:4])
        torch.cuda.synchronize()
        dist.barrier(local_rank)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record()
        for ln in lanes:
            ln.wait_stream(cur)
        in_flight(sched)
        for ln in lanes:
            cur.wait_stream(ln)
        p1.record()
        torch.cuda.synchronize()
        dist.barrier(local_rank)
        pel = dist.max_over_ranks(p0.elapsed_time(p1) / 1e3, dev)
        pipelined = {"value": total_frames / pel, "unit": UNIT, "frames_in_flight": 2, "ms_per_step": pel * 1e3 / args.steps,
                     "note": "the same K frames, alternately through the scene and a pvg_fork_scene of it (shared model, two "
                             "workspaces) on two streams; `value`, the per-kernel times and the roofline above are one frame at a time"}

    # ---- end to end through the C ABI with HOST buffers (D2H of the images inside the timed region)
    e2e = None
    if not args.no_e2e:
        def pinned(v):
            return (torch.empty(v[0].shape, pin_memory=True), torch.empty(v[1].shape, pin_memory=True),
                    torch.empty(v[2].shape, pin_memory=True))
        # two frames in flight (scene + fork), two host image sets per handle and camera: frame k is copied out while
        # the next frames render
        host = [{k: (pinned(v), pinned(v)) for k, v in out_by_cam.items()} for _ in handles]

        def e2e_loop(seq):
            for i, (cam, t) in enumerate(seq):
                with torch.cuda.stream(lanes[i % 2]):
                    handles[i % 2].render_host_async(cams[id(cam)], t, host[i % 2][id(cam)][(i // 2) % 2])
            for h in handles:
                h.wait_host()

        e2e_loop(warm[:4])
        dist.barrier(local_rank)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e2e_loop(sched)
        torch.cuda.synchronize()
        el = dist.max_over_ranks(time.perf_counter() - t0, dev)
        dist.barrier(local_rank)
        d2h = sum(cam.width * cam.height * 5 * 4 for cam, _ in sched)
        e2e = {"value": total_frames / el, "unit": UNIT,
               "h2d_bytes_per_step": int(pvg.C.sizeof(pvg.CameraC) + 4), "d2h_bytes_per_step": int(d2h // len(sched)),
               "note": "pvg_render_host_async + pvg_wait_host, two frames in flight (scene + pvg_fork_scene): per-step input is "
                       "(camera, t); every frame's rgb+depth+alpha is copied to pinned host memory inside the timed region, the "
                       "copies overlapping the following renders"}
        del host
    handles[1].close()
    torch.cuda.synchronize()

    if rank != 0:
        scene.close()
        dist.shutdown()
        return

    # ---- per-kernel aggregation and roofline
    hbm_peak, sm_max_mhz, peak_src = measured_peaks()
    N = wl.scene.n
    S = scene.frame_stats()["survivors"] or N
    list_mode = scene.frame_stats()["list_mode"]
    lazy = list_mode == "blocks" and args.lazy_chunks != 0
    sm_mhz = (clocks or {}).get("sm_mhz") or sm_max_mhz
    nominal = calib["sms"] * 128 * sm_mhz * 1e6 / 1e12    # T thread-instr/s at the observed SM clock
    # the denominator of the ALU roofline: the best issue rate the microbenchmark reached on this device
    alu_peak = max(calib["ffma"], calib["ffma_lop3"])
    tab = kernel_table(main, stride, N, S, lazy, hbm_peak, alu_peak, pairs)
    kernels, agg, alg, K, Kall = tab["kernels"], tab["agg"], tab["alg"], tab["K"], tab["Kall"]
    dom = max(agg.items(), key=lambda kv: kv[1][0])[0]
    dk = kernels[f"{dom[1]}/{dom[0]}"]
    workload = CONFIG_NAMES[args.config]
    alu_src = (f"pvg_calibrate_fp32 on this device ({calib['sms']} SMs from cudaDeviceGetAttribute): FFMA+LOP3 {calib['ffma_lop3']:.2f}, "
               f"FFMA {calib['ffma']:.2f}, packed FFMA2 {calib['ffma2']:.2f} T thread-instr/s (an FFMA2 counts once); nominal "
               f"{calib['sms']} x 128 lanes x {sm_mhz:.0f} MHz = {nominal:.2f}")
    if dom[0] == "blend":
        roofline = {"bound": "alu", "achieved": dk["Tinstr_per_s"], "peak": alu_peak, "unit": "Tinstr/s",
                    "frac": dk["alu_frac"], "traffic": ncu_traffic("blend", workload), "kernel": "blend_kernel",
                    "peak_source": alu_src, "frac_of_nominal": dk["Tinstr_per_s"] / nominal}
    else:
        roofline = {"bound": "hbm", "achieved": dk.get("GBps"), "peak": hbm_peak, "unit": "GB/s", "frac": dk.get("hbm_frac"),
                    "traffic": ncu_traffic(dom[0], workload), "kernel": f"{dom[0]} ({dom[1]} stage)",
                    "peak_source": peak_src, "avg_launch_ms": dk["ms_avg"],
                    "algorithmic_bytes_per_launch": (alg[dom] / agg[dom][1]) if dom in alg else None}

    # ---- extra legs (1 GPU only): complete lists, a scene whose tiles park, a sustained loop
    legs = {}
    if ws == 1 and not args.no_legs and list_mode == "blocks":
        # (1) complete lists + eager records (PVG_OPT_LAZY_CHUNKS = 0): every list entry is formed, split and written
        scene.set_option(pvg.OPT_LAZY_CHUNKS, 0)
        warm_up(scene)
        sm1 = ClockSampler(physical_gpu_index(local_rank))
        time.sleep(0.3)
        run1 = timed_frames(pvg, torch, dist, scene, sched, cams, out_by_cam, local_rank, dev, stride, sm1.mark_start, sm1.mark_end)
        ck1 = sm1.stop()
        pairs1 = count_pairs(pvg, scene, sched, cams, out_by_cam)
        t1 = kernel_table(run1, stride, N, S, False, hbm_peak, alu_peak, pairs1)
        legs["complete_lists"] = {
            "value": total_frames / run1["elapsed_s"], "unit": UNIT, "ms_per_step": run1["elapsed_s"] * 1e3 / args.steps,
            "clocks": ck1, "stage_ms_per_frame": t1["stage_ms"],
            "kernels": {k: {a: v[a] for a in ("ms_per_frame", "launches", "GBps", "hbm_frac", "alu_frac", "Tinstr_per_s") if a in v}
                        for k, v in t1["kernels"].items()},
            "note": "PVG_OPT_LAZY_CHUNKS=0: full preprocess (records, SH), every block entry emitted and split, every tile list "
                    "written whole; same frames, same images bit for bit"}
        # (1b) exact tile lists on top of the complete lists (PVG_OPT_EXACT_TILES; SURVEY 8(f-4) at list-build time)
        scene.set_option(pvg.OPT_EXACT_TILES, 1)
        warm_up(scene)
        run1b = timed_frames(pvg, torch, dist, scene, sched, cams, out_by_cam, local_rank, dev, stride)
        t1b = kernel_table(run1b, stride, N, S, False, hbm_peak, alu_peak)
        legs["exact_tiles"] = {
            "value": total_frames / run1b["elapsed_s"], "unit": UNIT, "ms_per_step": run1b["elapsed_s"] * 1e3 / args.steps,
            "instances_rectangles": int(run1b["Ms"][-1]), "instances_exact": int(scene.frame_stats()["M_exact"]),
            "stage_ms_per_frame": t1b["stage_ms"],
            "kernels": {k: {"ms_per_frame": v["ms_per_frame"], "launches": v["launches"]} for k, v in t1b["kernels"].items()},
            "note": "complete lists of only the tiles each Gaussian's ellipse can reach (P13): masks refined in bin_emit, tile "
                    "counts counted, ranges rebuilt; images bit-identical. Compare with complete_lists (the rectangle lists)"}
        scene.set_option(pvg.OPT_EXACT_TILES, 0)
        scene.set_option(pvg.OPT_LAZY_CHUNKS, args.lazy_chunks if args.lazy_chunks >= 0 else 2)

        # (2) a scene whose tiles do NOT saturate inside the list prefixes: opacity x 0.05 -> tiles park, the second
        #     round forms the remaining entries and writes the rest of the parked tiles' lists
        s0 = wl.scene
        thin = pvg.Scene(s0.mu, s0.quat, s0.scale, (s0.opacity * 0.05).astype(np.float32), s0.sh, s0.tau, s0.beta, s0.vel,
                         s0.cycle, s0.sh_degree)
        warm_up(thin)
        run2 = timed_frames(pvg, torch, dist, thin, sched, cams, out_by_cam, local_rank, dev, stride)
        t2 = kernel_table(run2, stride, N, thin.frame_stats()["survivors"] or N, True, hbm_peak, alu_peak)
        legs["parked"] = {
            "value": total_frames / run2["elapsed_s"], "unit": UNIT, "ms_per_step": run2["elapsed_s"] * 1e3 / args.steps,
            "parked_tiles_last_frame": run2["parked"], "tiles": int(frames[0][0].width // 16 * (frames[0][0].height // 16)),
            "instances_per_frame_mean": t2["Msum"] / t2["K"], "stage_ms_per_frame": t2["stage_ms"],
            "kernels": {k: {"ms_per_frame": v["ms_per_frame"], "launches": v["launches"]} for k, v in t2["kernels"].items()},
            "note": "the same scene with every opacity x 0.05 (default lazy options): pixels do not saturate inside the list "
                    "prefixes, the tiles park and the second round completes their lists"}
        thin.close()
        del thin
        torch.cuda.synchronize()

        # (3) sustained: the 50-frame sweep looped for >= sustained_seconds of device time, clocks sampled throughout
        warm_up(scene)
        sm3 = ClockSampler(physical_gpu_index(local_rank))
        time.sleep(0.3)
        sweep = [frames[k % len(frames)] for k in range(max(len(frames), 50))]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        sm3.mark_start()
        w0 = time.perf_counter()
        nfr = 0
        e0.record()
        while time.perf_counter() - w0 < args.sustained_seconds:
            for cam, t in sweep:
                scene.render(cams[id(cam)], t, out_by_cam[id(cam)])
            nfr += len(sweep)
        e1.record()
        torch.cuda.synchronize()
        sm3.mark_end()
        sus_s = e0.elapsed_time(e1) / 1e3
        legs["sustained"] = {"value": nfr / sus_s, "unit": UNIT, "frames": nfr, "seconds": sus_s, "ms_per_step": sus_s * 1e3 / nfr,
                             "clocks": sm3.stop(),
                             "note": "the time sweep looped back to back (one frame at a time, no per-kernel events) for the stated "
                                     "seconds of device time"}

    # ---- CPU oracle on ONE whole frame (reported baseline, not the target)
    cpu = None
    if not args.no_cpu_baseline and ws == 1:
        import oracle
        cam, t = frames[len(frames) // 2]
        est, det = oracle_frame_time(wl, cam, float(np.float32(t)))
        cpu = {"value": 1.0 / est, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"frame t={t:.3f}: Oracle-P on all {N} Gaussians ({det['preprocess_s']:.2f} s) + Oracle-R (binned) on "
                         f"all {det['tiles_total']} tiles ({det['tiles_s']:.2f} s): one whole frame, no extrapolation"}

    line = {"metric": METRIC, "value": fps, "unit": UNIT, "n_gpus": ws, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": elapsed_s * 1e3 / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": base_config(args, N, frames, ws),
            "run_details": {"survivors_last_frame": S, "instances_per_frame_mean": tab["Msum"] / K,
                            "block_entries_per_frame_mean": tab["Mbsum"] / K, "list_mode": list_mode,
                            "lists": ("lazy (PVG_OPT_LAZY_CHUNKS/SLAB defaults): list prefixes, the remainder only for parked tiles; "
                                      f"parked tiles in the last frame: {main['parked']}") if lazy else "complete",
                            "arithmetic": "fp32; the position chain mu~(t) -> p_cam -> mean2D and the record's conic in fp64 (DESIGN.md 5)",
                            "presort_depth": args.presort},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "pipelined": pipelined, "clocks": clocks,
            "gpu_launches": int(round(len(main["krecs"]) * Kall / K)),
            "kernel_events": f"recorded on every {stride}th frame of the timed region ({K} of {Kall} frames, {len(main['krecs'])} launches)",
            "gaussians_per_s": N * fps, "stage_ms_per_frame": tab["stage_ms"],
            "stage_gaussians_per_s": tab["stage_gaussians_per_s"], "alu_calibration_Tinstr_per_s": calib,
            "kernels": kernels}
    line.update(legs)
    print(json.dumps(line), flush=True)
    scene.close()
    dist.shutdown()


def run_band_split(args):
    """Within-frame split; NOT the contract's line (that is run_ours). Every rank holds the
    scene, renders its band of tile rows of the same frame and the bands are all-gathered, so every rank ends
    each step with the whole frame. Strong scaling: value = frames/s of the job."""
    import torch
    import paper_2311_18561_b200 as pvg
    from paper_2311_18561_b200 import build as pvg_build, dist
    from workloads import make_config

    rank, local_rank, ws = dist.init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the render path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if rank == 0:
        pvg_build.build()
    dist.barrier(local_rank)
    wl = make_config(args.config, args.n)
    frames = list(wl.frames())
    sched = [frames[s % len(frames)] for s in range(args.steps)]
    warm = [frames[s % len(frames)] for s in range(max(args.warmup, 3))]
    scene = pvg.Scene.from_workload_scene(wl.scene)
    scene.set_option(pvg.OPT_KERNEL_EVENTS, 0)
    cams = {id(c): pvg.camera_struct(c) for c, _ in frames}
    out_by_cam = {id(c): (torch.zeros((3, c.height, c.width), device=dev), torch.zeros((c.height, c.width), device=dev),
                          torch.zeros((c.height, c.width), device=dev)) for c, _ in frames}
    parts = ws if ws > 1 else max(args.bands, 1)

    def step(cam, t, part):
        ty = (cam.height + 15) // 16
        b, e = dist.band_rows(part, parts, ty)
        if e > b:
            scene.set_tile_rows(b, e)
            scene.render(cams[id(cam)], t, out_by_cam[id(cam)])
        if ws > 1:
            dist.gather_bands(out_by_cam[id(cam)], ty)

    per_band = []
    for part in ([rank] if ws > 1 else range(parts)):
        for cam, t in warm:
            step(cam, t, part)
        torch.cuda.synchronize()
        dist.barrier(local_rank)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for cam, t in sched:
            step(cam, t, part)
        e1.record()
        torch.cuda.synchronize()
        dist.barrier(local_rank)
        per_band.append(e0.elapsed_time(e1) / 1e3)
    elapsed_s = dist.max_over_ranks(max(per_band), dev)
    if rank == 0:
        c0 = frames[0][0]
        line = {"metric": METRIC, "value": args.steps / elapsed_s, "unit": UNIT, "n_gpus": ws, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": elapsed_s * 1e3 / args.steps, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"config {args.config}", "n_gaussians": wl.scene.n,
                           "resolution": f"{c0.width}x{c0.height}",
                           "parallelism": (f"tile-row bands over {ws} ranks + one all-gather of the bands per frame" if ws > 1 else
                                           f"ONE GPU timing each band of a {parts}-way split in turn; value = slowest band, "
                                           "no collective (a projection of the per-rank compute, not a multi-GPU result)"),
                           "band_ms_per_frame": [x * 1e3 / args.steps for x in per_band]}}
        print(json.dumps(line), flush=True)
    scene.close()
    dist.shutdown()


if __name__ == "__main__":
    a = parse_args()
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the ranks ourselves (one process per GPU), so that `--gpus N` is real
        sys.exit(spawn_ranks(a))
    if a.selftest_spawn:
        run_selftest_spawn(a)
    elif a.impl == "reference":
        run_reference(a)
    elif a.split == "band":
        run_band_split(a)
    else:
        run_ours(a)
