"""N > 1 host logic on CPU: world_size-2 gloo processes exercise the frame schedule (frames
sharded over ranks, no data-path collective) and the barrier / max-over-ranks timing that
bench.py uses. The render itself needs a GPU and is covered by the -m gpu tests."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, steps: int, out_q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2311_18561_b200 import dist
    r, lr, ws = dist.init("gloo")
    assert (r, lr, ws) == (rank, rank, world)
    frames = [("cam", k / 49.0) for k in range(50)]
    sched = dist.frame_schedule(rank, ws, steps, frames)
    dist.barrier()
    elapsed = 0.010 * (rank + 1)                      # rank 1 is the slow one
    mx = dist.max_over_ranks(elapsed)
    total = dist.sum_over_ranks(len(sched))
    out_q.put((rank, [f[1] for f in sched], mx, total))
    dist.barrier()
    dist.shutdown()


def test_frame_sharding_and_max_timing_world2():
    world, steps = 2, 30
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, steps, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ts0, ts1 = res[0][1], res[1][1]
    frames = [k / 49.0 for k in range(50)]
    # weak scaling: every rank renders `steps` frames; together they walk the sweep in order
    assert len(ts0) == len(ts1) == steps
    inter = [t for pair in zip(ts0, ts1) for t in pair]
    assert inter == [frames[f % 50] for f in range(world * steps)]
    assert set(ts0).isdisjoint(ts1[:25])              # no frame rendered twice within one sweep
    # the timed region's duration is the max over ranks; the frame count is summed
    assert abs(res[0][2] - 0.020) < 1e-12 and abs(res[1][2] - 0.020) < 1e-12
    assert res[0][3] == res[1][3] == world * steps


def test_single_process_defaults():
    sys.path.insert(0, ROOT)
    from paper_2311_18561_b200 import dist
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert dist.world() == (0, 0, 1)
    assert dist.max_over_ranks(1.5) == 1.5
    assert dist.frame_schedule(0, 1, 3, ["a", "b"]) == ["a", "b", "a"]


def test_band_rows_partition():
    sys.path.insert(0, ROOT)
    from paper_2311_18561_b200 import dist
    for ty in (1, 7, 56, 80):
        for ws in (1, 2, 3, 8, 16):
            rows = [dist.band_rows(r, ws, ty) for r in range(ws)]
            assert rows[0][0] == 0 and rows[-1][1] == ty
            assert all(rows[k][1] == rows[k + 1][0] for k in range(ws - 1))
            h = [e - b for b, e in rows]
            assert max(h) - min(h) <= 1 and min(h) >= 0


def _band_worker(rank: int, world: int, port: int, H: int, W: int, out_q):
    import torch
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2311_18561_b200 import dist
    dist.init("gloo")
    TY = (H + 15) // 16
    g = torch.Generator().manual_seed(7)
    full = (torch.rand((3, H, W), generator=g), torch.rand((H, W), generator=g), torch.rand((H, W), generator=g))
    b, e = dist.band_rows(rank, world, TY)
    mine = tuple(torch.full_like(x, float("nan")) for x in full)      # only the own band is valid
    for m, f in zip(mine, full):
        m[..., b * 16:min(e * 16, H), :] = f[..., b * 16:min(e * 16, H), :]
    dist.gather_bands(mine, TY)
    out_q.put((rank, all(torch.equal(m, f) for m, f in zip(mine, full))))
    dist.barrier()
    dist.shutdown()


def test_gather_bands_world2_ragged_last_row():
    """Within-frame split: each rank holds its band of a 3-image frame; one all-gather assembles the frame on
    every rank. H = 886 = 55 tile rows + 6 pixels (the ragged last row of config 4's side cameras); 56 rows
    over 2 ranks."""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_band_worker, args=(r, world, port, 886, 96, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


def test_bench_gpus_n_starts_its_own_ranks():
    """`python bench.py --gpus 2` outside torchrun must start two ranks itself (torch.distributed.run, 127.0.0.1) and
    print ONE line from rank 0 with n_gpus = 2. --selftest-spawn runs the rendezvous, barrier and max-over-ranks over
    gloo without any CUDA work, so the launch path is covered on a CPU box."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-spawn", "--steps", "9"],
                       capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["frames_total"] == 18 and abs(d["elapsed_max_s"] - 2e-3) < 1e-12


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """--impl reference under a 2-rank launch: rank 0 alone runs the oracle (whole frames) and prints the line, the
    other rank exits 0 without work."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "0",
                        "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert "no extrapolation" in d["cpu_baseline"]["sample"] and d["cpu_baseline"]["cores"] >= 1
