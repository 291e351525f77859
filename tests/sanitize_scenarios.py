"""Scenarios for compute-sanitizer (memcheck / racecheck / synccheck on configs 0 and 1).

    compute-sanitizer --tool memcheck  python tests/sanitize_scenarios.py
    compute-sanitizer --tool racecheck python tests/sanitize_scenarios.py
    compute-sanitizer --tool synccheck python tests/sanitize_scenarios.py

One tool per run (B200_PROFILING.md). Renders BASELINE.json configs 0 and 1 through every list builder and round
structure of the library -- the default block path with lazy lists, complete lists, exact tile lists, compact keys,
64-bit keys, index-order (no depth presort), a scene whose tiles park (second round), the sky and dynamics targets,
a band render -- and checks each frame against the default mode's image, so that the kernels built on relaxed
look-back words, tickets and last-CTA patterns all run under the tool. Independently of the tool, every device buffer
of the library carries 4 KB guard bands (pvg_guard_bands) that are verified after every scenario: an out-of-bounds
write of any kernel into the neighbourhood of a workspace buffer fails the run even where compute-sanitizer is closed. Device memory comes from plain cudaMalloc
(torch_allocator=False), so that memcheck sees every allocation's bounds. Not a pytest module."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2311_18561_b200 as pvg  # noqa: E402
from workloads import make_config, sky_cubemap  # noqa: E402


def main():
    assert torch.cuda.is_available()
    pvg.use_torch_allocator(False)
    pvg.guard_bands(True)     # every workspace buffer carries 4 KB guard bands: checked after every scenario
    frames = 0
    checked = 0

    def guards(label):
        nonlocal checked
        bad, n = pvg.check_guards()
        assert bad == 0 and n > 10, (label, bad, n)
        checked += n

    for cfg, n in ((0, None), (1, 60_000)):
        wl = make_config(cfg, n=n)
        cam = wl.cameras[0]
        s = wl.scene
        sc = pvg.Scene(s.mu, s.quat, s.scale, s.opacity, s.sh, s.tau, s.beta, s.vel, s.cycle, s.sh_degree, torch_allocator=False)
        ref = [x.clone() for x in sc.render(cam, 0.37)]
        frames += 1

        def same(label):
            nonlocal frames
            out = sc.render(cam, 0.37)
            torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(ref, out)), label
            sc.debug(["vals_sorted", "ranges", "counts"])
            guards(label)
            frames += 1

        sc.set_option(pvg.OPT_LAZY_CHUNKS, 0); same("complete lists")
        sc.set_option(pvg.OPT_EXACT_TILES, 1); same("exact tile lists")
        sc.set_option(pvg.OPT_EXACT_TILES, 0)
        sc.set_option(pvg.OPT_LAZY_CHUNKS, 1); sc.set_option(pvg.OPT_LAZY_SLAB, 48); same("lazy, one chunk, small slab")
        sc.set_option(pvg.OPT_LAZY_CHUNKS, 2); sc.set_option(pvg.OPT_LAZY_SLAB, 16)
        sc.set_option(pvg.OPT_BLOCK_BINS, 0); same("compact keys")
        sc.set_option(pvg.OPT_COMPACT_KEYS, 0); same("64-bit keys, depth presort")
        sc.set_option(pvg.OPT_PRESORT_DEPTH, 0); same("64-bit keys, index order")
        sc.set_option(pvg.OPT_PRESORT_DEPTH, 1); sc.set_option(pvg.OPT_COMPACT_KEYS, 1); sc.set_option(pvg.OPT_BLOCK_BINS, 1)
        sc.set_option(pvg.OPT_LAZY_DEPTH, 2); same("front-first depth order")
        sc.set_option(pvg.OPT_LAZY_SLAB, 64); same("front-first depth order, small slab")
        sc.set_option(pvg.OPT_LAZY_SLAB, 16); sc.set_option(pvg.OPT_LAZY_DEPTH, 1)
        sc.set_option(pvg.OPT_BLEND_CULL, 0); same("no staging cull")
        sc.set_option(pvg.OPT_BLEND_CULL, 1)
        # sky, dynamics target, temporal-smoothing state, a band of tile rows
        sc.set_sky(sky_cubemap(64, seed=1)); sc.render(cam, 0.37); sc.set_sky(None)
        sc.render(cam, 0.37, target="dynamics", dt=0.01, rho_max=3.0)
        ty = (cam.height + 15) // 16
        sc.set_tile_rows(1, max(2, ty - 1)); sc.render(cam, 0.37); sc.set_tile_rows(0, 0)
        frames += 3
        guards("targets and band")
        sc.close()
        # a scene whose tiles park: nearly transparent, so the first blend phase runs out of list prefix
        thin = pvg.Scene(s.mu, s.quat, s.scale * 1.5, (s.opacity * 0.03).astype(np.float32), s.sh, s.tau, s.beta, s.vel, s.cycle,
                         s.sh_degree, torch_allocator=False)
        thin.set_option(pvg.OPT_LAZY_CHUNKS, 0)
        full = [x.clone() for x in thin.render(cam, 0.37)]
        thin.set_option(pvg.OPT_LAZY_CHUNKS, 1); thin.set_option(pvg.OPT_LAZY_SLAB, 64)
        for ld in (1, 2, 2):   # front-first order: the first parking frame runs the device-launched second round, the next the host's
            thin.set_option(pvg.OPT_LAZY_DEPTH, ld)
            lazy = thin.render(cam, 0.37)
            torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(full, lazy)), "parked scene"
            guards("parked scene")
            frames += 1
        print(f"config {cfg}: parked tiles {thin.frame_stats()['parked_tiles']}")
        thin.close()
        frames += 1
    # the sort primitive on its own
    keys = torch.randint(0, 2 ** 62, (300_003,), dtype=torch.int64, device="cuda")
    vals = torch.arange(300_003, dtype=torch.int32, device="cuda")
    ko, vo = pvg.sort_pairs(keys.clone(), vals.clone())
    assert torch.equal(ko, torch.sort(keys, stable=True)[0])
    torch.cuda.synchronize()
    print(f"sanitize scenarios ok: {frames} frames, {checked} guarded allocations checked, none damaged")


if __name__ == "__main__":
    main()
