"""Lazy tile lists (include/pvg.h PVG_OPT_LAZY_CHUNKS): the lists are written only as far as the first k chunks of
every 8x8-tile block reach, the blend runs on those prefixes, and the tiles that still have a live pixel at the end
of their prefix are parked, get the rest of their lists written and resume. What is unique is the image -- every
pixel must see the same entries in the same order with the same arithmetic -- so the images are compared BIT FOR
BIT with k = 0 (complete lists, which the other parity tests tie to the oracle), on scenes chosen so that no,
some and all tiles park; the evaluation counters must agree too. The lists themselves are checked against the
oracle by every other parity test: pvg_debug_view completes them on demand."""
import numpy as np
import pytest
import torch

import oracle
import paper_2311_18561_b200 as pvg
from workloads import make_config, sky_cubemap

pytestmark = pytest.mark.gpu


def _scene(wl, opacity_scale=1.0, scale_scale=1.0):
    s = wl.scene
    return pvg.Scene(s.mu, s.quat, s.scale * np.float32(scale_scale), np.clip(s.opacity * np.float32(opacity_scale), 1e-4, 0.999),
                     s.sh, s.tau, s.beta, s.vel, s.cycle, s.sh_degree)


def _render(sc, k, cam, t, slab=8, **kw):
    sc.set_option(pvg.OPT_LAZY_CHUNKS, k)
    sc.set_option(pvg.OPT_LAZY_SLAB, slab)
    sc.set_option(pvg.OPT_COUNT_PAIRS, 1)
    out = [x.clone() for x in sc.render(cam, t, **kw)]
    torch.cuda.synchronize()
    return out, sc.blend_counters(), sc.frame_stats()["parked_tiles"]


@pytest.mark.parametrize("cfg,n,cam_i,op,sc_scale", [
    (1, 200_000, 0, 1.0, 1.0),     # dense and opaque: nothing parks
    (1, 200_000, 0, 0.03, 1.0),    # nearly transparent: every tile with a long list parks
    (1, 200_000, 0, 0.3, 0.6),     # in between
    (4, 150_000, 3, 0.15, 1.0),    # ragged last tile row, yawed camera
    (2, 300_000, 0, 0.1, 1.5),
])
def test_lazy_lists_give_bit_identical_images(cfg, n, cam_i, op, sc_scale):
    wl = make_config(cfg, n=n)
    cam, t = wl.cameras[cam_i], 0.4
    sc = _scene(wl, op, sc_scale)
    try:
        full, ctr_full, _ = _render(sc, 0, cam, t)
        parked = []
        for k in (1, 2, 5):
            lazy, ctr, p = _render(sc, k, cam, t, slab=1)      # every entry formed up front
            parked.append(p)
            for a, b in zip(full, lazy):
                assert torch.equal(a, b), f"k={k}"
            assert ctr == ctr_full, f"k={k}: evaluations {ctr} vs {ctr_full}"
        print("parked tiles for k = 1, 2, 5:", parked, "of", ((cam.width + 15) // 16) * ((cam.height + 15) // 16))
        if op < 0.05:
            assert parked[0] > 0
        assert parked[0] >= parked[1] >= parked[2]
        # lazy emission: only the first 1/slab of the entries exists in the first round
        for k, slab in ((2, 8), (1, 64), (5, 3), (2, 4096)):
            lazy, ctr, p = _render(sc, k, cam, t, slab=slab)
            for a, b in zip(full, lazy):
                assert torch.equal(a, b), f"k={k} slab={slab}"
            assert ctr == ctr_full
            print(f"k={k} slab={slab}: parked {p}")
    finally:
        sc.close()


def test_lazy_lists_park_some_tiles_and_the_lists_complete_on_demand():
    """A scene whose upper half is nearly transparent: those tiles park, the others do not. After the lazy render the
    debug view must still return every tile's whole list (it writes what the frame never needed)."""
    wl = make_config(1, n=120_000)
    s = wl.scene
    cam, t = wl.cameras[0], 0.5
    rec_o, _ = oracle.preprocess_scene(s, cam, t)
    upper = rec_o[:, 20] < cam.height / 2          # projected y of the oracle's wide record
    opacity = np.where(upper, s.opacity * 0.02, s.opacity).astype(np.float32)
    sc = pvg.Scene(s.mu, s.quat, s.scale, opacity, s.sh, s.tau, s.beta, s.vel, s.cycle, s.sh_degree)
    try:
        full, _, _ = _render(sc, 0, cam, t)
        dbg_full = sc.debug(["vals_sorted", "ranges"])
        lazy, _, parked = _render(sc, 1, cam, t, slab=1)
        tiles = ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
        assert 0 < parked < tiles, parked
        for a, b in zip(full, lazy):
            assert torch.equal(a, b)
        dbg = sc.debug(["vals_sorted", "ranges"])
        assert np.array_equal(dbg["ranges"], dbg_full["ranges"])
        assert np.array_equal(dbg["vals_sorted"], dbg_full["vals_sorted"])
        # the same with lazy emission, whether or not the frame itself had to form the remaining entries
        for slab in (16, 4096):
            lazy, _, _ = _render(sc, 1, cam, t, slab=slab)
            for a, b in zip(full, lazy):
                assert torch.equal(a, b)
            assert np.array_equal(sc.debug(["vals_sorted"])["vals_sorted"], dbg_full["vals_sorted"])
    finally:
        sc.close()


@pytest.mark.parametrize("variant", ["sky", "dynamics", "band", "state"])
def test_lazy_lists_with_the_other_render_modes(variant):
    wl = make_config(1, n=150_000)
    cam, t = wl.cameras[0], 0.3
    sc = _scene(wl, 0.08)
    kw = {}
    try:
        if variant == "sky":
            sc.set_sky(sky_cubemap(8, 3))
        elif variant == "dynamics":
            kw = dict(target="dynamics")
        elif variant == "band":
            sc.set_tile_rows(7, 23)
        elif variant == "state":
            kw = dict(dt=0.02, rho_min=0.2)
        outs = {}
        for k in (0, 1, 3):
            sc.set_option(pvg.OPT_LAZY_CHUNKS, k)
            o = (torch.zeros((3, cam.height, cam.width), device="cuda"), torch.zeros((cam.height, cam.width), device="cuda"),
                 torch.zeros((cam.height, cam.width), device="cuda"))
            outs[k] = [x.clone() for x in sc.render(cam, t, out=o, **kw)]
        torch.cuda.synchronize()
        assert sc.frame_stats()["parked_tiles"] >= 0
        for k in (1, 3):
            for a, b in zip(outs[0], outs[k]):
                assert torch.equal(a, b), (variant, k)
    finally:
        sc.close()


def test_non_finite_sh_coefficients_are_culled_the_same_way():
    """The geometry-only preprocess of the lazy mode must still cull a Gaussian whose COLOUR is not finite (P11): the
    flagged Gaussians evaluate their SH there. Parity (P), (I), (R) against the oracle in the default (lazy)
    configuration, and images bit-identical to the eager mode."""
    from test_gpu_parity import full_parity
    wl = make_config(1, n=40_000)
    s = wl.scene
    sh = s.sh.copy()
    rng = np.random.default_rng(5)
    bad = rng.choice(s.n, size=600, replace=False)
    sh[bad[:200], rng.integers(0, 16, 200), rng.integers(0, 3, 200)] = np.nan
    sh[bad[200:400], rng.integers(0, 16, 200), rng.integers(0, 3, 200)] = np.inf
    sh[bad[400:], 0, :] = -np.inf
    import dataclasses
    scene = dataclasses.replace(s, sh=sh)
    cam, t = wl.cameras[0], 0.6
    st = full_parity(scene, cam, t, end_to_end=False)
    assert st["I"]["M"] > 0
    sc = pvg.Scene.from_workload_scene(scene)
    try:
        eager, _, _ = _render(sc, 0, cam, t)
        lazy, _, _ = _render(sc, 2, cam, t)
        for a, b in zip(eager, lazy):
            assert torch.equal(a, b)
        # (a colour of -inf or NaN clamps to 0 and survives, +inf is culled: what matters is that the oracle agrees,
        # which full_parity has checked Gaussian by Gaussian)
        dbg = sc.debug(["counts"])
        print("culled among the Gaussians with non-finite coefficients:", int((dbg["counts"][bad] == 0).sum()), "of", len(bad))
    finally:
        sc.close()
