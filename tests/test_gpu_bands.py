"""Tile-row bands (include/pvg.h PVG_OPT_TILE_ROW_BEGIN / END): a render restricted to
the tile rows [begin, end) duplicates into, sorts and composites the tiles of that band only.
What is unique and checked bit for bit:
  * bands rendered one after another into the same images give exactly the full frame (which the other
    parity tests tie to the oracle), and rows outside the band are not written;
  * the band's per-Gaussian counts are the areas of the ORACLE's rectangles clamped to the band, its M their
    sum, and the sorted list of every tile of the band equals that tile's list in the full frame / the
    oracle's direct per-tile computation.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2311_18561_b200 as pvg
from paper_2311_18561_b200 import dist
from workloads import make_config

pytestmark = pytest.mark.gpu

MODES = {"blocks": dict(block=1, compact=1, presort=1), "compact": dict(block=0, compact=1, presort=1),
         "keys64": dict(block=0, compact=0, presort=0)}


def _set_mode(sc, mode):
    m = MODES[mode]
    sc.set_option(pvg.OPT_PRESORT_DEPTH, m["presort"])
    sc.set_option(pvg.OPT_COMPACT_KEYS, m["compact"])
    sc.set_option(pvg.OPT_BLOCK_BINS, m["block"])


def _nan_images(cam):
    return (torch.full((3, cam.height, cam.width), float("nan"), device="cuda"),
            torch.full((cam.height, cam.width), float("nan"), device="cuda"),
            torch.full((cam.height, cam.width), float("nan"), device="cuda"))


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("cfg,n,cam_i,parts", [(1, 60_000, 0, 3), (4, 20_000, 3, 8), (0, None, 0, 2)])
def test_bands_stitch_to_the_full_frame_bit_exactly(mode, cfg, n, cam_i, parts):
    wl = make_config(cfg, n=n)
    cam, t = wl.cameras[cam_i], 0.25
    TY = (cam.height + 15) // 16
    sc = pvg.Scene.from_workload_scene(wl.scene)
    try:
        _set_mode(sc, mode)
        full = [x.clone() for x in sc.render(cam, t)]
        out = _nan_images(cam)
        for r in range(parts):
            b, e = dist.band_rows(r, parts, TY)
            if b == e:
                continue
            sc.set_tile_rows(b, e)
            sc.render(cam, t, out=out)
            torch.cuda.synchronize()
            # nothing below the bands rendered so far has been written yet
            if e * 16 < cam.height:
                assert torch.isnan(out[1][e * 16:]).all() and torch.isnan(out[0][:, e * 16:]).all()
        for a, b_ in zip(full, out):
            assert torch.equal(a, b_)
        sc.set_tile_rows(0, 0)
        again = sc.render(cam, t)
        assert all(torch.equal(a, b_) for a, b_ in zip(full, again))
    finally:
        sc.close()


@pytest.mark.parametrize("mode", list(MODES))
def test_band_integer_chain_against_the_oracle(mode):
    wl = make_config(1, n=60_000)
    cam, t = wl.cameras[0], 0.5
    W, H = cam.width, cam.height
    TX, TY = (W + 15) // 16, (H + 15) // 16
    sc = pvg.Scene.from_workload_scene(wl.scene)
    try:
        _set_mode(sc, mode)
        sc.set_option(pvg.OPT_KEEP_UNSORTED, 1)
        sc.render(cam, t)
        whole = sc.debug(["record", "counts", "ranges", "vals_sorted"])
        b, e = 5, 13
        sc.set_tile_rows(b, e)
        sc.render(cam, t)
        band = sc.debug(["record", "counts", "ranges", "vals_sorted"])
    finally:
        sc.close()
    rects, counts, _ = oracle.tile_counts(whole["record"], W, H)
    v = counts > 0
    y0 = np.maximum(rects[:, 1].astype(np.int64), b)
    y1 = np.minimum(rects[:, 3].astype(np.int64), e - 1)
    area = np.where(v & (y0 <= y1), (rects[:, 2].astype(np.int64) - rects[:, 0] + 1) * (y1 - y0 + 1), 0)
    assert np.array_equal(band["counts"], area.astype(np.uint32))
    assert band["M"] == int(area.sum()) and 0 < band["M"] < whole["M"]
    # the record of a Gaussian that reaches the band is the full frame's; the others are culled (zeroed)
    wr, br = whole["record"].view(np.uint32), band["record"].view(np.uint32)
    assert np.array_equal(br[area > 0], wr[area > 0]) and not br[area == 0].any()
    # every tile: lists of the band's tiles as in the full frame, the others empty
    rw, rb = whole["ranges"].astype(np.int64), band["ranges"].astype(np.int64)
    ln_w, ln_b = rw[:, 1] - rw[:, 0], rb[:, 1] - rb[:, 0]
    in_band = np.zeros(TX * TY, dtype=bool)
    in_band[b * TX:e * TX] = True
    assert np.array_equal(ln_b, np.where(in_band, ln_w, 0))
    assert rb[b * TX, 0] == 0 and rb[e * TX - 1, 1] == band["M"]
    first, last = int(rw[b * TX, 0]), int(rw[e * TX - 1, 1])
    assert np.array_equal(band["vals_sorted"][:band["M"]], whole["vals_sorted"][first:last])
    for tl in (b * TX, b * TX + TX // 2, (e - 1) * TX + TX - 1, int(np.argmax(np.where(in_band, ln_w, -1)))):
        _, v_o = oracle.tile_list(whole["record"], W, H, tl)
        assert np.array_equal(band["vals_sorted"][rb[tl, 0]:rb[tl, 1]], v_o)


def test_band_options_validate():
    wl = make_config(0)
    cam = wl.cameras[0]
    TY = (cam.height + 15) // 16
    sc = pvg.Scene.from_workload_scene(wl.scene)
    try:
        with pytest.raises(pvg.PvgError):
            sc.set_option(pvg.OPT_TILE_ROW_BEGIN, -1)
        sc.set_tile_rows(TY, 0)                     # begins past the last tile row of this camera
        with pytest.raises(pvg.PvgError):
            sc.render(cam, 0.5)
        sc.set_tile_rows(TY - 1, 2048)              # END beyond the image = to the last row
        out = _nan_images(cam)
        sc.render(cam, 0.5, out=out)
        torch.cuda.synchronize()
        assert torch.isnan(out[2][:(TY - 1) * 16]).all() and not torch.isnan(out[2][(TY - 1) * 16:]).any()
    finally:
        sc.close()
