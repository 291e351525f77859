"""Writes tests/golden/cfg0_oracle.json from the oracle alone (never from the CUDA path)."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from workloads import make_config  # noqa: E402


def summary():
    wl = make_config(0)
    cam = wl.cameras[0]
    out = {}
    for t in wl.timestamps:
        wide, rec = oracle.preprocess_scene(wl.scene, cam, t)
        _, counts, M = oracle.tile_counts(rec, cam.width, cam.height)
        img = oracle.render(rec, cam.width, cam.height, mode="binned")
        out[repr(t)] = dict(
            survivors=int((rec[:, 3] > 0).sum()), M=int(M),
            cull_hist=[int(x) for x in np.bincount(wide[:, 26].astype(int), minlength=6)],
            rgb_sum=float(img["rgb"].sum()), depth_sum=float(img["depth"].sum()),
            alpha_sum=float(img["alpha"].sum()), contributed=int(img["contributed"]),
            pixel_40_60=[float(img["rgb"][c, 40, 60]) for c in range(3)])
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.json")
    with open(path, "w") as f:
        json.dump(summary(), f, indent=1, sort_keys=True)
    print("wrote", path)
