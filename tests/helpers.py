"""Shared test helpers: tiny hand-built scenes and records. No method arithmetic."""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np

from workloads import Camera, Scene, pinhole_camera  # noqa: F401


def one_scene(mu=(0, 0, 5), quat=(1, 0, 0, 0), scale=(0.1, 0.1, 0.1), opacity=0.8, sh=None,
              tau=0.0, beta=np.inf, vel=(0, 0, 0), cycle=0.2, sh_degree=3) -> Scene:
    """Scene from per-point lists (each argument may be a single point or a list of points)."""
    mu = np.atleast_2d(np.asarray(mu, dtype=np.float32))
    n = mu.shape[0]

    def rows(a, k):
        a = np.asarray(a, dtype=np.float32)
        if a.ndim == 1 and k > 1:
            a = np.tile(a, (n, 1))
        elif a.ndim == 0:
            a = np.full((n,), float(a), dtype=np.float32)
        return np.ascontiguousarray(a.reshape((n, k) if k > 1 else (n,)), dtype=np.float32)

    if sh is None:
        sh = np.zeros((n, 16, 3), dtype=np.float32)
    sh = np.ascontiguousarray(np.asarray(sh, dtype=np.float32).reshape(n, 16, 3))
    return Scene(mu, rows(quat, 4), rows(scale, 3), rows(opacity, 1), sh, rows(tau, 1), rows(beta, 1),
                 rows(vel, 3), cycle=cycle, sh_degree=sh_degree)


def record_row(mx, my, z, op, a, b, c, rgb=(1.0, 1.0, 1.0), hx=1e4, hy=1e4) -> np.ndarray:
    """One fp32 record row (mx,my,z,op | a,b,c,hx | r,g,b,hy)."""
    return np.array([mx, my, z, op, a, b, c, hx, rgb[0], rgb[1], rgb[2], hy], dtype=np.float32)


def cam_simple(width=64, height=48, f=50.0, bg=(0.0, 0.0, 0.0)) -> Camera:
    cam = pinhole_camera(width, height, f)
    cam.bg = tuple(bg)
    return cam


def ns(**kw):
    return SimpleNamespace(**kw)
