"""CPU oracle for the PVG forward render -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over oracle/pvg_oracle.cpp (plain C++, double precision,
written from the paper; see that file's header for citations and pins). Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package. It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import build as _build

SLOTS = dict(mu=slice(0, 3), op=3, pcam=slice(4, 7), sigma=slice(7, 13), cov=slice(13, 16),
             conic=slice(16, 19), mean=slice(19, 21), ext=slice(21, 23), rgb=slice(23, 26),
             cull=26, rect=slice(27, 31), count=31)
CULL_REASONS = {0: "valid", 1: "opacity", 2: "near", 3: "det", 4: "rect", 5: "nonfinite", 6: "staticness"}


class _Cam(C.Structure):
    _fields_ = [("width", C.c_int), ("height", C.c_int), ("fx", C.c_double), ("fy", C.c_double),
                ("cx", C.c_double), ("cy", C.c_double), ("w2c", C.c_double * 12),
                ("znear", C.c_double), ("bg", C.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.oracle_tile_counts.restype = C.c_uint64
        L.oracle_tile_list.restype = C.c_uint64
        L.oracle_tile_counts_ex.restype = C.c_uint64
        L.oracle_tile_list_ex.restype = C.c_uint64
        L.oracle_record_stride.restype = C.c_int
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _cam(cam) -> _Cam:
    c = _Cam()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    w2c = np.asarray(cam.world_to_cam, dtype=np.float64).reshape(12)
    for i in range(12):
        c.w2c[i] = float(w2c[i])
    c.znear = float(cam.znear)
    for i in range(3):
        c.bg[i] = float(cam.bg[i])
    return c


def _f32(a, shape):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.shape == shape, (a.shape, shape)
    return a


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(C.c_int(int(n)))


def preprocess(mu, quat, scale, opacity, sh, tau, beta, vel, cycle, sh_degree, cam, t, dt=0.0, rho_min=0.0,
               rho_max=float("inf")):
    """Oracle-P. Returns (wide [n,32] float64, rec32 [n,12] float32).
    dt != 0: the temporal-smoothing state H^(t) built from t - dt (Eq. 12); rho_min / rho_max: staticness filter."""
    n = int(np.asarray(mu).shape[0])
    mu = _f32(mu, (n, 3)); quat = _f32(quat, (n, 4)); scale = _f32(scale, (n, 3))
    opacity = _f32(opacity, (n,)); sh = _f32(sh, (n, 16, 3)); tau = _f32(tau, (n,))
    beta = _f32(beta, (n,)); vel = _f32(vel, (n, 3))
    wide = np.empty((n, 32), dtype=np.float64)
    rec = np.empty((n, 12), dtype=np.float32)
    c = _cam(cam)
    lib().oracle_preprocess_state(C.c_uint64(n), _p(mu), _p(quat), _p(scale), _p(opacity), _p(sh), _p(tau),
                                  _p(beta), _p(vel), C.c_double(float(cycle)), C.c_int(int(sh_degree)),
                                  C.byref(c), C.c_double(float(t)), C.c_double(float(dt)), C.c_double(float(rho_min)),
                                  C.c_double(float(rho_max)), _p(wide), _p(rec))
    return wide, rec


def preprocess_scene(scene, cam, t, dt=0.0, rho_min=0.0, rho_max=float("inf")):
    """Oracle-P on an object with the workloads.Scene attribute names."""
    return preprocess(scene.mu, scene.quat, scene.scale, scene.opacity, scene.sh, scene.tau,
                      scene.beta, scene.vel, scene.cycle, scene.sh_degree, cam, t, dt, rho_min, rho_max)


def sh_basis(d: Sequence[float]) -> np.ndarray:
    d = np.ascontiguousarray(d, dtype=np.float64)
    Y = np.empty(16, dtype=np.float64)
    lib().oracle_sh_basis(_p(d), _p(Y))
    return Y


def tile_counts(rec, width, height, exact: bool = False):
    """Integer chain step 1. Returns (rects [n,4] int32 inclusive, counts [n] uint32, M). exact: count only the tiles
    of the rectangle that pass the ellipse-versus-tile test P13."""
    rec = np.ascontiguousarray(rec, dtype=np.float32)
    n = rec.shape[0]
    assert rec.shape == (n, 12)
    rects = np.empty((n, 4), dtype=np.int32)
    counts = np.empty(n, dtype=np.uint32)
    M = lib().oracle_tile_counts_ex(C.c_uint64(n), _p(rec), C.c_int(width), C.c_int(height), C.c_int(1 if exact else 0),
                                    _p(rects), _p(counts))
    return rects, counts, int(M)


def tile_hist(rec, width, height, exact: bool = False) -> np.ndarray:
    """List length of every tile [tiles] uint64 (row-major), from the per-Gaussian tile sets (no sort)."""
    rec = np.ascontiguousarray(rec, dtype=np.float32)
    n = rec.shape[0]
    ntiles = ((width + 15) // 16) * ((height + 15) // 16)
    out = np.zeros(ntiles, dtype=np.uint64)
    lib().oracle_tile_hist_ex(C.c_uint64(n), _p(rec), C.c_int(width), C.c_int(height), C.c_int(1 if exact else 0), _p(out))
    return out


def keys(rec, width, height, order_mode=0, exact: bool = False):
    """Integer chain step 2 (offsets, unsorted list, std::stable_sort, ranges)."""
    rec = np.ascontiguousarray(rec, dtype=np.float32)
    n = rec.shape[0]
    _, _, M = tile_counts(rec, width, height, exact)
    ntiles = ((width + 15) // 16) * ((height + 15) // 16)
    out = dict(M=M,
               offsets=np.zeros(n, dtype=np.uint64),
               keys_unsorted=np.zeros(M, dtype=np.uint64), vals_unsorted=np.zeros(M, dtype=np.uint32),
               keys_sorted=np.zeros(M, dtype=np.uint64), vals_sorted=np.zeros(M, dtype=np.uint32),
               ranges=np.zeros((ntiles, 2), dtype=np.uint32))
    lib().oracle_keys_ex(C.c_uint64(n), _p(rec), C.c_int(width), C.c_int(height), C.c_int(order_mode),
                         C.c_int(1 if exact else 0), _p(out["offsets"]), _p(out["keys_unsorted"]), _p(out["vals_unsorted"]),
                      _p(out["keys_sorted"]), _p(out["vals_sorted"]), _p(out["ranges"]))
    return out


def tile_list(rec, width, height, tile, exact: bool = False):
    """Sorted instance list of one tile, computed directly. Returns (keys u64, vals u32)."""
    rec = np.ascontiguousarray(rec, dtype=np.float32)
    n = rec.shape[0]
    L = lib()
    ex = C.c_int(1 if exact else 0)
    cnt = int(L.oracle_tile_list_ex(C.c_uint64(n), _p(rec), C.c_int(width), C.c_int(height),
                                    C.c_uint32(tile), ex, C.c_uint64(0), None, None))
    k = np.zeros(cnt, dtype=np.uint64)
    v = np.zeros(cnt, dtype=np.uint32)
    if cnt:
        L.oracle_tile_list_ex(C.c_uint64(n), _p(rec), C.c_int(width), C.c_int(height), C.c_uint32(tile), ex,
                              C.c_uint64(cnt), _p(k), _p(v))
    return k, v


def render(rec, width, height, bg=(0.0, 0.0, 0.0), mode="binned", tiles: Optional[Sequence[int]] = None,
           tie_budget: bool = False, slack=None):
    """Oracle-R on an fp32 record. mode 'brute' or 'binned'. Returns dict of float64
    images: rgb [3,H,W], depth, alpha, budget, cond, derived [H,W], plus visited / contributed.
    slack [n,6] (end-to-end comparison only): how far another fp32 record of the same scene may lie from `rec`,
    per Gaussian (d mx, d my, d conic, d ln o~, d colour, d z in ulps); `derived` is the per-pixel allowance it
    propagates to, and the fragile windows (alpha cutoff, T stop, depth ties) widen by the same uncertainty."""
    rec = np.ascontiguousarray(rec, dtype=np.float32)
    n = rec.shape[0]
    assert rec.shape == (n, 12)
    H, W = int(height), int(width)
    rgb = np.empty((3, H, W)); depth = np.empty((H, W)); alpha = np.empty((H, W))
    budget = np.empty((H, W)); cond = np.empty((H, W)); derived = np.zeros((H, W))
    sl = None
    if slack is not None:
        sl = np.ascontiguousarray(slack, dtype=np.float64)
        assert sl.shape == (n, 6), sl.shape
    stats = np.zeros(2, dtype=np.uint64)
    bg = np.ascontiguousarray(bg, dtype=np.float64)
    tl, ntl = None, 0
    if tiles is not None:
        tl_arr = np.ascontiguousarray(tiles, dtype=np.uint32)
        tl, ntl = _p(tl_arr), tl_arr.shape[0]
    lib().oracle_render(C.c_uint64(n), _p(rec), C.c_int(W), C.c_int(H), _p(bg),
                        C.c_int({"brute": 0, "binned": 1, "binned_exact": 2}[mode]), tl, C.c_uint64(ntl),
                        C.c_int(1 if tie_budget else 0), _p(rgb), _p(depth), _p(alpha), _p(budget),
                        _p(cond), _p(stats), _p(sl) if sl is not None else None, _p(derived))
    # c_max: the colour scale of budget and cond (largest colour of a non-culled Gaussian or of the background)
    live = rec[:, 3] > 0
    c_max = float(max(rec[live, 8:11].max(initial=0.0), float(np.max(bg))))
    return dict(rgb=rgb, depth=depth, alpha=alpha, budget=budget, cond=cond, derived=derived,
                visited=int(stats[0]), contributed=int(stats[1]), c_max=c_max)


def sky_sample(cube, d):
    """f_sky(d): bilinear lookup in a cube map [6][R][R][3] (face = 2 axis + (d_axis < 0))."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    res = cube.shape[1]
    assert cube.shape == (6, res, res, 3)
    d = np.ascontiguousarray(d, dtype=np.float64)
    out = np.empty(3, dtype=np.float64)
    lib().oracle_sky_sample(_p(cube), C.c_int(res), _p(d), _p(out))
    return out


def sky_composite(cam, cube, rgb, alpha):
    """C_f = C + (1 - O) f_sky(d) on an Oracle-R image rendered with bg = 0. Returns a new rgb."""
    cube = np.ascontiguousarray(cube, dtype=np.float32)
    res = cube.shape[1]
    assert cube.shape == (6, res, res, 3)
    out = np.array(rgb, dtype=np.float64, order="C", copy=True)
    alpha = np.ascontiguousarray(alpha, dtype=np.float64)
    c = _cam(cam)
    lib().oracle_sky_composite(C.byref(c), _p(cube), C.c_int(res), _p(out), _p(alpha))
    return out


def dynamics(scene, cam):
    """(vbar in camera axes, clamp(rho, 0, 2)) per point: float64 [n, 4] (Eq. 10)."""
    n = int(scene.mu.shape[0])
    beta = _f32(scene.beta, (n,)); vel = _f32(scene.vel, (n, 3))
    out = np.empty((n, 4), dtype=np.float64)
    c = _cam(cam)
    lib().oracle_dynamics(C.c_uint64(n), _p(beta), _p(vel), C.c_double(float(scene.cycle)), C.byref(c), _p(out))
    return out
