"""Counter-based, order-independent generators for BASELINE.json's five configs.

Recipe (DESIGN.md §"Input recipe"):
  u64   = splitmix64(splitmix64(seed * K + stream) + index)
  U[0,1) = (u64 >> 11) * 2**-53
  N(0,1) = Box-Muller in float64 on the uniforms at indices (2i, 2i+1)
One stream per attribute, so every array is a pure function of
(seed, stream, index) and identical on every machine. All scene arrays are
rounded to float32 once, here, and both the oracle and the CUDA library read
those same float32 values.

These inputs STAND IN for the paper's Waymo/KITTI scenes,
which are not available: point count ~1e6 with a near/far mix, five cameras,
~50 timestamps per clip at l = 0.2.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence

import numpy as np

_K = np.uint64(0x9E3779B97F4A7C15)
_MASK = (1 << 64) - 1

# attribute -> stream id
STREAMS = {
    "x": 1, "y": 2, "z": 3, "scale": 4, "quat": 5, "opacity": 6, "sh_dc": 7,
    "sh_rest": 8, "dyn": 9, "vel": 10, "tau": 11, "beta": 12, "near": 13,
    "azimuth": 14, "scale_far": 15,
}


def splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output step on an array of uint64 states."""
    with np.errstate(over="ignore"):
        z = (x.astype(np.uint64) + _K)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def _stream_base(seed: int, stream: int) -> np.uint64:
    s = (seed * 0x9E3779B97F4A7C15 + stream) & _MASK
    return splitmix64(np.array([s], dtype=np.uint64))[0]


def rng_uniform(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """float64 U[0,1) for counters offset .. offset+n-1 of (seed, stream)."""
    base = _stream_base(seed, stream)
    idx = np.arange(offset, offset + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        u = splitmix64(base + idx)
    return (u >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def rng_normal(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """float64 N(0,1) number i from uniforms 2i, 2i+1 of (seed, stream)."""
    u = rng_uniform(seed, stream, 2 * n, 2 * offset)
    u1 = 1.0 - u[0::2]            # (0,1]
    u2 = u[1::2]
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


@dataclass
class Camera:
    """Pinhole camera. world_to_cam is row-major 3x4 [R|T], p_cam = R p_world + T,
    +z forward, +x right, +y down; pixel (i,j) centre at (i+0.5, j+0.5)."""
    width: int
    height: int
    fx: float
    fy: float
    cx: float
    cy: float
    world_to_cam: np.ndarray = field(default_factory=lambda: np.array(
        [1, 0, 0, 0, 0, 1, 0, 0, 0, 0, 1, 0], dtype=np.float32))
    znear: float = 0.2
    bg: Sequence[float] = (0.0, 0.0, 0.0)
    name: str = "front"


@dataclass
class Scene:
    mu: np.ndarray        # [n,3] f32
    quat: np.ndarray      # [n,4] f32 (w,x,y,z), unit
    scale: np.ndarray     # [n,3] f32 activated std-devs
    opacity: np.ndarray   # [n]   f32 activated in (0,1)
    sh: np.ndarray        # [n,16,3] f32
    tau: np.ndarray       # [n]   f32
    beta: np.ndarray      # [n]   f32
    vel: np.ndarray       # [n,3] f32
    cycle: float = 0.2
    sh_degree: int = 3

    @property
    def n(self) -> int:
        return int(self.mu.shape[0])

    def arrays(self) -> Dict[str, np.ndarray]:
        return dict(mu=self.mu, quat=self.quat, scale=self.scale, opacity=self.opacity,
                    sh=self.sh, tau=self.tau, beta=self.beta, vel=self.vel)


@dataclass
class Workload:
    config_id: int
    seed: int
    scene: Scene
    cameras: List[Camera]
    timestamps: List[float]
    description: str

    def frames(self):
        """(camera, t) pairs in render order."""
        for cam in self.cameras:
            for t in self.timestamps:
                yield cam, t


CONFIG_IDS = (0, 1, 2, 3, 4)

_DEFAULT_N = {0: 4096, 1: 200_000, 2: 1_000_000, 3: 3_000_000, 4: 6_000_000}


def pinhole_camera(width: int, height: int, f: float, yaw_deg: float = 0.0,
                   name: str = "front") -> Camera:
    """Camera at the origin; camera->world = R_y(yaw), +yaw turns toward +x."""
    psi = math.radians(yaw_deg)
    c, s = math.cos(psi), math.sin(psi)
    r_c2w = np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]], dtype=np.float64)
    r_w2c = r_c2w.T
    w2c = np.concatenate([r_w2c, np.zeros((3, 1))], axis=1).astype(np.float32).reshape(12)
    return Camera(width, height, float(f), float(f), width / 2.0, height / 2.0, w2c, 0.2,
                  (0.0, 0.0, 0.0), name)


def _f32(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _common(seed: int, n: int, dyn_frac: float):
    """Attributes shared by all configs (SURVEY.md §8(d) 'Common to all configs')."""
    q = rng_normal(seed, STREAMS["quat"], 4 * n).reshape(n, 4)
    q /= np.maximum(np.linalg.norm(q, axis=1, keepdims=True), 1e-12)
    o = 1.0 / (1.0 + np.exp(-rng_normal(seed, STREAMS["opacity"], n)))
    sh = np.empty((n, 16, 3), dtype=np.float32)
    sh[:, 0, :] = (0.5 * rng_normal(seed, STREAMS["sh_dc"], 3 * n)).reshape(n, 3)
    chunk = 1 << 18
    for s0 in range(0, n, chunk):                      # bounded temporaries
        m = min(chunk, n - s0)
        sh[s0:s0 + m, 1:, :] = (0.05 * rng_normal(seed, STREAMS["sh_rest"], 45 * m, 45 * s0)
                                ).reshape(m, 15, 3)
    tau = rng_uniform(seed, STREAMS["tau"], n)
    dyn = rng_uniform(seed, STREAMS["dyn"], n) < dyn_frac
    return q, o, sh, tau, dyn


def make_scene(config_id: int, n: Optional[int] = None, seed: Optional[int] = None) -> Scene:
    """Scene arrays of BASELINE.json config `config_id`; `n` overrides the point count
    (same distributions, used for reduced-size parity cases)."""
    if config_id not in CONFIG_IDS:
        raise ValueError(f"unknown config {config_id}")
    n = _DEFAULT_N[config_id] if n is None else int(n)
    seed = config_id if seed is None else int(seed)

    if config_id in (0, 1):
        dyn_frac = 0.3 if config_id == 0 else 0.2
        zmax = 20.0 if config_id == 0 else 80.0
        s_mu, s_sd = (-2.5, 0.5) if config_id == 0 else (-2.0, 0.7)
        q, o, sh, tau, dyn = _common(seed, n, dyn_frac)
        x = -3.0 + 6.0 * rng_uniform(seed, STREAMS["x"], n)
        y = -3.0 + 6.0 * rng_uniform(seed, STREAMS["y"], n)
        z = 2.0 + (zmax - 2.0) * rng_uniform(seed, STREAMS["z"], n)
        mu = np.stack([x, y, z], axis=1)
        scale = np.exp(s_mu + s_sd * rng_normal(seed, STREAMS["scale"], 3 * n)).reshape(n, 3)
        vel = np.where(dyn[:, None], rng_normal(seed, STREAMS["vel"], 3 * n).reshape(n, 3), 0.0)
        beta = np.where(dyn, np.exp(-1.5 + 0.3 * rng_normal(seed, STREAMS["beta"], n)), 1e3)
    else:
        q, o, sh, tau, dyn = _common(seed, n, 0.15)
        near = rng_uniform(seed, STREAMS["near"], n) < 0.7
        uz = rng_uniform(seed, STREAMS["z"], n)
        rng_near = 2.0 + 58.0 * uz
        rng_far = 60.0 * np.exp(uz * math.log(1000.0 / 60.0))          # log-uniform[60,1000]
        rho = np.where(near, rng_near, rng_far)
        g = rng_normal(seed, STREAMS["scale"], 3 * n).reshape(n, 3)
        s_near = np.exp(-2.0 + 0.6 * g)
        s_far = np.exp(0.5 * g) * (rho[:, None] / 100.0)
        scale = np.where(near[:, None], s_near, s_far)
        b = -0.4 + 0.8 * rng_uniform(seed, STREAMS["y"], n)
        if config_id == 4:
            scale = scale * 1.5
            phi = np.radians(-120.0 + 240.0 * rng_uniform(seed, STREAMS["azimuth"], n))
            mu = np.stack([rho * np.sin(phi), b * rho, rho * np.cos(phi)], axis=1)
        else:
            a = -0.6 + 1.2 * rng_uniform(seed, STREAMS["x"], n)
            mu = np.stack([a * rho, b * rho, rho], axis=1)
        vel = np.zeros((n, 3))
        vel[:, 0] = np.where(dyn, 5.0 * rng_normal(seed, STREAMS["vel"], n), 0.0)
        beta = np.where(dyn, np.exp(-1.0 + 0.4 * rng_normal(seed, STREAMS["beta"], n)), 1e3)

    return Scene(_f32(mu), _f32(q), _f32(scale), _f32(o), sh, _f32(tau), _f32(beta), _f32(vel),
                 cycle=0.2, sh_degree=3)


def make_config(config_id: int, n: Optional[int] = None, seed: Optional[int] = None) -> Workload:
    """Scene + cameras + timestamps of BASELINE.json config `config_id`."""
    scene = make_scene(config_id, n, seed)
    seed = config_id if seed is None else int(seed)
    if config_id == 0:
        cams = [pinhole_camera(128, 96, 100.0)]
        ts = [0.0, 0.37, 0.5]
        desc = "cfg0 tiny: 4096 Gaussians, 128x96, t in {0,0.37,0.5}"
    elif config_id == 1:
        cams = [pinhole_camera(960, 640, 700.0)]
        ts = [0.5]
        desc = "cfg1 mid: 200k Gaussians, 960x640, t=0.5"
    elif config_id == 2:
        cams = [pinhole_camera(1920, 1280, 2000.0)]
        ts = [0.5]
        desc = "cfg2 urban frame: 1M Gaussians, 1920x1280, t=0.5"
    elif config_id == 3:
        cams = [pinhole_camera(1920, 1280, 2000.0)]
        ts = [k / 49.0 for k in range(50)]
        desc = "cfg3 time sweep: 3M Gaussians, 1920x1280, 50 timestamps in [0,1]"
    else:
        cams = [pinhole_camera(1920, 1280, 2000.0, 0.0, "front")]
        for yaw in (45.0, -45.0, 90.0, -90.0):
            cams.append(pinhole_camera(1920, 886, 2000.0, yaw, f"side{int(yaw):+d}"))
        ts = [0.25, 0.75]
        desc = "cfg4 stress: 6M Gaussians x1.5 scale, 5 cameras, t in {0.25,0.75}"
    if n is not None:
        desc += f" [n overridden to {scene.n}]"
    return Workload(config_id, seed, scene, cams, ts, desc)


def sky_cubemap(res: int = 256, seed: int = 0) -> np.ndarray:
    """Synthetic sky for the cube-map background (the trained map is not available): a smooth
    function of the world direction -- horizon-to-zenith gradient (+y is down, so up is -y) plus a sun lobe --
    sampled at the texel centres of the layout include/pvg.h documents: cube[face][j][i], face = 2 a + (d_a < 0),
    u = d_b / |d_a| = (2 i + 1) / res - 1, v = d_c / |d_a| = (2 j + 1) / res - 1, (b, c) = next axes in cyclic order.
    Returns float32 [6, res, res, 3]."""
    c = (2.0 * np.arange(res, dtype=np.float64) + 1.0) / res - 1.0
    u, v = np.meshgrid(c, c, indexing="xy")            # u varies along i (last index), v along j
    sun = np.array([0.3 + 0.1 * seed, -0.5, 0.8])
    sun /= np.linalg.norm(sun)
    cube = np.empty((6, res, res, 3), dtype=np.float32)
    for face in range(6):
        a, sign = face // 2, (1.0 if face % 2 == 0 else -1.0)
        d = np.empty((res, res, 3))
        d[..., a] = sign
        d[..., (a + 1) % 3] = u
        d[..., (a + 2) % 3] = v
        d /= np.linalg.norm(d, axis=-1, keepdims=True)
        up = -d[..., 1]
        t = np.clip(0.5 + 0.5 * up, 0.0, 1.0)
        base = np.stack([0.75 - 0.45 * t, 0.82 - 0.32 * t, 0.95 - 0.10 * t], -1)
        lobe = np.clip((d * sun).sum(-1), 0.0, 1.0) ** 64
        cube[face] = (base + lobe[..., None] * np.array([1.0, 0.9, 0.6])).astype(np.float32)
    return cube
