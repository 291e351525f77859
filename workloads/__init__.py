"""Seeded synthetic inputs for the PVG forward render (BASELINE.json configs 0-4).

This package serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic: it only draws scene parameters, cameras and
timestamps from the distributions DESIGN.md states. numpy only.
"""
from .gen import (  # noqa: F401
    Camera,
    Scene,
    Workload,
    CONFIG_IDS,
    make_config,
    make_scene,
    pinhole_camera,
    rng_uniform,
    rng_normal,
    sky_cubemap,
    splitmix64,
)
