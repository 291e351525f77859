"""CPU-only checks of the C-ABI boundary: the library builds and loads without a GPU, exports
every symbol include/pvg.h declares, the ctypes mirrors match the C structs, and argument
validation that needs no device works. No compute call is made here."""
import ctypes as C
import os
import re
import subprocess
import tempfile

import numpy as np
import pytest

import paper_2311_18561_b200 as pvg
from paper_2311_18561_b200 import build as pvg_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pvg.h")


@pytest.fixture(scope="module")
def lib():
    pvg_build.build()
    return pvg.load_library()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pvg_[a-z0-9_]+)\s*\(", src)) - {"pvg_alloc_fn", "pvg_free_fn"})


def test_header_functions_match_binding_list():
    assert declared_functions() == sorted(pvg.EXPORTS)


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), name


def test_no_torch_or_cpp_types_cross_the_boundary():
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)     # code only, comments stripped
    assert "torch" not in src.lower() and "std::" not in src and "at::" not in src and "#include <cuda" not in src
    out = subprocess.run(["nm", "-D", "--defined-only", pvg.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = [l.split()[-1] for l in out.splitlines() if " T " in l]
    assert set(pvg.EXPORTS) <= set(exported)


def test_struct_layouts_match_c(lib):
    prog = r'''
#include <stdio.h>
#include <stddef.h>
#include "pvg.h"
int main(void) {
  printf("%zu %zu %zu %zu\n", sizeof(pvg_scene_desc), offsetof(pvg_scene_desc, vel), offsetof(pvg_scene_desc, cycle), offsetof(pvg_scene_desc, pointers_on_device));
  printf("%zu %zu %zu %zu\n", sizeof(pvg_camera), offsetof(pvg_camera, world_to_cam), offsetof(pvg_camera, znear), offsetof(pvg_camera, bg));
  printf("%zu %zu %zu %zu\n", sizeof(pvg_debug), offsetof(pvg_debug, record), offsetof(pvg_debug, keys_sorted), offsetof(pvg_debug, ranges));
  printf("%d %d\n", PVG_NUM_STAGES, PVG_ERR_BAD_OPTION);
  printf("%zu %zu %zu %d\n", sizeof(pvg_state), offsetof(pvg_state, rho_max), offsetof(pvg_state, target), PVG_ERR_BAD_STATE);
  return 0;
}'''
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "t.c"), "w").write(prog)
        subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(d, "t"),
                        os.path.join(d, "t.c")], check=True)   # also proves the header is plain C
        rows = [list(map(int, l.split())) for l in subprocess.run([os.path.join(d, "t")], capture_output=True, text=True, check=True).stdout.splitlines()]
    S, Cm, D = pvg.SceneDesc, pvg.CameraC, pvg.DebugC
    assert rows[0] == [C.sizeof(S), S.vel.offset, S.cycle.offset, S.pointers_on_device.offset]
    assert rows[1] == [C.sizeof(Cm), Cm.world_to_cam.offset, Cm.znear.offset, Cm.bg.offset]
    assert rows[2] == [C.sizeof(D), D.record.offset, D.keys_sorted.offset, D.ranges.offset]
    assert rows[3] == [pvg.NUM_STAGES, -7]
    St = pvg.StateC
    assert rows[4] == [C.sizeof(St), St.rho_max.offset, St.target.offset, -8]


def test_argument_validation_without_device(lib):
    assert lib.pvg_version() >= 100
    assert lib.pvg_strerror(0) == b"ok" and b"camera" in lib.pvg_strerror(-3)
    h = C.c_void_p()
    assert lib.pvg_create_scene(None, C.byref(h)) == -1
    a = np.zeros(48, dtype=np.float32)
    p = a.ctypes.data
    for kw, code in ((dict(n=0), -2), (dict(cycle=0.0), -2), (dict(cycle=float("nan")), -2), (dict(sh_degree=4), -2),
                     (dict(mu=None), -1)):
        args = dict(n=1, mu=p, quat=p, scale=p, opacity=p, sh=p, tau=p, beta=p, vel=p, cycle=0.2, sh_degree=3,
                    pointers_on_device=0)
        args.update(kw)
        d = pvg.SceneDesc(**args)
        assert lib.pvg_create_scene(C.byref(d), C.byref(h)) == code, kw
    assert lib.pvg_destroy(None) == -1 and lib.pvg_set_option(None, 1, 0) == -1
    assert lib.pvg_render(None, None, 0.0, None, None, None) == -1


def test_binding_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    z = np.zeros((1, 3), np.float32)
    with pytest.raises(pvg.PvgError):
        pvg.Scene(z, np.zeros((1, 4), np.float32), z, np.zeros(1, np.float32), np.zeros((1, 16, 3), np.float32),
                  np.zeros(1, np.float32), np.ones(1, np.float32), z)


def test_camera_marshalling():
    from workloads import pinhole_camera
    cam = pinhole_camera(1920, 886, 2000.0, 45.0)
    c = pvg.camera_struct(cam)
    assert (c.width, c.height, c.fx, c.cx, c.cy) == (1920, 886, 2000.0, 960.0, 443.0)
    assert np.allclose(list(c.world_to_cam), cam.world_to_cam) and abs(c.znear - 0.2) < 1e-7
