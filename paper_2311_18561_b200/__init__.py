"""paper_2311_18561_b200 -- Python binding of libpvg.so (include/pvg.h).

Argument marshalling only: every step of the render runs in the CUDA kernels of
csrc/. PyTorch provides device memory (caching-allocator hooks), the stream and
output tensors. There is no CPU fallback: if the library cannot be loaded, or no
CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("PVG_LIB") or os.path.join(_HERE, "libpvg.so")   # PVG_LIB: tuning builds only

PVG_OK = 0
STATUS = {0: "PVG_OK", -1: "PVG_ERR_NULL", -2: "PVG_ERR_BAD_DESC", -3: "PVG_ERR_BAD_CAMERA",
          -4: "PVG_ERR_OOM", -5: "PVG_ERR_INSTANCE_OVERFLOW", -6: "PVG_ERR_CUDA", -7: "PVG_ERR_BAD_OPTION", -8: "PVG_ERR_BAD_STATE",
          -9: "PVG_ERR_TOO_LARGE"}
OPT_PRESORT_DEPTH, OPT_KEEP_UNSORTED, OPT_KERNEL_EVENTS, OPT_COUNT_PAIRS, OPT_COMPACT_KEYS, OPT_BLOCK_BINS = 1, 2, 3, 4, 5, 6
OPT_BLEND_CULL, OPT_EVENT_STRIDE = 7, 8
OPT_TILE_ROW_BEGIN, OPT_TILE_ROW_END = 9, 10
OPT_LAZY_CHUNKS, OPT_LAZY_SLAB, OPT_EXACT_TILES, OPT_LAZY_DEPTH = 11, 12, 13, 14
STAGES = ("preprocess", "depth_sort", "duplicate", "sort", "ranges", "blend")
NUM_STAGES = len(STAGES)

# every symbol include/pvg.h declares
EXPORTS = ("pvg_set_allocator", "pvg_set_stream", "pvg_create_scene", "pvg_render", "pvg_render_host",
           "pvg_render_host_async", "pvg_wait_host", "pvg_render_state", "pvg_set_sky",
           "pvg_destroy", "pvg_fork_scene", "pvg_set_option", "pvg_debug_view", "pvg_stage_times_ms", "pvg_kernel_times_ms", "pvg_kernel_timeline_ms",
           "pvg_sort_pairs", "pvg_sort_pairs_static", "pvg_sort_pairs_static_max_n", "pvg_frame_stats", "pvg_blend_counters", "pvg_memcpy_d2h", "pvg_calibrate_fp32", "pvg_guard_bands", "pvg_check_guards", "pvg_strerror", "pvg_last_cuda_error", "pvg_version")


class PvgError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        super().__init__(f"{STATUS.get(code, code)}: {detail}")


class SceneDesc(C.Structure):
    _fields_ = [("n", C.c_uint64), ("mu", C.c_void_p), ("quat", C.c_void_p), ("scale", C.c_void_p),
                ("opacity", C.c_void_p), ("sh", C.c_void_p), ("tau", C.c_void_p), ("beta", C.c_void_p),
                ("vel", C.c_void_p), ("cycle", C.c_float), ("sh_degree", C.c_int),
                ("pointers_on_device", C.c_int)]


class CameraC(C.Structure):
    _fields_ = [("width", C.c_int), ("height", C.c_int), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("world_to_cam", C.c_float * 12),
                ("znear", C.c_float), ("bg", C.c_float * 3)]


class StateC(C.Structure):
    _fields_ = [("t", C.c_float), ("dt", C.c_float), ("rho_min", C.c_float), ("rho_max", C.c_float),
                ("target", C.c_int)]


class DebugC(C.Structure):
    _fields_ = [("n", C.c_uint64), ("num_instances", C.c_uint64), ("tiles_x", C.c_uint32),
                ("tiles_y", C.c_uint32), ("sort_begin_bit", C.c_uint32), ("sort_end_bit", C.c_uint32),
                ("record", C.c_void_p), ("counts", C.c_void_p), ("visit_order", C.c_void_p),
                ("offsets", C.c_void_p), ("keys_unsorted", C.c_void_p), ("vals_unsorted", C.c_void_p),
                ("keys_sorted", C.c_void_p), ("vals_sorted", C.c_void_p), ("ranges", C.c_void_p)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

_lib = None
_hooks = None  # keeps the ctypes callbacks alive


def load_library(path: Optional[str] = None):
    """dlopen libpvg.so (no CUDA call is made). Fails loudly if it has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise ImportError(f"{p} is missing: build it with `python -m paper_2311_18561_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(p)
    L.pvg_strerror.restype = C.c_char_p
    L.pvg_last_cuda_error.restype = C.c_char_p
    L.pvg_set_stream.argtypes = [C.c_void_p, C.c_void_p]
    L.pvg_create_scene.argtypes = [C.POINTER(SceneDesc), C.POINTER(C.c_void_p)]
    L.pvg_render.argtypes = [C.c_void_p, C.POINTER(CameraC), C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    L.pvg_render_state.argtypes = [C.c_void_p, C.POINTER(CameraC), C.POINTER(StateC), C.c_void_p, C.c_void_p, C.c_void_p]
    L.pvg_set_sky.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int]
    L.pvg_render_host.argtypes = [C.c_void_p, C.POINTER(CameraC), C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    L.pvg_render_host_async.argtypes = [C.c_void_p, C.POINTER(CameraC), C.c_float, C.c_void_p, C.c_void_p, C.c_void_p]
    L.pvg_wait_host.argtypes = [C.c_void_p]
    L.pvg_destroy.argtypes = [C.c_void_p]
    L.pvg_fork_scene.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
    L.pvg_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int64]
    L.pvg_debug_view.argtypes = [C.c_void_p, C.POINTER(DebugC)]
    L.pvg_stage_times_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    L.pvg_kernel_times_ms.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_int),
                                      C.POINTER(C.c_float)]
    L.pvg_kernel_timeline_ms.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_float),
                                         C.POINTER(C.c_float)]
    L.pvg_sort_pairs.argtypes = [C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                 C.c_void_p]
    L.pvg_sort_pairs_static.argtypes = [C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                        C.c_void_p]
    L.pvg_sort_pairs_static_max_n.restype = C.c_uint64
    L.pvg_sort_pairs_static_max_n.argtypes = []
    L.pvg_frame_stats.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
    L.pvg_blend_counters.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
    L.pvg_memcpy_d2h.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
    L.pvg_set_allocator.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.pvg_calibrate_fp32.argtypes = [C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.pvg_guard_bands.argtypes = [C.c_int]
    L.pvg_check_guards.argtypes = [C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    if path is None:
        _lib = L
    return L


def _check(rc: int):
    if rc != PVG_OK:
        L = load_library()
        detail = L.pvg_strerror(rc).decode()
        if rc in (-6, -9):
            detail += " | " + L.pvg_last_cuda_error().decode()
        raise PvgError(rc, detail)


def use_torch_allocator(enable: bool = True) -> None:
    """Route the library's device allocations through PyTorch's caching allocator."""
    global _hooks
    import torch
    L = load_library()
    if not enable:
        _check(L.pvg_set_allocator(None, None, None))
        _hooks = None
        return

    def _alloc(nbytes, stream, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream) if stream else None)
        except Exception:
            return 0

    def _free(ptr, _user):
        try:
            torch.cuda.caching_allocator_delete(ptr)
        except Exception:
            pass

    a, f = ALLOC_FN(_alloc), FREE_FN(_free)
    _check(L.pvg_set_allocator(C.cast(a, C.c_void_p), C.cast(f, C.c_void_p), None))
    _hooks = (a, f)


def camera_struct(cam) -> CameraC:
    """pvg_camera from any object with the fields of workloads.Camera."""
    c = CameraC()
    c.width, c.height = int(cam.width), int(cam.height)
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    w2c = np.asarray(cam.world_to_cam, dtype=np.float32).reshape(12)
    for i in range(12):
        c.world_to_cam[i] = float(w2c[i])
    c.znear = float(getattr(cam, "znear", 0.0))
    bg = getattr(cam, "bg", (0.0, 0.0, 0.0))
    for i in range(3):
        c.bg[i] = float(bg[i])
    return c


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


class Scene:
    """Owns a pvg_scene. Arrays may be numpy (host) or torch CUDA tensors (all one kind)."""

    def __init__(self, mu, quat, scale, opacity, sh, tau, beta, vel, cycle: float = 0.2, sh_degree: int = 3,
                 torch_allocator: bool = True):
        import torch
        if not torch.cuda.is_available():
            raise PvgError(-6, "no CUDA device: this package has no CPU fallback")
        self._L = load_library()
        if torch_allocator and _hooks is None:
            use_torch_allocator(True)
        arrs = [mu, quat, scale, opacity, sh, tau, beta, vel]
        shapes = [(3,), (4,), (3,), (), (16, 3), (), (), (3,)]
        on_dev = all(_is_torch(a) and a.is_cuda for a in arrs)
        n = int(arrs[0].shape[0])
        keep = []
        ptrs = []
        for a, shp in zip(arrs, shapes):
            if on_dev:
                a = a.detach().to(torch.float32).contiguous()
                assert tuple(a.shape) == (n,) + shp, (tuple(a.shape), shp)
                ptrs.append(a.data_ptr())
            else:
                if _is_torch(a):
                    a = a.detach().cpu().numpy()
                a = np.ascontiguousarray(a, dtype=np.float32)
                assert a.shape == (n,) + shp, (a.shape, shp)
                ptrs.append(a.ctypes.data)
            keep.append(a)
        d = SceneDesc(n, *ptrs, float(cycle), int(sh_degree), 1 if on_dev else 0)
        h = C.c_void_p()
        _check(self._L.pvg_create_scene(C.byref(d), C.byref(h)))
        self._h = h
        self.n = n

    @classmethod
    def from_workload_scene(cls, sc, **kw) -> "Scene":
        return cls(sc.mu, sc.quat, sc.scale, sc.opacity, sc.sh, sc.tau, sc.beta, sc.vel, sc.cycle, sc.sh_degree, **kw)

    def fork(self) -> "Scene":
        """A second handle on the same model with its own workspace (include/pvg.h pvg_fork_scene): render
        alternate frames through a scene and its fork, each under its own torch stream, to keep two frames in
        flight."""
        h = C.c_void_p()
        _check(self._L.pvg_fork_scene(self._h, C.byref(h)))
        other = object.__new__(Scene)
        other._L, other._h, other.n = self._L, h, self.n
        return other

    def render_many(self, frames: Sequence, outs: Optional[Sequence] = None, in_flight: int = 2) -> List[Tuple]:
        """Frames [(cam, t), ...] with `in_flight` of them overlapping (this scene and in_flight - 1 forks of it,
        round-robin, each under its own torch stream). Returns the per-frame (rgb, depth, alpha); the calling
        stream waits for all of them. Only stream and handle bookkeeping happens here."""
        import torch
        in_flight = max(1, min(int(in_flight), len(frames)))
        forks = getattr(self, "_forks", None) or []
        while len(forks) < in_flight - 1:
            forks.append(self.fork())
        self._forks = forks
        lanes = getattr(self, "_lanes", None) or []
        while len(lanes) < in_flight:
            lanes.append(torch.cuda.Stream())
        self._lanes = lanes
        handles = [self] + forks
        cur = torch.cuda.current_stream()
        for ln in lanes[:in_flight]:
            ln.wait_stream(cur)
        res = []
        for i, (cam, t) in enumerate(frames):
            with torch.cuda.stream(lanes[i % in_flight]):
                o = handles[i % in_flight].render(cam, t, None if outs is None else outs[i])
            for x in o:
                x.record_stream(cur)
            res.append(o)
        for ln in lanes[:in_flight]:
            cur.wait_stream(ln)
        return res

    # -- the path ---------------------------------------------------------------------------
    def render(self, cam, t: float, out: Optional[Tuple] = None, dt: float = 0.0, rho_min: float = 0.0,
               rho_max: float = float("inf"), target: str = "color"):
        """Frame at time t into torch CUDA tensors (rgb [3,H,W], depth [H,W], alpha [H,W]).
        dt != 0 renders the temporal-smoothing state H^(t) built from t - dt (Eq. 12); rho_min / rho_max
        keep only the points whose staticness beta / l lies in [rho_min, rho_max]. target="dynamics": the first
        tensor holds sum T a vbar (camera axes) and the second sum T a clamp(rho, 0, 2)."""
        import torch
        c = cam if isinstance(cam, CameraC) else camera_struct(cam)
        if out is None:
            out = (torch.empty((3, c.height, c.width), dtype=torch.float32, device="cuda"),
                   torch.empty((c.height, c.width), dtype=torch.float32, device="cuda"),
                   torch.empty((c.height, c.width), dtype=torch.float32, device="cuda"))
        _check(self._L.pvg_set_stream(self._h, torch.cuda.current_stream().cuda_stream))
        tg = {"color": 0, "dynamics": 1}[target]
        if dt == 0.0 and rho_min == 0.0 and rho_max == float("inf") and tg == 0:
            _check(self._L.pvg_render(self._h, C.byref(c), float(t), out[0].data_ptr(), out[1].data_ptr(),
                                      out[2].data_ptr()))
        else:
            st = StateC(float(t), float(dt), float(rho_min), float(rho_max), tg)
            _check(self._L.pvg_render_state(self._h, C.byref(c), C.byref(st), out[0].data_ptr(), out[1].data_ptr(),
                                            out[2].data_ptr()))
        return out

    def set_tile_rows(self, begin: int = 0, end: int = 0) -> None:
        """Restrict the following renders to the tile rows [begin, end) (end = 0: to the last row): only the
        pixel rows [16 begin, 16 end) of the output images are written (include/pvg.h PVG_OPT_TILE_ROW_BEGIN)."""
        self.set_option(OPT_TILE_ROW_BEGIN, int(begin))
        self.set_option(OPT_TILE_ROW_END, int(end))

    def render_host(self, cam, t: float, out: Optional[Tuple] = None):
        """Frame at time t into HOST buffers (torch CPU tensors, pinned if allocated here)."""
        import torch
        c = cam if isinstance(cam, CameraC) else camera_struct(cam)
        if out is None:
            out = (torch.empty((3, c.height, c.width), dtype=torch.float32, pin_memory=True),
                   torch.empty((c.height, c.width), dtype=torch.float32, pin_memory=True),
                   torch.empty((c.height, c.width), dtype=torch.float32, pin_memory=True))
        _check(self._L.pvg_set_stream(self._h, torch.cuda.current_stream().cuda_stream))
        _check(self._L.pvg_render_host(self._h, C.byref(c), float(t), out[0].data_ptr(), out[1].data_ptr(),
                                       out[2].data_ptr()))
        return out

    def set_sky(self, cube) -> None:
        """Sky cube map [6, R, R, 3] (numpy or torch CUDA tensor; copied), or None to switch it off:
        rgb = C + (1 - O) f_sky(d)."""
        import torch
        _check(self._L.pvg_set_stream(self._h, torch.cuda.current_stream().cuda_stream))
        if cube is None:
            _check(self._L.pvg_set_sky(self._h, None, 0, 0))
            return
        if _is_torch(cube) and cube.is_cuda:
            c = cube.detach().to(torch.float32).contiguous()
            assert c.dim() == 4 and c.shape[0] == 6 and c.shape[1] == c.shape[2] and c.shape[3] == 3
            _check(self._L.pvg_set_sky(self._h, c.data_ptr(), int(c.shape[1]), 1))
        else:
            c = np.ascontiguousarray(cube.detach().cpu().numpy() if _is_torch(cube) else cube, dtype=np.float32)
            assert c.ndim == 4 and c.shape[0] == 6 and c.shape[1] == c.shape[2] and c.shape[3] == 3
            _check(self._L.pvg_set_sky(self._h, c.ctypes.data, int(c.shape[1]), 0))

    def render_host_async(self, cam, t: float, out: Tuple):
        """Pipelined render into pinned HOST tensors; read them only after wait_host()."""
        import torch
        c = cam if isinstance(cam, CameraC) else camera_struct(cam)
        _check(self._L.pvg_set_stream(self._h, torch.cuda.current_stream().cuda_stream))
        _check(self._L.pvg_render_host_async(self._h, C.byref(c), float(t), out[0].data_ptr(), out[1].data_ptr(),
                                             out[2].data_ptr()))
        return out

    def wait_host(self) -> None:
        _check(self._L.pvg_wait_host(self._h))

    # -- options / hooks ----------------------------------------------------------------------
    def set_option(self, option: int, value: int) -> None:
        _check(self._L.pvg_set_option(self._h, int(option), int(value)))

    def stage_times_ms(self) -> Dict[str, float]:
        ms = (C.c_float * NUM_STAGES)()
        _check(self._L.pvg_stage_times_ms(self._h, ms))
        return {STAGES[i]: float(ms[i]) for i in range(NUM_STAGES)}

    def kernel_times_ms(self) -> List[Tuple[str, str, float]]:
        cap = 1 << 16
        names = (C.c_char_p * cap)()
        stages = (C.c_int * cap)()
        ms = (C.c_float * cap)()
        cnt = self._L.pvg_kernel_times_ms(self._h, cap, names, stages, ms)
        if cnt < 0:
            _check(cnt)
        return [(names[i].decode(), STAGES[stages[i]], float(ms[i])) for i in range(min(cnt, cap))]

    def kernel_timeline_ms(self) -> List[Tuple[str, float, float]]:
        """(kernel, start relative to the frame's first launch, duration) of the last render, in launch order."""
        cap = 4096
        names = (C.c_char_p * cap)()
        start = (C.c_float * cap)()
        dur = (C.c_float * cap)()
        cnt = self._L.pvg_kernel_timeline_ms(self._h, cap, names, start, dur)
        if cnt < 0:
            _check(cnt)
        return [(names[i].decode(), float(start[i]), float(dur[i])) for i in range(min(cnt, cap))]

    def frame_stats(self) -> Dict[str, int]:
        """Sizes of the last render (no device work)."""
        out = (C.c_uint64 * 10)()
        _check(self._L.pvg_frame_stats(self._h, out))
        return {"n": int(out[0]), "M": int(out[1]), "tiles_x": int(out[2]), "tiles_y": int(out[3]),
                "block_entries": int(out[4]), "list_mode": ("keys64", "compact", "blocks", "blocks_exact")[int(out[5])],
                "survivors": int(out[6]), "parked_tiles": int(out[7]), "M_exact": int(out[8]), "front": int(out[9])}

    def blend_counters(self) -> Tuple[int, int]:
        """(pairs evaluated, pairs contributing) of the last render with OPT_COUNT_PAIRS=1."""
        out = (C.c_uint64 * 2)()
        _check(self._L.pvg_blend_counters(self._h, out))
        return int(out[0]), int(out[1])

    def debug_info(self) -> DebugC:
        d = DebugC()
        _check(self._L.pvg_debug_view(self._h, C.byref(d)))
        return d

    def debug(self, fields: Optional[List[str]] = None) -> Dict[str, np.ndarray]:
        """Host copies (numpy) of the last render's intermediates."""
        d = self.debug_info()
        n, M, tiles = int(d.n), int(d.num_instances), int(d.tiles_x) * int(d.tiles_y)
        spec = {"record": (d.record, (n, 12), np.float32), "counts": (d.counts, (n,), np.uint32),
                "visit_order": (d.visit_order, (n,), np.uint32), "offsets": (d.offsets, (n,), np.uint32),
                "keys_unsorted": (d.keys_unsorted, (M,), np.uint64), "vals_unsorted": (d.vals_unsorted, (M,), np.uint32),
                "keys_sorted": (d.keys_sorted, (M,), np.uint64), "vals_sorted": (d.vals_sorted, (M,), np.uint32),
                "ranges": (d.ranges, (tiles, 2), np.uint32)}
        out: Dict[str, np.ndarray] = {"M": M, "tiles_x": int(d.tiles_x), "tiles_y": int(d.tiles_y),
                                      "sort_bits": (int(d.sort_begin_bit), int(d.sort_end_bit))}
        for k, (ptr, shape, dt) in spec.items():
            if fields is not None and k not in fields:
                continue
            if not ptr:
                out[k] = None if int(np.prod(shape)) else np.zeros(shape, dtype=dt)
                continue
            a = np.empty(shape, dtype=dt)
            _check(self._L.pvg_memcpy_d2h(a.ctypes.data, ptr, a.nbytes))
            out[k] = a
        return out

    def close(self) -> None:
        for f in getattr(self, "_forks", None) or []:
            f.close()
        self._forks = []
        if getattr(self, "_h", None):
            self._L.pvg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sort_pairs(keys, vals, begin_bit: int = 0, end_bit: int = 64):
    """Onesweep LSD radix sort of torch CUDA tensors (keys int64 holding uint64 bit patterns,
    vals int32 holding uint32). Returns new (keys, vals); inputs are clobbered."""
    import torch
    L = load_library()
    assert keys.is_cuda and vals.is_cuda and keys.dtype == torch.int64 and vals.dtype == torch.int32
    n = keys.numel()
    ko, vo = torch.empty_like(keys), torch.empty_like(vals)
    _check(L.pvg_sort_pairs(n, keys.data_ptr(), vals.data_ptr(), ko.data_ptr(), vo.data_ptr(), int(begin_bit),
                            int(end_bit), torch.cuda.current_stream().cuda_stream))
    return ko, vo


def sort_pairs_static_max_n() -> int:
    """Largest n pvg_sort_pairs_static accepts (PVG_SORT_STATIC_MAX_N of the built library)."""
    return int(load_library().pvg_sort_pairs_static_max_n())


def sort_pairs_static(keys, vals, keys_out, vals_out, begin_bit: int = 0, end_bit: int = 64) -> None:
    """pvg_sort_pairs_static (include/pvg.h): the same sort with its scratch in a static device array of the library
    -- no allocation anywhere in the call, which is why the caller passes the outputs too. At most
    sort_pairs_static_max_n() pairs (PvgError PVG_ERR_TOO_LARGE beyond). Asynchronous on torch's current stream; calls
    that overlap on the GPU race on the shared scratch. Inputs are clobbered."""
    import torch
    L = load_library()
    for x in (keys, vals, keys_out, vals_out):
        assert x.is_cuda and x.is_contiguous()
    assert keys.dtype == keys_out.dtype == torch.int64 and vals.dtype == vals_out.dtype == torch.int32
    n = keys.numel()
    assert vals.numel() == n and keys_out.numel() == n and vals_out.numel() == n
    _check(L.pvg_sort_pairs_static(n, keys.data_ptr(), vals.data_ptr(), keys_out.data_ptr(), vals_out.data_ptr(),
                                   int(begin_bit), int(end_bit), torch.cuda.current_stream().cuda_stream))


def calibrate_fp32(mode: int = 1):
    """(thread-level instructions per second, SM count) of the current CUDA device, measured by the library's
    register-only microbenchmark (include/pvg.h pvg_calibrate_fp32): mode 0 FFMA, 1 FFMA + LOP3, 2 packed FFMA2."""
    import torch
    L = load_library()
    rate, sms = C.c_double(0.0), C.c_int(0)
    _check(L.pvg_calibrate_fp32(int(mode), torch.cuda.current_stream().cuda_stream, C.byref(rate), C.byref(sms)))
    return float(rate.value), int(sms.value)


def guard_bands(enable: bool = True) -> None:
    """Test hook (include/pvg.h pvg_guard_bands): allocations made from now on carry guard bands."""
    _check(load_library().pvg_guard_bands(1 if enable else 0))


def check_guards():
    """(damaged, checked) live guarded allocations (include/pvg.h pvg_check_guards)."""
    bad, n = C.c_uint64(0), C.c_uint64(0)
    _check(load_library().pvg_check_guards(C.byref(bad), C.byref(n)))
    return int(bad.value), int(n.value)
