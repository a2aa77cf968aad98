"""Thin Python binding of the C ABI in include/splats.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libsplats.so; this file converts
torch tensors / numpy cameras into raw pointers and turns error codes into exceptions.
PyTorch is used for device memory and streams, nothing else.  There is no CPU fallback:
if the shared library is missing and cannot be built, importing the symbols raises.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

import numpy as np
import torch

from . import build as _build

NUM_STAGES = 9
STAGE_NAMES = ("bounds", "unproject_morton_compact", "sort", "tree_1", "tree_2", "render", "pack", "points", "march")
OPT_REFIT, REFIT_PYRAMID, REFIT_ATOMIC, REFIT_TILED = 0, 0, 1, 2
OPT_SORT, SORT_HYBRID, SORT_LSD8, SORT_LSD8_LAUNCHES, SORT_HYBRID_LSD = 1, 0, 1, 2, 3
RADIUS_FOOTPRINT, RADIUS_CONSTANT, RADIUS_OPACITY = 0, 1, 2
OPT_PDL = 2
OPT_OVERLAP = 3
OPT_EXACT_NODES = 4


class SplatsError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"splats error {code}: {msg}")
        self.code = code


class wr_quant(ctypes.Structure):
    _fields_ = [("lo", ctypes.c_float * 3), ("hi", ctypes.c_float * 3), ("r_max", ctypes.c_float)]


class wr_transfer(ctypes.Structure):
    _fields_ = [("n_tents", ctypes.c_int), ("iso", ctypes.c_float * 4), ("alpha", ctypes.c_float * 4),
                ("rgb", (ctypes.c_float * 3) * 4), ("half_width", ctypes.c_float), ("shade", ctypes.c_float),
                ("depth_alpha", ctypes.c_float), ("stop_alpha", ctypes.c_float)]


class wr_camera(ctypes.Structure):
    _fields_ = [("eye", ctypes.c_float * 3), ("right", ctypes.c_float * 3), ("up", ctypes.c_float * 3),
                ("fwd", ctypes.c_float * 3), ("tan_half_fovy", ctypes.c_float)]


_lib = None
_vp = ctypes.c_void_p
_ci = ctypes.c_int


def lib() -> ctypes.CDLL:
    """Load libsplats.so (building it with nvcc if it is stale or missing)."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not Path(path).exists():
            raise RuntimeError(f"{path} is missing: the CUDA extension is required (no CPU fallback)")
        L = ctypes.CDLL(str(path))
        cam_p = ctypes.POINTER(wr_camera)
        L.splats_create.argtypes = [_vp, _ci, _ci]
        L.splats_update.argtypes = [_vp, _vp, cam_p, _ci, _ci, ctypes.c_float]
        L.splats_update_begin.argtypes = [_vp, _vp, cam_p, _ci, _ci, ctypes.c_float]
        L.splats_render.argtypes = [cam_p, _ci, _ci, _vp]
        L.splats_render_first_hit.argtypes = [cam_p, _ci, _ci, _vp]
        L.splats_render_rgba8.argtypes = [cam_p, _ci, _ci, _vp]
        L.splats_render_host_rgba8.argtypes = [cam_p, _ci, _ci, _vp]
        L.splats_render_points.argtypes = [cam_p, _ci, _ci, _ci, _vp]
        L.splats_march.argtypes = [_vp, _ci, ctypes.POINTER(wr_transfer), cam_p, _ci, _ci, _vp, _vp]
        L.splats_pack.argtypes = [_vp, _vp, cam_p, _ci, _ci, ctypes.c_float, ctypes.POINTER(wr_quant), _vp, _vp, _vp]
        L.splats_update_packed.argtypes = [_vp, _vp, ctypes.c_uint, ctypes.POINTER(wr_quant)]
        L.splats_pack_noalloc.argtypes = [_vp, _vp, cam_p, _ci, _ci, ctypes.c_float, _ci, ctypes.c_float, ctypes.POINTER(wr_quant),
                                          _vp, _vp, _vp, _vp]
        L.splats_update_packed_host.argtypes = [_vp, _vp, ctypes.c_uint, ctypes.POINTER(wr_quant)]
        L.splats_update_host.argtypes = [_vp, _vp, cam_p, _ci, _ci, ctypes.c_float]
        L.splats_render_host.argtypes = [cam_p, _ci, _ci, _vp]
        L.splats_count.argtypes = [ctypes.POINTER(ctypes.c_uint)]
        L.splats_export.argtypes = [_vp, _vp, _vp, _vp, _vp]
        L.splats_export_splats.argtypes = [_vp, _vp, _vp]
        L.splats_export_child_boxes.argtypes = [_vp]
        L.splats_export_qnodes.argtypes = [_vp, _vp]
        L.splats_set_profiling.argtypes = [_ci]
        L.splats_set_option.argtypes = [_ci, _ci]
        L.splats_set_radius.argtypes = [_ci, ctypes.c_float]
        L.splats_stage_ms.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_uint)]
        L.splats_launch_count.restype = ctypes.c_ulonglong
        L.splats_traced_pixels.argtypes = [ctypes.POINTER(ctypes.c_ulonglong), _ci]
        L.splats_last_error.restype = ctypes.c_char_p
        L.splats_destroy.restype = None
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise SplatsError(rc, lib().splats_last_error().decode())


def _cam(cam) -> wr_camera:
    a = np.ascontiguousarray(np.asarray(cam, dtype=np.float32).reshape(13))
    c = wr_camera()
    ctypes.memmove(ctypes.byref(c), a.ctypes.data, 13 * 4)
    return c


def _dev_ptr(t: torch.Tensor, dtype, numel: int | None = None) -> int:
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise TypeError(f"expected a contiguous CUDA tensor of dtype {dtype}")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"tensor too small: {t.numel()} < {numel}")
    return t.data_ptr()


def _host_ptr(t, numel: int) -> int:
    if isinstance(t, torch.Tensor):
        if t.is_cuda or not t.is_contiguous() or t.dtype != torch.float32 or t.numel() < numel:
            raise TypeError("expected a contiguous float32 host tensor of sufficient size")
        return t.data_ptr()
    a = t
    if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and a.size >= numel):
        raise TypeError("expected a contiguous float32 numpy array of sufficient size")
    return a.ctypes.data


# ----------------------------------------------------------------------------- the C calls
def splats_create(max_W: int, max_H: int, stream: torch.cuda.Stream | None = None) -> None:
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: this library has no CPU fallback")
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib().splats_create(_vp(s.cuda_stream), int(max_W), int(max_H)))


def splats_update(color: torch.Tensor, depth: torch.Tensor, src_camera, W: int, H: int, r_scale: float) -> None:
    c = _cam(src_camera)
    _check(lib().splats_update(_dev_ptr(color, torch.float32, W * H * 4), _dev_ptr(depth, torch.float32, W * H),
                               ctypes.byref(c), int(W), int(H), float(r_scale)))


def splats_update_begin(color: torch.Tensor, depth: torch.Tensor, src_camera, W: int, H: int, r_scale: float) -> None:
    c = _cam(src_camera)
    _check(lib().splats_update_begin(_dev_ptr(color, torch.float32, W * H * 4), _dev_ptr(depth, torch.float32, W * H),
                                     ctypes.byref(c), int(W), int(H), float(r_scale)))


def splats_update_commit() -> None:
    _check(lib().splats_update_commit())


def splats_render(dst_camera, W2: int, H2: int, out_rgba: torch.Tensor) -> None:
    c = _cam(dst_camera)
    _check(lib().splats_render(ctypes.byref(c), int(W2), int(H2), _dev_ptr(out_rgba, torch.float32, W2 * H2 * 4)))


def splats_render_first_hit(dst_camera, W2: int, H2: int, out_rgba: torch.Tensor) -> None:
    c = _cam(dst_camera)
    _check(lib().splats_render_first_hit(ctypes.byref(c), int(W2), int(H2), _dev_ptr(out_rgba, torch.float32, W2 * H2 * 4)))


def splats_render_points(dst_camera, W2: int, H2: int, point_px: int, out_rgba: torch.Tensor) -> None:
    c = _cam(dst_camera)
    _check(lib().splats_render_points(ctypes.byref(c), int(W2), int(H2), int(point_px),
                                      _dev_ptr(out_rgba, torch.float32, W2 * H2 * 4)))


def make_transfer(tents, half_width=0.05, shade=0.45, depth_alpha=0.5, stop_alpha=0.999) -> wr_transfer:
    """tents = [(iso, alpha_max, (r, g, b)), ...] (at most 4)."""
    t = wr_transfer()
    t.n_tents = len(tents)
    for i, (iso, a, rgb) in enumerate(tents):
        t.iso[i], t.alpha[i] = iso, a
        for k in range(3):
            t.rgb[i][k] = rgb[k]
    t.half_width, t.shade, t.depth_alpha, t.stop_alpha = half_width, shade, depth_alpha, stop_alpha
    return t


def splats_march(volume: torch.Tensor, n: int, tf: wr_transfer, camera, W: int, H: int, color: torch.Tensor,
                 depth: torch.Tensor) -> None:
    c = _cam(camera)
    _check(lib().splats_march(_dev_ptr(volume, torch.float32, n * n * n), int(n), ctypes.byref(tf), ctypes.byref(c),
                              int(W), int(H), _dev_ptr(color, torch.float32, W * H * 4), _dev_ptr(depth, torch.float32, W * H)))


def _quant(q) -> wr_quant:
    a = np.ascontiguousarray(np.asarray(q, dtype=np.float32).reshape(7))
    out = wr_quant()
    ctypes.memmove(ctypes.byref(out), a.ctypes.data, 7 * 4)
    return out


def splats_pack(color: torch.Tensor, depth: torch.Tensor, src_camera, W: int, H: int, r_scale: float, quant,
                samples: torch.Tensor, colors: torch.Tensor, count: torch.Tensor) -> None:
    """samples: int64 CUDA tensor (uint64 words) of >= W*H, colors: int32 of >= W*H, count: int32 of 1."""
    c, q = _cam(src_camera), _quant(quant)
    _check(lib().splats_pack(_dev_ptr(color, torch.float32, W * H * 4), _dev_ptr(depth, torch.float32, W * H),
                             ctypes.byref(c), int(W), int(H), float(r_scale), ctypes.byref(q),
                             _dev_ptr(samples, torch.int64, W * H), _dev_ptr(colors, torch.int32, W * H),
                             _dev_ptr(count, torch.int32, 1)))


NOALLOC_MAX_PIXELS = 4096 * 4096


def splats_noalloc_setup() -> None:
    """Look up the static scratch array's address on the current device ahead of the first splats_pack_noalloc."""
    _check(lib().splats_noalloc_setup())


def splats_pack_noalloc(color: torch.Tensor, depth: torch.Tensor, src_camera, W: int, H: int, r_scale: float, quant,
                        samples: torch.Tensor, colors: torch.Tensor, count: torch.Tensor,
                        radius_mode: int = 0, radius_param: float = 0.0, stream=None) -> None:
    """splats_pack without a context and without any allocation (include/splats.h): W*H <= NOALLOC_MAX_PIXELS.
    stream: a torch.cuda.Stream (default: torch's current stream)."""
    c, q = _cam(src_camera), _quant(quant)
    if int(W) * int(H) > NOALLOC_MAX_PIXELS:   # let the library say so: no buffer of that size is needed for the check
        ptrs = [t.data_ptr() for t in (color, depth, samples, colors, count)]
    else:
        ptrs = [_dev_ptr(color, torch.float32, W * H * 4), _dev_ptr(depth, torch.float32, W * H),
                _dev_ptr(samples, torch.int64, W * H), _dev_ptr(colors, torch.int32, W * H), _dev_ptr(count, torch.int32, 1)]
    st = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
    _check(lib().splats_pack_noalloc(ptrs[0], ptrs[1], ctypes.byref(c), int(W), int(H), float(r_scale), int(radius_mode),
                                     float(radius_param), ctypes.byref(q), ptrs[2], ptrs[3], ptrs[4], ctypes.c_void_p(st)))


def splats_update_packed(samples: torch.Tensor, colors: torch.Tensor, n: int, quant) -> None:
    q = _quant(quant)
    _check(lib().splats_update_packed(_dev_ptr(samples, torch.int64, n) if n else None,
                                      _dev_ptr(colors, torch.int32, n) if n else None, int(n), ctypes.byref(q)))


def splats_update_packed_host(samples: torch.Tensor, colors: torch.Tensor, n: int, quant) -> None:
    """samples: int64 host tensor (uint64 words), colors: int32 host tensor; pinned for asynchronous copies."""
    for t, dt in ((samples, torch.int64), (colors, torch.int32)):
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous() and t.dtype == dt and t.numel() >= n):
            raise TypeError(f"expected a contiguous host tensor of dtype {dt} with >= {n} elements")
    q = _quant(quant)
    _check(lib().splats_update_packed_host(samples.data_ptr() if n else None, colors.data_ptr() if n else None, int(n),
                                           ctypes.byref(q)))


def splats_update_host(color, depth, src_camera, W: int, H: int, r_scale: float) -> None:
    c = _cam(src_camera)
    _check(lib().splats_update_host(_host_ptr(color, W * H * 4), _host_ptr(depth, W * H), ctypes.byref(c),
                                    int(W), int(H), float(r_scale)))


def splats_render_host(dst_camera, W2: int, H2: int, out_rgba) -> None:
    c = _cam(dst_camera)
    _check(lib().splats_render_host(ctypes.byref(c), int(W2), int(H2), _host_ptr(out_rgba, W2 * H2 * 4)))


def splats_render_rgba8(dst_camera, W2: int, H2: int, out_rgba8: torch.Tensor) -> None:
    """out_rgba8: int32 CUDA tensor of >= W2*H2 (uint32 words R | G<<8 | B<<16 | A<<24)."""
    c = _cam(dst_camera)
    _check(lib().splats_render_rgba8(ctypes.byref(c), int(W2), int(H2), _dev_ptr(out_rgba8, torch.int32, W2 * H2)))


def splats_render_host_rgba8(dst_camera, W2: int, H2: int, out_rgba8) -> None:
    """out_rgba8: contiguous int32 host tensor (pinned for asynchronous copies) of >= W2*H2."""
    if not (isinstance(out_rgba8, torch.Tensor) and not out_rgba8.is_cuda and out_rgba8.is_contiguous()
            and out_rgba8.dtype == torch.int32 and out_rgba8.numel() >= W2 * H2):
        raise TypeError("expected a contiguous int32 host tensor of sufficient size")
    c = _cam(dst_camera)
    _check(lib().splats_render_host_rgba8(ctypes.byref(c), int(W2), int(H2), out_rgba8.data_ptr()))


def splats_count() -> int:
    n = ctypes.c_uint(0)
    _check(lib().splats_count(ctypes.byref(n)))
    return int(n.value)


def splats_export(aabbs: bool = True):
    """dict of CUDA tensors: keys (int64 view of uint64), perm, children, parents, node_aabbs
    (the exact boxes: they need OPT_EXACT_NODES during the build; aabbs=False skips them)."""
    n = splats_count()
    dev = torch.device("cuda", torch.cuda.current_device())
    keys = torch.empty(n, dtype=torch.int64, device=dev)
    perm = torch.empty(n, dtype=torch.int32, device=dev)
    children = torch.empty((max(n - 1, 0), 2), dtype=torch.int32, device=dev)
    parents = torch.empty(max(2 * n - 1, 0), dtype=torch.int32, device=dev)
    boxes = torch.empty((max(2 * n - 1, 0), 6), dtype=torch.float32, device=dev) if aabbs else None
    if n:
        _check(lib().splats_export(keys.data_ptr(), perm.data_ptr(), children.data_ptr() if n > 1 else None,
                                   parents.data_ptr(), boxes.data_ptr() if aabbs else None))
    return dict(N=n, keys=keys, perm=perm, children=children, parents=parents, node_aabbs=boxes)


def splats_export_qnodes():
    """(N-1, 8) int32 CUDA tensor (uint32 bit patterns): the 32-byte records the traversal reads;
    and frame = 7 float32: bounds of the centres lo xyz, hi xyz and the largest radius."""
    n = splats_count()
    dev = torch.device("cuda", torch.cuda.current_device())
    q = torch.empty((max(n - 1, 0), 8), dtype=torch.int32, device=dev)
    frame = torch.empty(7, dtype=torch.float32, device=dev)
    _check(lib().splats_export_qnodes(q.data_ptr() if n > 1 else None, frame.data_ptr()))
    return dict(N=n, qnodes=q, frame=frame)


def splats_export_child_boxes():
    """(N-1, 12) float32 CUDA tensor: the two child boxes stored in every internal node's record."""
    n = splats_count()
    dev = torch.device("cuda", torch.cuda.current_device())
    boxes = torch.empty((max(n - 1, 0), 12), dtype=torch.float32, device=dev)
    if n > 1:
        _check(lib().splats_export_child_boxes(boxes.data_ptr()))
    return boxes


def splats_export_splats():
    n = splats_count()
    dev = torch.device("cuda", torch.cuda.current_device())
    sphere = torch.empty((n, 4), dtype=torch.float32, device=dev)
    rgba = torch.empty((n, 4), dtype=torch.float32, device=dev)
    lo_hi = torch.empty(6, dtype=torch.float32, device=dev)
    _check(lib().splats_export_splats(sphere.data_ptr() if n else None, rgba.data_ptr() if n else None,
                                      lo_hi.data_ptr()))
    return dict(N=n, sphere=sphere, rgba=rgba, lo_hi=lo_hi)


def splats_set_option(option: int, value: int) -> None:
    _check(lib().splats_set_option(int(option), int(value)))


def splats_set_radius(mode: int, param: float = 0.0) -> None:
    _check(lib().splats_set_radius(int(mode), float(param)))


def splats_set_profiling(on: bool) -> None:
    _check(lib().splats_set_profiling(1 if on else 0))


def splats_stage_ms() -> dict:
    """{stage name: (sum of durations in ms, number of runs)} since the last query."""
    ms = (ctypes.c_float * NUM_STAGES)()
    calls = (ctypes.c_uint * NUM_STAGES)()
    _check(lib().splats_stage_ms(ms, calls))
    return {name: (float(ms[i]), int(calls[i])) for i, name in enumerate(STAGE_NAMES)}


def splats_launch_count() -> int:
    return int(lib().splats_launch_count())


def splats_traced_pixels(reset: bool = False) -> int:
    """Destination pixels for which the renders set up a ray since the last reset (synchronises)."""
    v = ctypes.c_ulonglong(0)
    _check(lib().splats_traced_pixels(ctypes.byref(v), 1 if reset else 0))
    return int(v.value)


def splats_synchronize() -> None:
    _check(lib().splats_synchronize())


def splats_last_error() -> str:
    return lib().splats_last_error().decode()


def splats_destroy() -> None:
    lib().splats_destroy()
