"""CPU oracle for the client hot path of arxiv 2006.14726 -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  The product (paper_2006_14726_b200) never does, and
this package never imports the product.  The arithmetic lives in splat_oracle.cpp
(single-threaded C++, float32 with the op order of DESIGN.md sec. 3); this file
compiles it and marshals numpy arrays.  One step is stated here in numpy instead:
quantise_child_boxes (O7b), the 16-bit storage format of the node boxes -- a reading
of this repository (S13), not something the paper defines.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "splat_oracle.cpp"
_LIB = _HERE / "libsplatoracle.so"
_lib = None

_vp = ctypes.c_void_p
_i32 = ctypes.c_int
_i64 = ctypes.c_int64


def _cpu_has_fma() -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return " fma " in (line + " ")
    except OSError:
        pass
    return False


def build(force: bool = False) -> Path:
    """g++ -O2 -ffp-contract=off: the only fused multiply-adds are explicit fmaf().
    -mfma (when the host has it) merely inlines fmaf(); the result is the same
    correctly rounded value libm's fmaf() returns."""
    if os.environ.get("ORACLE_SANITIZE"):
        return _build_sanitized()
    stamp = _HERE / ".built_with_fma"
    want_fma = _cpu_has_fma()
    stale = (not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime
             or (stamp.exists() and not want_fma))
    if force or stale:
        cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC"]
        if want_fma:
            cmd.append("-mfma")
        cmd += [str(_SRC), "-o", str(_LIB)]
        subprocess.run(cmd, check=True)
        if want_fma:
            stamp.write_text("1")
        elif stamp.exists():
            stamp.unlink()
    return _LIB


def _build_sanitized() -> Path:
    """ORACLE_SANITIZE=1: the same source with -fsanitize=address,undefined, in its own
    file.  Run the pins with
        ORACLE_SANITIZE=1 LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" \
        ASAN_OPTIONS=detect_leaks=0 UBSAN_OPTIONS=halt_on_error=1 python -m pytest tests -q -m "not gpu"
    (the preload is needed because the interpreter itself is not instrumented)."""
    global _LIB
    out = _HERE / "libsplatoracle_san.so"
    if not out.exists() or out.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
               "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", str(_SRC), "-o", str(out)]
        subprocess.run(cmd, check=True)
    _LIB = out
    return out


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(str(_LIB))
        L.oracle_pixel_ray.argtypes = [_vp, _i32, _i32, _i32, _i32, _vp, _vp]
        L.oracle_unproject.argtypes = [_vp, _vp, _i32, _i32, ctypes.c_float, _i32, ctypes.c_float, _vp, _vp, _vp]
        L.oracle_unproject.restype = _i64
        L.oracle_pack.argtypes = [_vp, _vp, _vp, _i32, _i32, ctypes.c_float, _i32, ctypes.c_float, _vp, _vp, _vp]
        L.oracle_pack.restype = _i64
        L.oracle_decode.argtypes = [_vp, _vp, _i64, _vp, _vp, _vp, _vp]
        L.oracle_bounds.argtypes = [_vp, _vp, _i64, _vp, _vp]
        L.oracle_morton_point.argtypes = [_vp, _vp, _vp]
        L.oracle_morton_point.restype = ctypes.c_uint64
        L.oracle_compact_codes.argtypes = [_vp, _vp, _i64, _vp, _vp, _vp, _vp]
        L.oracle_compact_codes.restype = _i64
        L.oracle_sort.argtypes = [_vp, _i64, _vp]
        L.oracle_tree.argtypes = [_vp, _i64, _vp, _vp, _vp]
        L.oracle_refit.argtypes = [_vp, _vp, _i64, _vp]
        L.oracle_ray_sphere.argtypes = [_vp, _vp, _vp, _vp]
        L.oracle_ray_sphere.restype = _i32
        L.oracle_composite.argtypes = [_i32, _vp, _vp, _vp, _vp]
        L.oracle_composite.restype = _i32
        L.oracle_render_brute.argtypes = [_vp, _vp, _vp, _i64, _vp, _i32, _i32, _vp, _i64, _i32, _vp, _vp]
        L.oracle_render_bvh.argtypes = [_vp, _vp, _vp, _i64, _vp, _vp, _vp, _i32, _i32, _vp, _i64, _i32, _vp, _vp]
        L.oracle_quantise_image.argtypes = [_vp, _i64, _vp]
        L.oracle_march.argtypes = [_vp, _i32, _vp, _vp, _vp, _i32, _i32, _vp, _vp]
        L.oracle_render_points.argtypes = [_vp, _vp, _vp, _i64, _vp, _i32, _i32, _i32, _vp]
        _lib = L
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a):
    return a.ctypes.data if a is not None else None


# ------------------------------------------------------------------ single steps
def pixel_ray(cam, W, H, x, y):
    cam = _f32(cam)
    d = np.empty(3, np.float32)
    ln = np.empty(1, np.float32)
    lib().oracle_pixel_ray(_ptr(cam), W, H, x, y, _ptr(d), _ptr(ln))
    return d, float(ln[0])


RADIUS_FOOTPRINT, RADIUS_CONSTANT, RADIUS_OPACITY = 0, 1, 2


def unproject(depth, cam, W, H, r_scale, radius_mode=RADIUS_FOOTPRINT, radius_param=0.0, color=None):
    depth, cam = _f32(depth).reshape(-1), _f32(cam)
    assert depth.size == W * H
    sphere = np.empty((W * H, 4), np.float32)
    valid = np.empty(W * H, np.uint8)
    col = _f32(color).reshape(W * H, 4) if radius_mode == RADIUS_OPACITY else None
    n = lib().oracle_unproject(_ptr(depth), _ptr(cam), W, H, float(r_scale), int(radius_mode), float(radius_param),
                               _ptr(col), _ptr(sphere), _ptr(valid))
    return sphere, valid, int(n)


def pack(color, depth, cam, W, H, r_scale, quant, radius_mode=RADIUS_FOOTPRINT, radius_param=0.0):
    """Server side of the wire format: (samples uint64[n], colours uint32[n]).
    quant = (lo xyz, hi xyz, r_max)."""
    color, depth, cam, quant = _f32(color).reshape(W * H, 4), _f32(depth).reshape(-1), _f32(cam), _f32(quant)
    assert quant.size == 7
    samples = np.empty(W * H, np.uint64)
    colours = np.empty(W * H, np.uint32)
    n = lib().oracle_pack(_ptr(color), _ptr(depth), _ptr(cam), W, H, float(r_scale), int(radius_mode), float(radius_param),
                          _ptr(quant), _ptr(samples), _ptr(colours))
    return samples[:n].copy(), colours[:n].copy()


def decode(samples, colours, quant):
    """Client side: (sphere float32[n,4], rgba float32[n,4], valid uint8[n])."""
    samples = np.ascontiguousarray(samples, dtype=np.uint64)
    colours = np.ascontiguousarray(colours, dtype=np.uint32)
    quant = _f32(quant)
    n = samples.size
    sphere = np.empty((n, 4), np.float32)
    rgba = np.empty((n, 4), np.float32)
    valid = np.empty(n, np.uint8)
    lib().oracle_decode(_ptr(samples), _ptr(colours), n, _ptr(quant), _ptr(sphere), _ptr(rgba), _ptr(valid))
    return sphere, rgba, valid


def bounds(sphere, valid):
    lo, hi = np.empty(3, np.float32), np.empty(3, np.float32)
    lib().oracle_bounds(_ptr(sphere), _ptr(valid), sphere.shape[0], _ptr(lo), _ptr(hi))
    return lo, hi


def morton_point(c, lo, hi) -> int:
    c, lo, hi = _f32(c), _f32(lo), _f32(hi)
    return int(lib().oracle_morton_point(_ptr(c), _ptr(lo), _ptr(hi)))


def compact_codes(sphere, valid, lo, hi, n):
    ids = np.empty(n, np.uint32)
    codes = np.empty(n, np.uint64)
    lo, hi = _f32(lo), _f32(hi)
    m = lib().oracle_compact_codes(_ptr(sphere), _ptr(valid), sphere.shape[0], _ptr(lo), _ptr(hi), _ptr(ids), _ptr(codes))
    assert m == n
    return ids, codes


def sort_codes(codes):
    codes = np.ascontiguousarray(codes, dtype=np.uint64)
    order = np.empty(codes.size, np.uint32)
    lib().oracle_sort(_ptr(codes), codes.size, _ptr(order))
    return order


def tree(sorted_codes):
    sorted_codes = np.ascontiguousarray(sorted_codes, dtype=np.uint64)
    n = sorted_codes.size
    children = np.full((max(n - 1, 0), 2), -1, np.int32)
    parents = np.full(max(2 * n - 1, 0), -2, np.int32)
    ranges = np.full((max(n - 1, 0), 2), -1, np.int32)
    lib().oracle_tree(_ptr(sorted_codes), n, _ptr(children), _ptr(parents), _ptr(ranges))
    return children, parents, ranges


def refit(sphere_sorted, children):
    sphere_sorted = _f32(sphere_sorted)
    n = sphere_sorted.shape[0]
    aabbs = np.zeros((max(2 * n - 1, 0), 6), np.float32)
    lib().oracle_refit(_ptr(sphere_sorted), _ptr(children), n, _ptr(aabbs))
    return aabbs


def ray_sphere(o, d, sphere4):
    o, d, s = _f32(o), _f32(d), _f32(sphere4)
    t = np.zeros(1, np.float32)
    hit = lib().oracle_ray_sphere(_ptr(o), _ptr(d), _ptr(s), _ptr(t))
    return bool(hit), float(t[0])


def composite(t, ids, rgba):
    t, rgba = _f32(t), _f32(rgba)
    ids = np.ascontiguousarray(ids, dtype=np.uint32)
    out = np.zeros(4, np.float32)
    used = lib().oracle_composite(t.size, _ptr(t), _ptr(ids), _ptr(rgba), _ptr(out))
    return out, int(used)


# ------------------------------------------------------------------ whole path
def build_scene(color, depth, cam, W, H, r_scale, radius_mode=RADIUS_FOOTPRINT, radius_param=0.0):
    """O1..O7 on one 2.5D frame.  Returns a dict of numpy arrays (see keys below)."""
    color = _f32(color).reshape(W * H, 4)
    sphere, valid, n = unproject(depth, cam, W, H, r_scale, radius_mode, radius_param, color)
    lo, hi = bounds(sphere, valid)
    ids, codes = compact_codes(sphere, valid, lo, hi, n)
    order = sort_codes(codes)
    sorted_ids = ids[order]
    sorted_codes = codes[order]
    sphere_sorted = np.ascontiguousarray(sphere[sorted_ids])
    rgba_sorted = np.ascontiguousarray(color[sorted_ids])
    children, parents, ranges = tree(sorted_codes)
    aabbs = refit(sphere_sorted, children)
    return dict(N=n, W=W, H=H, sphere=sphere, valid=valid, lo=lo, hi=hi, ids=ids, codes=codes, order=order,
                sorted_ids=sorted_ids, sorted_codes=sorted_codes, sphere_sorted=sphere_sorted,
                rgba_sorted=rgba_sorted, children=children, parents=parents, ranges=ranges, aabbs=aabbs)


def build_scene_packed(samples, colours, quant):
    """O4..O7 on a received buffer of packed samples (ids = position in the buffer)."""
    sphere, rgba, valid = decode(samples, colours, quant)
    n = int(valid.sum())
    lo, hi = bounds(sphere, valid)
    ids, codes = compact_codes(sphere, valid, lo, hi, n)
    order = sort_codes(codes)
    sorted_ids = ids[order]
    sorted_codes = codes[order]
    sphere_sorted = np.ascontiguousarray(sphere[sorted_ids])
    rgba_sorted = np.ascontiguousarray(rgba[sorted_ids])
    children, parents, ranges = tree(sorted_codes)
    aabbs = refit(sphere_sorted, children)
    return dict(N=n, sphere=sphere, valid=valid, lo=lo, hi=hi, ids=ids, codes=codes, order=order,
                sorted_ids=sorted_ids, sorted_codes=sorted_codes, sphere_sorted=sphere_sorted,
                rgba_sorted=rgba_sorted, children=children, parents=parents, ranges=ranges, aabbs=aabbs)


def quantise_child_boxes(scene):
    """O7b (S13; the paper says nothing about how node boxes are stored): the traversal
    records that follow from the exact tree of O6 / O7.  Frame: rmax = largest splat radius,
    qlo_a = lo_a - rmax, ext_a = (hi_a + rmax) - qlo_a (lo / hi: bounds of the centres, O3),
    s_a = 65535 / ext_a (0 for a zero extent).  A lower plane x of a child box becomes
    clamp(floor((x - qlo_a) * s_a), 0, 65535), an upper plane clamp(ceil(...), 0, 65535); every
    operation rounded to float32 on its own.  Returns (records, frame):
      records  (N-1, 8) uint32 per internal node: words 0..2 = axis x, y, z of the left child box,
               q_lo | q_hi << 16; words 3..5 the right child's; words 6, 7 = left / right link
               (internal node index, or 0x80000000 | sorted position of a leaf)
      frame    7 float32: lo xyz, hi xyz, rmax"""
    n = scene["N"]
    f32 = np.float32
    if n < 2:
        return np.zeros((0, 8), np.uint32), None
    rmax = f32(scene["sphere_sorted"][:, 3].max())
    lo, hi = scene["lo"].astype(f32), scene["hi"].astype(f32)
    qlo = (lo - rmax).astype(f32)
    ext = ((hi + rmax).astype(f32) - qlo).astype(f32)
    with np.errstate(divide="ignore"):
        s = np.where(ext > 0, (f32(65535.0) / ext).astype(f32), f32(0.0)).astype(f32)
    boxes = scene["aabbs"][scene["children"]].astype(f32)               # (n-1, 2, 6): lo xyz, hi xyz of each child
    ul = np.floor(((boxes[:, :, 0:3] - qlo).astype(f32) * s).astype(f32))
    uh = np.ceil(((boxes[:, :, 3:6] - qlo).astype(f32) * s).astype(f32))
    ql = np.clip(ul, 0, 65535).astype(np.uint32)
    qh = np.clip(uh, 0, 65535).astype(np.uint32)
    rec = np.zeros((n - 1, 8), dtype=np.uint32)
    rec[:, 0:6] = (ql | (qh << np.uint32(16))).reshape(n - 1, 6)
    ch = scene["children"].astype(np.int64)
    rec[:, 6:8] = np.where(ch >= n - 1, 0x80000000 | (ch - (n - 1)), ch).astype(np.uint32)
    return rec, np.concatenate([lo, hi, [rmax]]).astype(f32)


def render(scene, cam, W2, H2, mode="bvh", pixels=None, return_hits=False, first_hit=False):
    """O8..O9.  mode 'brute' = L0 (definition), 'bvh' = L1 (walk of the oracle's tree).
    pixels: optional int64 array of destination pixel indices (y*W2+x).
    first_hit: the paper's first-hit query instead of compositing every hit."""
    cam = _f32(cam)
    n = scene["N"]
    if pixels is not None:
        pixels = np.ascontiguousarray(pixels, dtype=np.int64)
        total = pixels.size
    else:
        total = W2 * H2
    out = np.zeros((total, 4), np.float32)
    used = np.zeros(total, np.int32)
    sp, co, ids = scene["sphere_sorted"], scene["rgba_sorted"], scene["sorted_ids"]
    if mode == "brute":
        lib().oracle_render_brute(_ptr(sp), _ptr(co), _ptr(ids), n, _ptr(cam), W2, H2, _ptr(pixels), total,
                                  1 if first_hit else 0, _ptr(out), _ptr(used))
    elif mode == "bvh":
        lib().oracle_render_bvh(_ptr(sp), _ptr(co), _ptr(ids), n, _ptr(scene["children"]), _ptr(scene["aabbs"]),
                                _ptr(cam), W2, H2, _ptr(pixels), total, 1 if first_hit else 0, _ptr(out), _ptr(used))
    else:
        raise ValueError(mode)
    if pixels is None:
        out = out.reshape(H2, W2, 4)
        used = used.reshape(H2, W2)
    return (out, used) if return_hits else out


def render_points(scene, cam, W2, H2, point_px=1):
    """The [ZAL12] point-primitive warp the paper compares against: splat
    centres as fixed-size points with a per-point depth test.  Returns float32 [H2, W2, 4]."""
    cam = _f32(cam)
    out = np.zeros((H2, W2, 4), np.float32)
    lib().oracle_render_points(_ptr(scene["sphere_sorted"]), _ptr(scene["rgba_sorted"]), _ptr(scene["sorted_ids"]),
                               scene["N"], _ptr(cam), W2, H2, int(point_px), _ptr(out))
    return out


def make_transfer(tents, half_width=0.05, shade=0.45, depth_alpha=0.5, stop_alpha=0.999):
    """wr_transfer as (int32[1], float32[24]): tents = [(iso, alpha_max, (r, g, b)), ...] (<= 4)."""
    assert 1 <= len(tents) <= 4
    f = np.zeros(24, np.float32)
    for i, (iso, a, rgb) in enumerate(tents):
        f[i], f[4 + i] = iso, a
        f[8 + 3 * i: 11 + 3 * i] = rgb
    f[20:24] = (half_width, shade, depth_alpha, stop_alpha)
    return np.array([len(tents)], np.int32), f


# BASELINE.json configs[0]: "opacity peaks 0.8 at iso 0.35 and 0.95 at iso 0.7"; colours as in synth/
BASELINE_TENTS = [(0.35, 0.8, (0.95, 0.55, 0.15)), (0.70, 0.95, (0.25, 0.60, 0.95))]


def march(volume, cam, W, H, transfer=None):
    """Server-side ray marcher: (color float32 [H,W,4] premultiplied, depth float32 [H,W])."""
    vol = _f32(volume)
    n = vol.shape[0]
    assert vol.shape == (n, n, n)
    tn, tf = transfer if transfer is not None else make_transfer(BASELINE_TENTS)
    cam = _f32(cam)
    color = np.empty((H, W, 4), np.float32)
    depth = np.empty((H, W), np.float32)
    lib().oracle_march(_ptr(vol), n, _ptr(tn), _ptr(tf), _ptr(cam), W, H, _ptr(color), _ptr(depth))
    return color, depth


def quantise_image(rgba):
    """RGBA8 words (uint32, R | G<<8 | B<<16 | A<<24) of a float image, rounding as the wire's colours."""
    a = _f32(rgba)
    out = np.empty(a.shape[:-1], np.uint32)
    lib().oracle_quantise_image(_ptr(a), out.size, _ptr(out))
    return out
