"""Seeded synthetic inputs shared by the oracle, the CUDA path, the tests and bench.py.

This package is a module of its own on purpose: it holds *none* of the client
method's arithmetic (no splats, Morton codes, BVH or sphere tests).  It produces
the 2.5D frames (premultiplied RGBA float32 + one depth float32 per pixel) of the
five BASELINE.json configs, standing in for the paper's server-side ray marcher
(sec. 4.1, sec. 4.2) on its unnamed data set, plus the
cameras of each config's scripted sequence.  Recipe: DESIGN.md "Input recipe".
"""
from __future__ import annotations

import ctypes
import hashlib
import math
import os
import subprocess
from dataclasses import dataclass, field
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gen.cpp"
_LIB = _HERE / "libsynthgen.so"
_lib = None

CENTER = np.array([0.5, 0.5, 0.5], dtype=np.float64)
DIAG = math.sqrt(3.0)
FOVY_DEG = 45.0
BASE_SEED = 14726


def build(force: bool = False) -> Path:
    """Compile gen.cpp into libsynthgen.so (g++, OpenMP)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["g++", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", str(_SRC), "-o", str(_LIB)]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        lib.synth_volume.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_uint64]
        lib.synth_volume.restype = None
        lib.synth_march.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                    ctypes.c_void_p, ctypes.c_void_p]
        lib.synth_march.restype = None
        _lib = lib
    return _lib


# ----------------------------------------------------------------------------- cameras
def look_at(eye, center=CENTER, world_up=(0.0, 1.0, 0.0), fovy_deg: float = FOVY_DEG) -> np.ndarray:
    """13 float32: eye, right, up, fwd (orthonormal), tan(fovy/2) -- the wr_camera POD."""
    eye = np.asarray(eye, dtype=np.float64)
    fwd = np.asarray(center, dtype=np.float64) - eye
    fwd /= np.linalg.norm(fwd)
    right = np.cross(fwd, np.asarray(world_up, dtype=np.float64))
    right /= np.linalg.norm(right)
    up = np.cross(right, fwd)
    cam = np.concatenate([eye, right, up, fwd, [math.tan(math.radians(fovy_deg) / 2.0)]])
    return cam.astype(np.float32)


def orbit_camera(az_deg: float = 0.0, el_deg: float = 0.0, dist: float = 2.0 * DIAG,
                 shift_right: float = 0.0) -> np.ndarray:
    """Camera on a sphere of radius `dist` about the volume centre, looking at it.
    Azimuth 0 = +z, rotation about the world-up (+y) axis through the centre."""
    az, el = math.radians(az_deg), math.radians(el_deg)
    eye = CENTER + dist * np.array([math.sin(az) * math.cos(el), math.sin(el), math.cos(az) * math.cos(el)])
    cam = look_at(eye)
    if shift_right != 0.0:
        cam64 = cam.astype(np.float64)
        cam64[0:3] += shift_right * cam64[3:6]
        cam = cam64.astype(np.float32)
    return cam


def _u01(seed: int, i: int) -> float:
    z = (seed + (i + 1) * 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & 0xFFFFFFFFFFFFFFFF
    z ^= z >> 31
    return (z >> 11) / 9007199254740992.0


# ----------------------------------------------------------------------------- configs
@dataclass
class Config:
    index: int
    vol_n: int
    n_gauss: int
    noise_amp: float
    W: int
    H: int
    r_scale: float
    src_cams: list = field(default_factory=list)        # one per BVH build
    dst_cams: list = field(default_factory=list)        # one per render
    dst_src: list = field(default_factory=list)         # which build each render uses
    rebuild_before: list = field(default_factory=list)  # render indices preceded by a rebuild

    @property
    def seed(self) -> int:
        return BASE_SEED + self.index

    @property
    def name(self) -> str:
        return f"config{self.index}_{self.W}x{self.H}_vol{self.vol_n}"


def make_config(index: int, *, W: int | None = None, H: int | None = None, vol_n: int | None = None,
                n_frames: int | None = None) -> Config:
    """The five BASELINE.json configs.  W/H/vol_n/n_frames overrides give reduced
    variants of the same recipe for quick tests (the defaults are the full sizes)."""
    d0 = 2.0 * DIAG
    if index == 0:
        c = Config(0, vol_n or 32, 8, 0.0, W or 64, H or 64, 1.0)
        c.src_cams = [orbit_camera(0.0)]
        c.dst_cams = [orbit_camera(5.0)]
        c.dst_src = [0]
    elif index == 1:
        c = Config(1, vol_n or 128, 32, 0.0, W or 512, H or 512, 1.0)
        c.src_cams = [orbit_camera(0.0)]
        c.dst_cams = [orbit_camera(a) for a in (2.0, 10.0, 20.0)]
        c.dst_src = [0, 0, 0]
    elif index == 2:
        c = Config(2, vol_n or 256, 64, 0.05, W or 1024, H or 1024, 1.0)
        nf = n_frames or 60
        amp = 2.0 + 5.0 * _u01(c.seed + 1000, 0)
        phase = 2.0 * math.pi * _u01(c.seed + 1000, 1)
        c.src_cams = [orbit_camera(0.0)]
        c.dst_cams = [orbit_camera(0.5 * (f + 1), amp * math.sin(2.0 * math.pi * f / 60.0 + phase)) for f in range(nf)]
        c.dst_src = [0] * nf
    elif index == 3:
        c = Config(3, vol_n or 256, 64, 0.05, W or 1920, H or 1080, 1.0)
        nf = n_frames or 60
        cams = [orbit_camera(0.0, 0.0, d0 * (1.0 - 0.5 * f / 59.0)) for f in range(nf)]
        c.dst_cams = cams
        c.src_cams = [cams[f] for f in range(0, nf, 4)]
        c.dst_src = [f // 4 for f in range(nf)]
    elif index == 4:
        c = Config(4, vol_n or 512, 128, 0.0, W or 3840, H or 2160, 2.0)
        c.src_cams = [orbit_camera(0.0)]
        c.dst_cams = [orbit_camera(15.0), orbit_camera(15.0, shift_right=0.25 * DIAG)]
        c.dst_src = [0, 0]
    else:
        raise ValueError(f"no such config: {index}")
    seen = set()
    for i, s in enumerate(c.dst_src):
        if s not in seen:
            seen.add(s)
            c.rebuild_before.append(i)
    return c


TABLE1_DIST = 1.4688   # camera distance at which config 2's volume fills 59.5 % of a 1024 x 1024 frame


def table1_config(n_views: int = 3) -> Config:
    """A frame shaped like the one behind the paper's Table 1: 1024 x 1024 viewport,
    623,584 of 1,048,576 samples valid (59.5 %).  The paper's data set is not available, so this
    is config 2's volume (256^3, 64 Gaussians + noise) with the camera moved in until the fill
    matches (distance found by bisection on the generator's own output: 1.4688 gives 0.5949); three
    display views rotated 2, 10 and 20 degrees at the same distance stand in for "View 1..3"."""
    c = Config(2, 256, 64, 0.05, 1024, 1024, 1.0)
    c.src_cams = [orbit_camera(0.0, 0.0, TABLE1_DIST)]
    c.dst_cams = [orbit_camera(a, 0.0, TABLE1_DIST) for a in (2.0, 10.0, 20.0)][:n_views]
    c.dst_src = [0] * len(c.dst_cams)
    c.rebuild_before = [0]
    return c


# ----------------------------------------------------------------------------- generation
_vol_cache: dict = {}


def _cache_dir() -> Path | None:
    d = os.environ.get("SYNTH_CACHE", "/tmp/synth_cache_2006_14726")
    if d in ("", "0", "off"):
        return None
    p = Path(d)
    try:
        p.mkdir(parents=True, exist_ok=True)
    except OSError:
        return None
    return p


def _src_hash() -> str:
    return hashlib.sha1(_SRC.read_bytes()).hexdigest()[:12]


def volume(cfg: Config) -> np.ndarray:
    key = (cfg.vol_n, cfg.n_gauss, cfg.noise_amp, cfg.seed)
    if key not in _vol_cache:
        lib = _load()
        vol = np.empty((cfg.vol_n,) * 3, dtype=np.float32)
        lib.synth_volume(vol.ctypes.data, cfg.vol_n, cfg.n_gauss, float(cfg.noise_amp), cfg.seed)
        _vol_cache.clear()  # keep at most one volume (512^3 = 512 MB)
        _vol_cache[key] = vol
    return _vol_cache[key]


def source_frame(cfg: Config, build_index: int = 0):
    """(color float32 [H,W,4] premultiplied, depth float32 [H,W]) for build `build_index`."""
    cam = np.ascontiguousarray(cfg.src_cams[build_index], dtype=np.float32)
    cd = _cache_dir()
    path = None
    if cd is not None:
        h = hashlib.sha1(cam.tobytes()).hexdigest()[:12]
        path = cd / f"{_src_hash()}_{cfg.vol_n}_{cfg.n_gauss}_{cfg.noise_amp}_{cfg.seed}_{cfg.W}x{cfg.H}_{h}.npz"
        if path.exists():
            try:
                z = np.load(path)
                return z["color"], z["depth"]
            except Exception:
                pass
    lib = _load()
    vol = volume(cfg)
    color = np.empty((cfg.H, cfg.W, 4), dtype=np.float32)
    depth = np.empty((cfg.H, cfg.W), dtype=np.float32)
    lib.synth_march(vol.ctypes.data, cfg.vol_n, cam.ctypes.data, cfg.W, cfg.H, color.ctypes.data, depth.ctypes.data)
    if path is not None:
        try:
            tmp = path.with_suffix(f".tmp{os.getpid()}.npz")
            np.savez(tmp, color=color, depth=depth)
            os.replace(tmp, path)
        except OSError:
            pass
    return color, depth


def random_frame(W: int, H: int, seed: int, fill: float = 0.6, cam: np.ndarray | None = None):
    """A structure-free stress frame: valid pixels chosen at random with probability
    `fill` (the paper's Table 1 fill is 0.595), depth uniform in
    [2.6, 4.3], random premultiplied colours with alpha in [0.05, 1].  Used by the
    edge-case tests (ragged tails, low-alpha stacks); not one of the five configs."""
    rng = np.random.default_rng(seed)
    depth = rng.uniform(2.6, 4.3, size=(H, W)).astype(np.float32)
    depth[rng.random((H, W)) >= fill] = 0.0
    a = rng.uniform(0.05, 1.0, size=(H, W, 1))
    rgb = rng.uniform(0.0, 1.0, size=(H, W, 3)) * a
    color = np.concatenate([rgb, a], axis=2).astype(np.float32)
    return color, depth, (orbit_camera(0.0) if cam is None else cam)


def dense_frame(W: int, H: int, seed: int, cam: np.ndarray | None = None):
    """A fully covered frame of a smooth undulating surface (every pixel valid, alpha in
    [0.5, 1]): the N = P upper bound of the build, where the build kernels
    are bandwidth bound.  Not one of the five configs."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:H, 0:W].astype(np.float32)
    depth = (3.4 + 0.35 * np.sin(x / W * 9.0) * np.cos(y / H * 7.0)
             + 0.05 * np.sin(x * 0.05) * np.sin(y * 0.043)).astype(np.float32)
    a = rng.uniform(0.5, 1.0, size=(H, W, 1))
    rgb = rng.uniform(0.0, 1.0, size=(H, W, 3)) * a
    color = np.concatenate([rgb, a], axis=2).astype(np.float32)
    return color, depth, (orbit_camera(0.0) if cam is None else cam)
