"""-m gpu: splats_render_points (the paper's comparison renderer) against
the oracle's point renderer.  Which pixels a point covers and which point wins are float32
decisions taken with the shared arithmetic of DESIGN.md sec. 3, so the images must be equal."""
import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_common import Session
from paper_2006_14726_b200 import binding as sp

pytestmark = pytest.mark.gpu


def _points(cam, W2, H2, size):
    out = torch.full((H2, W2, 4), -7.0, dtype=torch.float32, device="cuda")
    sp.splats_render_points(cam, W2, H2, size, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _same(got, ref, what):
    bad = int((got.reshape(-1, 4) != ref.reshape(-1, 4)).any(axis=1).sum())
    assert bad == 0, f"{what}: {bad} pixels differ"


def test_config0_points_all_sizes_and_views():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    with Session(128, 128) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
        for cam in (cfg.src_cams[0], cfg.dst_cams[0], synth.orbit_camera(40.0, -10.0, synth.DIAG)):
            for size, (W2, H2) in ((1, (64, 64)), (2, (64, 64)), (3, (100, 50)), (8, (128, 128))):
                _same(_points(cam, W2, H2, size), oracle.render_points(sc, cam, W2, H2, size), f"size {size}")
        # identity camera, one-pixel points: the source image itself
        got = _points(cfg.src_cams[0], cfg.W, cfg.H, 1)
        v = depth > 0
        assert np.array_equal(got[v], color[v]) and np.all(got[~v] == 0)
        # consecutive calls with different image sizes: the depth buffer is re-armed every time
        _same(_points(cfg.dst_cams[0], 37, 91, 2), oracle.render_points(sc, cfg.dst_cams[0], 37, 91, 2), "resized")
        with pytest.raises(sp.SplatsError):
            sp.splats_render_points(cfg.dst_cams[0], 64, 64, 0, torch.empty((64, 64, 4), device="cuda"))


@pytest.mark.parametrize("W,H,fill,size", [(97, 61, 0.7, 1), (130, 50, 1.0, 4), (640, 360, 1.0, 2)])
def test_points_overdraw_depth_test(W, H, fill, size):
    # many points per pixel (random depths, camera far away and eye inside the cloud): the depth
    # test decides, including points behind the eye plane that must be culled
    color, depth, cam = synth.random_frame(W, H, seed=H, fill=fill)
    sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
    inside = synth.orbit_camera(10.0, 5.0, 0.2)       # near the volume centre: half the points are behind
    with Session(W, H) as s:
        s.update(color, depth, cam, W, H, 1.0)
        for dst, (W2, H2) in ((synth.orbit_camera(0.0, 0.0, 12.0), (48, 27)), (inside, (W, H)), (synth.orbit_camera(25.0), (W, H))):
            _same(_points(dst, W2, H2, size), oracle.render_points(sc, dst, W2, H2, size), "overdraw")


def test_points_empty_scene_and_packed_input():
    cam = synth.orbit_camera(0.0)
    with Session(64, 64) as s:
        s.update(np.ones((8, 8, 4), np.float32), np.zeros((8, 8), np.float32), cam, 8, 8, 1.0)
        assert np.all(_points(cam, 20, 10, 3) == 0)
        cfg = synth.make_config(0)
        color, depth = synth.source_frame(cfg, 0)
        quant = [0, 0, 0, 1, 1, 1, 0.1]
        rs, rc = oracle.pack(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, quant)
        sc = oracle.build_scene_packed(rs, rc, quant)
        ws = torch.from_numpy(rs.view(np.int64).copy()).cuda()
        cs = torch.from_numpy(rc.view(np.int32).copy()).cuda()
        sp.splats_update_packed(ws, cs, len(rs), quant)
        _same(_points(cfg.dst_cams[0], 64, 64, 2), oracle.render_points(sc, cfg.dst_cams[0], 64, 64, 2), "packed")


def test_config3_points_full_size_and_the_papers_comparison():
    cfg = synth.make_config(3)
    b = 7
    color, depth = synth.source_frame(cfg, b)
    sc = oracle.build_scene(color, depth, cfg.src_cams[b], cfg.W, cfg.H, 1.0)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[b], cfg.W, cfg.H, 1.0)
        near = cfg.dst_cams[59]                         # the end of the dolly: the camera has moved in
        for size in (1, 2):
            _same(_points(near, cfg.W, cfg.H, size), oracle.render_points(sc, near, cfg.W, cfg.H, size), f"1080p size {size}")
        # PAPER.md:55 / Fig. 3: fixed-size points leave holes where the ray-traced spheres do not
        pts = (_points(near, cfg.W, cfg.H, 1)[..., 3] > 0).sum()
        sph = (s.render(near, cfg.W, cfg.H)[..., 3] > 0).sum()
        assert sph > 1.3 * pts
