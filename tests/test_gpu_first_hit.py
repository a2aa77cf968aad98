"""-m gpu: the paper's first-hit query (splats_render_first_hit; SURVEY.md
sec. 8(f) row 1) against the oracle's first-hit renderer.  The winner of a pixel is decided by
float32 arithmetic shared bit for bit (S8), so the images are compared for
equality, not within a tolerance."""
import numpy as np
import pytest

import oracle
import synth
from gpu_common import Session

pytestmark = pytest.mark.gpu


def _same(got, ref, what):
    bad = int((got.reshape(-1, 4) != ref.reshape(-1, 4)).any(axis=1).sum())
    assert bad == 0, f"{what}: {bad} pixels differ"


def test_config0_first_hit_brute_force():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        for cam in (cfg.dst_cams[0], synth.orbit_camera(-30.0, 12.0, 2.4)):
            got = s.render(cam, cfg.W, cfg.H, first_hit=True)
            ref = oracle.render(sc, cam, cfg.W, cfg.H, "brute", first_hit=True)
            _same(got, ref, "config 0")
            assert (ref[..., 3] > 0).mean() > 0.02
        # the all-hit image of the same view is a different picture where splats overlap
        allhit = s.render(cfg.dst_cams[0], cfg.W, cfg.H)
        assert (allhit != s.render(cfg.dst_cams[0], cfg.W, cfg.H, first_hit=True)).any()


@pytest.mark.parametrize("W,H,fill,r_scale", [(97, 61, 0.7, 1.0), (130, 50, 0.3, 2.5), (33, 200, 1.0, 4.0)])
def test_first_hit_random_frames_heavy_overlap(W, H, fill, r_scale):
    color, depth, cam = synth.random_frame(W, H, seed=W, fill=fill)
    sc = oracle.build_scene(color, depth, cam, W, H, r_scale)
    with Session(W, H) as s:
        s.update(color, depth, cam, W, H, r_scale)
        for dst, (W2, H2) in ((synth.orbit_camera(6.0), (W, H)), (synth.orbit_camera(-15.0, 5.0), (80, 45))):
            got = s.render(dst, W2, H2, first_hit=True)
            _same(got, oracle.render(sc, dst, W2, H2, "brute", first_hit=True), f"{W}x{H}")


def test_first_hit_coaxial_stack_and_equal_t():
    # 40 splats along the central ray, alpha 0.05: compositing needs them all, first hit takes #0;
    # the whole source column maps to one ray, and the ids decide between equal depths.
    W, H = 1, 40
    cam = synth.orbit_camera(0.0)
    depth = np.full((H, W), 3.0, np.float32)
    color = np.tile(np.array([0.01, 0.02, 0.03, 0.05], np.float32), (H, W, 1))
    color[:, 0, 0] = np.linspace(0.0, 0.04, H)
    sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
    with Session(16, 16) as s:
        s.update(color, depth, cam, W, H, 1.0)
        for dst in (cam, synth.orbit_camera(1.0)):
            _same(s.render(dst, 16, 16, first_hit=True), oracle.render(sc, dst, 16, 16, "brute", first_hit=True), "stack")


def test_first_hit_empty_and_single():
    cam = synth.orbit_camera(0.0)
    depth = np.zeros((8, 8), np.float32)
    color = np.ones((8, 8, 4), np.float32)
    with Session(8, 8) as s:
        s.update(color, depth, cam, 8, 8, 1.0)
        assert np.all(s.render(cam, 8, 8, first_hit=True) == 0)
        depth[3, 4] = 2.5
        color[3, 4] = (0.1, 0.2, 0.3, 0.4)
        s.update(color, depth, cam, 8, 8, 1.0)
        out = s.render(cam, 8, 8, first_hit=True)
        assert np.array_equal(out[3, 4], color[3, 4]) and out[..., 3].sum() == np.float32(0.4)


def test_config1_first_hit_full_frames():
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        for cam in cfg.dst_cams:
            _same(s.render(cam, cfg.W, cfg.H, first_hit=True),
                  oracle.render(sc, cam, cfg.W, cfg.H, "bvh", first_hit=True), "config 1")


def test_config2_first_hit_full_size():
    # the configuration closest to the paper's Table 1 (1024 x 1024, first hit)
    cfg = synth.make_config(2)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        for i in (0, 59):
            got = s.render(cfg.dst_cams[i], cfg.W, cfg.H, first_hit=True)
            _same(got, oracle.render(sc, cfg.dst_cams[i], cfg.W, cfg.H, "bvh", first_hit=True), f"config 2 frame {i}")
            rng = np.random.default_rng(i)
            px = rng.choice(np.nonzero(got.reshape(-1, 4)[:, 3] > 0)[0], size=256, replace=False).astype(np.int64)
            _same(got.reshape(-1, 4)[px], oracle.render(sc, cfg.dst_cams[i], cfg.W, cfg.H, "brute", pixels=px, first_hit=True), "brute")
