"""Radius variants: the paper's constant radius and an
opacity-weighted footprint (a reading of PAPER.md:109).  Oracle pins (not gpu) + GPU parity."""
import math

import numpy as np
import pytest

import oracle
import synth


def _frame():
    color, depth, cam = synth.random_frame(40, 24, seed=9, fill=0.7)
    return color, depth, cam, 40, 24


def test_constant_radius_is_half_a_voxel_diagonal_for_every_sample():
    # "we currently just set the footprint radius to half the size of a voxel's
    # diagonal"; unit cube sampled by 32^3 voxels: sqrt(3)/64
    color, depth, cam, W, H = _frame()
    half_diag = math.sqrt(3.0) / 32 / 2
    s0, v0, n0 = oracle.unproject(depth, cam, W, H, 1.0)
    s1, v1, n1 = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_CONSTANT, half_diag)
    assert n0 == n1 and np.array_equal(v0, v1)
    assert np.array_equal(s0[:, :3], s1[:, :3])                      # Eq. 1 is untouched
    assert np.all(s1[v1 == 1, 3] == np.float32(half_diag)) and np.all(s1[v1 == 0, 3] == 0)
    s2, _, _ = oracle.unproject(depth, cam, W, H, 2.0, oracle.RADIUS_CONSTANT, half_diag)
    assert np.all(s2[v1 == 1, 3] == np.float32(2.0) * np.float32(half_diag))
    # unlike the footprint radius it does not grow with depth (PAPER.md:55 is about the image, not r)
    assert len(np.unique(s0[v0 == 1, 3])) > 10


def test_constant_radius_single_sphere_entry_point():
    # closed form: sphere of radius r centred on the central ray at distance t0 is entered at t0 - r
    cam = synth.orbit_camera(0.0)
    depth = np.zeros((3, 3), np.float32); depth[1, 1] = 2.0
    color = np.full((3, 3, 4), 0.5, np.float32)
    sc = oracle.build_scene(color, depth, cam, 3, 3, 1.0, oracle.RADIUS_CONSTANT, 1.0)
    assert sc["sphere_sorted"][0, 3] == 1.0
    hit, t = oracle.ray_sphere(cam[:3], cam[9:12], sc["sphere_sorted"][0])
    assert hit and t == pytest.approx(1.0, abs=1e-6)
    # a radius this large covers the whole 3x3 image; the footprint radius covers one pixel
    assert (oracle.render(sc, cam, 3, 3, "brute")[..., 3] > 0).all()
    assert (oracle.render(oracle.build_scene(color, depth, cam, 3, 3, 1.0), cam, 3, 3, "brute")[..., 3] > 0).sum() == 1


def test_opacity_radius_limits_and_monotonicity():
    color, depth, cam, W, H = _frame()
    s0, v, _ = oracle.unproject(depth, cam, W, H, 1.0)
    ok = v == 1
    opaque = color.copy(); opaque[..., 3] = 1.0
    clear = color.copy(); clear[..., 3] = 0.0
    for f in (0.5, 0.25):   # 1 - f exact
        s1, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, f, opaque)
        assert np.array_equal(s1, s0)                                  # alpha = 1 keeps the footprint
        s2, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, f, clear)
        assert np.array_equal(s2[ok, 3], s0[ok, 3] * np.float32(f))    # alpha = 0: the floor
    s3, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, 1.0, color)
    assert np.array_equal(s3, s0)                                      # floor 1: no dependence on alpha
    s4, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, 0.0, color)
    a = color.reshape(-1, 4)[:, 3]
    np.testing.assert_allclose(s4[ok, 3], s0[ok, 3] * a[ok], rtol=3e-7)
    lo, hi = color.copy(), color.copy()
    lo[..., 3] = 0.3; hi[..., 3] = 0.6
    rl, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, 0.2, lo)
    rh, _, _ = oracle.unproject(depth, cam, W, H, 1.0, oracle.RADIUS_OPACITY, 0.2, hi)
    assert np.all(rh[ok, 3] > rl[ok, 3])


@pytest.mark.gpu
@pytest.mark.parametrize("radius", [(1, 0.004), (1, 0.02), (2, 0.25), (2, 0.0)])
def test_gpu_radius_variants_parity(radius):
    from gpu_common import Session, check_scene
    from paper_2006_14726_b200 import binding as sp
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    with Session(128, 128) as s:
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, [cfg.dst_cams[0]], mode="brute", radius=radius)
        c2, d2, cam2 = synth.random_frame(111, 77, seed=4, fill=0.5)
        check_scene(s, c2, d2, cam2, 111, 77, 1.5, [synth.orbit_camera(8.0)], mode="bvh", radius=radius)
        # atomic refit path gathers the spheres in another kernel: same radii
        sp.splats_set_option(sp.OPT_REFIT, sp.REFIT_ATOMIC)
        check_scene(s, c2, d2, cam2, 111, 77, 1.5, [synth.orbit_camera(8.0)], mode="bvh", radius=radius)
        with pytest.raises(sp.SplatsError):
            sp.splats_set_radius(1, 0.0)
        with pytest.raises(sp.SplatsError):
            sp.splats_set_radius(2, 1.5)
        with pytest.raises(sp.SplatsError):
            sp.splats_set_radius(7, 1.0)
        # back to the default: the footprint radius again
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, [cfg.dst_cams[0]], mode="brute")


@pytest.mark.gpu
def test_gpu_constant_radius_config1_half_voxel_diagonal():
    from gpu_common import Session, check_scene
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    half_diag = math.sqrt(3.0) / cfg.vol_n / 2      # PAPER.md:69 for this config's 128^3 volume
    with Session(cfg.W, cfg.H) as s:
        sc, stats = check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, cfg.dst_cams[:2], mode="bvh",
                                radius=(1, half_diag))
        assert np.all(sc["sphere_sorted"][:, 3] == np.float32(half_diag))
