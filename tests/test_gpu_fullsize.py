"""-m gpu: parity at BASELINE.json's full sizes (configs 2, 3, 4), in the launch configuration
bench.py times.  The BVH is compared in full (bit-exact); images are compared in full where the
oracle's BVH walk finishes in seconds, else on seeded random pixel samples, and always
spot-checked against the brute-force definition on a smaller sample."""
import numpy as np
import pytest

import oracle
import synth
from gpu_common import Session, assert_bvh_bit_exact, assert_rgba_close

pytestmark = pytest.mark.gpu


def _check_renders(s, sc, cams, W, H, full, n_bvh, n_brute, seed):
    for i, cam in enumerate(cams):
        got = s.render(cam, W, H)
        rng = np.random.default_rng(seed + i)
        if full:
            ref = oracle.render(sc, cam, W, H, "bvh")
            assert_rgba_close(got, ref, f"camera {i} full frame")
            assert (ref[..., 3] > 0).mean() > 0.01
        else:
            px = rng.choice(W * H, size=n_bvh, replace=False).astype(np.int64)
            assert_rgba_close(got.reshape(-1, 4)[px], oracle.render(sc, cam, W, H, "bvh", pixels=px), f"camera {i} sampled")
        # brute-force spot check, biased towards covered pixels
        covered = np.nonzero(got.reshape(-1, 4)[:, 3] > 0)[0]
        px = np.concatenate([rng.choice(covered, size=min(n_brute, covered.size), replace=False),
                             rng.choice(W * H, size=n_brute // 4, replace=False)]).astype(np.int64)
        assert_rgba_close(got.reshape(-1, 4)[px], oracle.render(sc, cam, W, H, "brute", pixels=px), f"camera {i} brute")


def test_config2_full_size():
    cfg = synth.make_config(2)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        assert_bvh_bit_exact(sc)
        _check_renders(s, sc, [cfg.dst_cams[i] for i in (0, 29, 59)], cfg.W, cfg.H, True, 0, 256, 20)


@pytest.mark.parametrize("build", [0, 7, 14])
def test_config3_full_size(build):
    cfg = synth.make_config(3)
    color, depth = synth.source_frame(cfg, build)
    sc = oracle.build_scene(color, depth, cfg.src_cams[build], cfg.W, cfg.H, cfg.r_scale)
    cams = [cfg.dst_cams[4 * build + j] for j in (0, 3)]
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[build], cfg.W, cfg.H, cfg.r_scale)
        assert_bvh_bit_exact(sc)
        _check_renders(s, sc, cams, cfg.W, cfg.H, True, 0, 256, 30 + build)
        # frame 4*build is rendered from its own source camera: identity reprojection
        got = s.render(cfg.dst_cams[4 * build], cfg.W, cfg.H)
        v = depth > 0
        assert np.array_equal(got[v], color[v]) and np.all(got[~v] == 0)


def test_config4_full_size():
    cfg = synth.make_config(4)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        assert_bvh_bit_exact(sc)
        _check_renders(s, sc, cfg.dst_cams, cfg.W, cfg.H, False, 200_000, 192, 40)


def test_config3_bench_step_in_bench_launch_configuration():
    # exactly what bench.py times: SPLATS_OPT_OVERLAP on, one update and its four renders into four
    # images enqueued back to back, no synchronisation in between; all four frames in full
    import torch
    from paper_2006_14726_b200 import binding as sp
    cfg = synth.make_config(3)
    build = 14
    color, depth = synth.source_frame(cfg, build)
    sc = oracle.build_scene(color, depth, cfg.src_cams[build], cfg.W, cfg.H, cfg.r_scale)
    with Session(cfg.W, cfg.H, exact_nodes=False):   # the library's defaults, as bench.py runs it
        sp.splats_set_option(sp.OPT_OVERLAP, 1)
        dc, dd = torch.from_numpy(color).cuda(), torch.from_numpy(depth).cuda()
        outs = [torch.full((cfg.H, cfg.W, 4), -7.0, dtype=torch.float32, device="cuda") for _ in range(4)]
        for rep in range(2):                      # the second step overwrites the images of the first
            sp.splats_update(dc, dd, cfg.src_cams[build], cfg.W, cfg.H, cfg.r_scale)
            for j in range(4):
                sp.splats_render(cfg.dst_cams[4 * build + j], cfg.W, cfg.H, outs[j])
        torch.cuda.synchronize()
        assert_bvh_bit_exact(sc, exact=False)
        for j in range(4):
            ref = oracle.render(sc, cfg.dst_cams[4 * build + j], cfg.W, cfg.H, "bvh")
            assert_rgba_close(outs[j].cpu().numpy(), ref, f"display frame {4 * build + j}")


def test_dense_1080p_leg_of_the_bench():
    # bench.py's `dense` leg: synth.dense_frame 1920x1080 (N = P), the library's defaults, its two cameras
    W, H = 1920, 1080
    color, depth, cam = synth.dense_frame(W, H, 0)
    sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
    assert sc["N"] == W * H
    with Session(W, H, exact_nodes=False) as s:
        s.update(color, depth, cam, W, H, 1.0)
        assert_bvh_bit_exact(sc, exact=False)
        _check_renders(s, sc, [synth.orbit_camera(0.0), synth.orbit_camera(3.0)], W, H, False, 100_000, 128, 50)


def test_table1_shape_leg_of_the_bench():
    # bench.py's `table1_shape` leg: 1024x1024, 59.5 % of the samples valid, all-hit and
    # first-hit queries of its three views
    cfg = synth.table1_config()
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    assert abs(sc["N"] / (cfg.W * cfg.H) - 0.595) < 0.005
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        assert_bvh_bit_exact(sc)
        _check_renders(s, sc, cfg.dst_cams, cfg.W, cfg.H, False, 100_000, 128, 60)
        rng = np.random.default_rng(61)
        for cam in cfg.dst_cams:
            px = rng.choice(cfg.W * cfg.H, size=50_000, replace=False).astype(np.int64)
            got = s.render(cam, cfg.W, cfg.H, first_hit=True).reshape(-1, 4)[px]
            assert np.array_equal(got, oracle.render(sc, cam, cfg.W, cfg.H, "bvh", pixels=px, first_hit=True))


def test_beyond_2_23_splats_four_global_sort_passes():
    # more than 2^23 splats: the windowed sort runs four global passes (an even number: the other input buffer)
    W, H = 4096, 2304
    color, depth, cam = synth.dense_frame(W, H, 0)
    sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
    assert sc["N"] == W * H > (1 << 23)
    with Session(W, H, exact_nodes=False) as s:
        s.update(color, depth, cam, W, H, 1.0)
        assert_bvh_bit_exact(sc, exact=False)
        _check_renders(s, sc, [synth.orbit_camera(2.0)], W, H, False, 20_000, 64, 70)
