"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element.

Bar (BASELINE.json north_star): Morton codes, sorted permutation, tree topology and AABBs
bit-exact; composited RGBA within 1e-3 per channel with at most 0.01 % of pixels beyond."""
import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_common import Session, assert_bvh_bit_exact, assert_rgba_close, check_scene
from paper_2006_14726_b200 import binding as sp

pytestmark = pytest.mark.gpu


def test_config0_full_brute_force():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        sc, stats = check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale,
                                cfg.dst_cams + cfg.src_cams, mode="brute")
        # identity camera: bit-exact reproduction of the source image (closed form (iii))
        got = s.render(cfg.src_cams[0], cfg.W, cfg.H)
        v = depth > 0
        assert np.array_equal(got[v], color[v]) and np.all(got[~v] == 0)


@pytest.mark.parametrize("W,H,fill,r_scale", [
    (33, 31, 0.9, 1.0), (48, 27, 0.6, 2.0), (127, 65, 0.3, 3.0), (256, 100, 0.6, 1.0), (7, 5, 1.0, 0.5),
])
def test_random_frames_ragged_sizes(W, H, fill, r_scale):
    color, depth, cam = synth.random_frame(W, H, seed=W * 1000 + H, fill=fill)
    dst = [synth.orbit_camera(5.0), synth.orbit_camera(-20.0, 10.0, 2.5), synth.orbit_camera(15.0, shift_right=0.4), cam]
    sizes = [(W, H), (40, 30), (W + 3, H + 1), (W, H)]
    with Session(max(W + 3, 40), max(H + 1, 30)) as s:
        check_scene(s, color, depth, cam, W, H, r_scale, dst, sizes, mode="brute" if W * H < 6000 else "bvh")


def test_low_alpha_stack_forces_relaunch():
    # alpha 0.05 everywhere, r_scale 4: every ray needs far more than the K = 4 entries of the k-buffer
    # (render.cuh KBUF), i.e. many re-launches from the cursor
    W, H = 40, 30
    color, depth, cam = synth.random_frame(W, H, seed=5, fill=1.0)
    color[..., 3] = 0.05
    color[..., :3] *= 0.05
    depth[...] = np.linspace(3.0, 3.4, W * H, dtype=np.float32).reshape(H, W)
    with Session(W, H) as s:
        sc, _ = check_scene(s, color, depth, cam, W, H, 4.0, [cam, synth.orbit_camera(3.0)], mode="brute")
        _, used = oracle.render(sc, cam, W, H, "brute", return_hits=True)
        assert used.max() > 16  # the oracle itself needed more than two k-buffers' worth


def test_coaxial_stack_closed_form_90_hits():
    # closed form (ii) on a frame whose splats all project onto the one destination pixel; parity with the oracle,
    # and the closed form whenever the oracle itself composited the full stack
    W, H = 12, 12
    color, depth, cam = synth.random_frame(W, H, seed=9, fill=1.0)
    color[...] = np.array([0.01, 0.02, 0.03, 0.05], np.float32)
    depth[...] = 3.0
    with Session(W, H) as s:
        s.update(color, depth, cam, W, H, 1.0)
        far = synth.orbit_camera(0.0, 0.0, 400.0)   # all 144 splats fall inside one far pixel's ray
        got = s.render(far, 1, 1)
        sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
        ref, used = oracle.render(sc, far, 1, 1, "brute", return_hits=True)
        assert_rgba_close(got, ref)
        if used[0, 0] >= 90:
            assert got[0, 0, 3] == pytest.approx(1 - 0.95 ** 90, abs=1e-5)


def test_coaxial_packed_stack_closed_form_unconditional():
    # closed form (ii), by construction: 100 samples of one constant radius on the axis of the only destination ray,
    # alpha = 13/255 (the wire's RGBA8), sent through splats_update_packed.  A_n = 1 - (1 - a)^n crosses 0.99 at
    # n* = 89 >> K = 4 k-buffer entries, so the ray is re-launched from the cursor more than twenty times.
    n = 100
    quant = [0.0, 0.0, 0.0, 1.0, 1.0, 1.0, 0.1]
    qx = np.uint64(32768)                                   # cell centre 0.50000763 on x and y
    qz = (np.floor((0.2 + 0.005 * np.arange(n)) * 65536.0)).astype(np.uint64)
    qr = np.uint64(6554)                                    # radius 6554 * 0.1 / 65535 ~ 0.01
    samples = (qx | (qx << np.uint64(16)) | (qz << np.uint64(32)) | (qr << np.uint64(48))).astype(np.uint64)
    colours = np.full(n, 1 | (2 << 8) | (3 << 16) | (13 << 24), dtype=np.uint32)
    a = np.float32(13) / np.float32(255)
    A, n_star = np.float32(0), 0
    while A < np.float32(0.99):                             # S9 in float32, one hit at a time
        A = np.float32(np.float64(np.float32(1) - A) * np.float64(a) + np.float64(A))   # T = 1 - A; A = fma(T, a, A)
        n_star += 1
    assert 80 <= n_star <= 95
    assert abs(float(A) - (1.0 - (1.0 - float(a)) ** n_star)) < 1e-5
    cam = synth.look_at((0.5, 0.5, -3.0), center=(0.5, 0.5, 0.5))   # its single pixel's ray is the z axis through (0.5, 0.5)
    with Session(16, 16) as s:
        d_s = torch.from_numpy(samples.view(np.int64)).cuda()
        d_c = torch.from_numpy(colours.view(np.int32)).cuda()
        sp.splats_update_packed(d_s, d_c, n, quant)
        got = s.render(cam, 1, 1)
        scp = oracle.build_scene_packed(samples, colours, quant)
        assert_bvh_bit_exact(scp)
        ref, used = oracle.render(scp, cam, 1, 1, "brute", return_hits=True)
        assert used[0, 0] == n_star                         # the oracle composited exactly the closed form's stack
        assert_rgba_close(got, ref)
        assert got[0, 0, 3] == pytest.approx(1.0 - (1.0 - float(a)) ** n_star, abs=1e-5)
        assert got[0, 0, 3] >= 0.99


def test_all_invalid_frame_renders_zeros():
    W, H = 64, 48
    color = np.ones((H, W, 4), np.float32)
    depth = np.zeros((H, W), np.float32)
    depth[3, 4] = np.nan
    depth[5, 6] = -1.0
    depth[7, 8] = np.inf
    cam = synth.orbit_camera(0.0)
    with Session(W, H) as s:
        s.update(color, depth, cam, W, H, 1.0)
        assert sp.splats_count() == 0
        assert np.all(s.render(cam, W, H) == 0)


@pytest.mark.parametrize("n", [1, 2, 3])
def test_tiny_splat_counts(n):
    W, H = 9, 7
    color, depth, cam = synth.random_frame(W, H, seed=n, fill=1.0)
    keep = np.zeros(W * H, bool)
    keep[[31, 32, 40][:n]] = True
    depth.reshape(-1)[~keep] = 0
    with Session(W, H) as s:
        check_scene(s, color, depth, cam, W, H, 1.0, [cam, synth.orbit_camera(2.0)], mode="brute")


def test_duplicate_morton_codes_from_outlier():
    # one far outlier stretches the bounds so most centres collapse into a few cells
    W, H = 64, 64
    color, depth, cam = synth.random_frame(W, H, seed=21, fill=0.8)
    depth[depth > 0] = 3.0
    depth[0, 0] = 3.0e7
    with Session(W, H) as s:
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(4.0)], mode="bvh")
        codes = sc["sorted_codes"]
        assert (codes[1:] == codes[:-1]).sum() > 100   # the case really has duplicates


def test_zero_extent_axis():
    # one-row image from an axis-aligned camera: every centre has exactly the eye's y
    W, H = 200, 1
    color, depth, cam = synth.random_frame(W, H, seed=4, fill=0.9)
    with Session(W, 8) as s:
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [cam, synth.orbit_camera(1.0)], [(W, 1), (W, 8)], mode="brute")
        assert sc["lo"][1] == sc["hi"][1]


def test_config1_full():
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale, cfg.dst_cams, mode="bvh")


@pytest.mark.parametrize("W,H", [(32, 32), (41, 25), (683, 3), (64, 64)])
def test_pyramid_block_boundaries(W, H):
    # N = 1024, 1025, 2049, 4096: exactly one pyramid block, one leaf into the next, ...
    color, depth, cam = synth.random_frame(W, H, seed=W + H, fill=1.0)
    with Session(W, H) as s:
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(3.0)], mode="bvh")
        assert sc["N"] == W * H


def test_atomic_refit_mode_gives_the_same_tree():
    # SPLATS_OPT_REFIT: the classic atomic-counter refit and the pyramid + per-node searches must give the
    # bit-identical BVH (the default is the tiled tree, which every other test exercises)
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        sp.splats_set_option(sp.OPT_REFIT, sp.REFIT_ATOMIC)
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale, cfg.dst_cams[:1], mode="bvh")
        c2, d2, cam2 = synth.random_frame(127, 65, seed=3, fill=0.4)
        check_scene(s, c2, d2, cam2, 127, 65, 2.0, [synth.orbit_camera(5.0)], mode="bvh")
        sp.splats_set_option(sp.OPT_REFIT, sp.REFIT_PYRAMID)
        check_scene(s, c2, d2, cam2, 127, 65, 2.0, [synth.orbit_camera(5.0)], mode="bvh")
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale, cfg.dst_cams[:1], mode="bvh")
        sp.splats_set_option(sp.OPT_REFIT, sp.REFIT_TILED)   # the default
        check_scene(s, c2, d2, cam2, 127, 65, 2.0, [synth.orbit_camera(5.0)], mode="bvh")
        with pytest.raises(sp.SplatsError):
            sp.splats_set_option(sp.OPT_REFIT, 7)
        with pytest.raises(sp.SplatsError):
            sp.splats_set_option(99, 0)


def _top_runs(codes):
    hi = codes >> np.uint64(31)   # the top 32 code bits: what four passes of the LSD hybrid sort put in order
    brk = np.flatnonzero(np.r_[True, hi[1:] != hi[:-1], True])
    return np.diff(brk)


@pytest.mark.parametrize("outlier,kind", [(300.0, "short"), (600.0, "short"), (2000.0, "long"), (5000.0, "long")])
def test_hybrid_sort_fixup_and_fallback(outlier, kind):
    # The LSD hybrid sort orders by the top 32 code bits and repairs runs that share them: an outlier
    # stretches the bounds until several splats fall into one cell of the top bits.  Short runs
    # (<= 32) are fixed in place, longer ones trigger the full 8-pass sort; same result either way.
    W, H = 64, 64
    color, depth, cam = synth.random_frame(W, H, seed=21, fill=0.8)
    depth[depth > 0] = 3.0
    depth[0, 0] = outlier
    with Session(W, H) as s:
        sp.splats_set_option(sp.OPT_SORT, sp.SORT_HYBRID_LSD)    # the LSD variant of the hybrid sort first ...
        check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(4.0)], mode="bvh")
        sp.splats_set_option(sp.OPT_SORT, sp.SORT_HYBRID)        # ... then the windowed one (default)
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(4.0)], mode="bvh")
        L = _top_runs(sc["sorted_codes"])
        if kind == "short":
            assert (L > 1).sum() > 100 and L.max() <= 32   # the case really exercises the fix-up
        else:
            assert L.max() > 32                             # ... and this one the fallback
        # a second frame in the same context: the fallback flag and barrier are re-armed
        c2, d2, cam2 = synth.random_frame(100, 37, seed=77, fill=0.5)
        check_scene(s, c2, d2, cam2, 100, 37, 1.0, [synth.orbit_camera(4.0)], [(64, 64)], mode="bvh")


@pytest.mark.parametrize("mode", ["lsd8", "lsd8_launches", "hybrid_lsd"])
def test_sort_modes_give_the_same_order(mode):
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        sp.splats_set_option(sp.OPT_SORT, {"lsd8": sp.SORT_LSD8, "lsd8_launches": sp.SORT_LSD8_LAUNCHES,
                                           "hybrid_lsd": sp.SORT_HYBRID_LSD}[mode])
        check_scene(s, color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale, cfg.dst_cams[:1], mode="bvh")
        c2, d2, cam2 = synth.random_frame(127, 65, seed=3, fill=0.4)
        check_scene(s, c2, d2, cam2, 127, 65, 2.0, [synth.orbit_camera(5.0)], mode="bvh")
        with pytest.raises(sp.SplatsError):
            sp.splats_set_option(sp.OPT_SORT, 9)


@pytest.mark.parametrize("W,H", [(128, 80), (200, 150)])
def test_windowed_sort_bucket_overflow_falls_back(W, H):
    # all splats but one at one depth and an outlier far away: the top code bits agree for (almost) all of
    # them, so one bucket of the windowed hybrid sort is larger than a window (4096): the launch must fall
    # back to the LSD passes (and, the runs being long, to all eight) and give the same order
    color, depth, cam = synth.random_frame(W, H, seed=33, fill=0.9)
    depth[depth > 0] = 3.0
    depth[0, 0] = 9000.0
    with Session(W, H) as s:
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(4.0)], mode="bvh", sample=2000)
        assert sc["N"] > 8192
        # and a well-behaved frame right after it: flags are re-armed
        cfg = synth.make_config(0)
        c2, d2 = synth.source_frame(cfg, 0)
        check_scene(s, c2, d2, cfg.src_cams[0], cfg.W, cfg.H, 1.0, cfg.dst_cams[:1], mode="bvh")


def test_dense_frame_five_pass_hybrid_sort_and_all_tile_sizes():
    # N > 2^19: the hybrid sort runs 5 passes (top 39 bits) starting from the second buffer;
    # then smaller frames in the same context walk through the 4096/2048/1024-element tile paths.
    W, H = 2304, 1000
    color, depth, cam = synth.dense_frame(W, H, seed=5)
    with Session(W, H) as s:
        sp.splats_set_option(sp.OPT_SORT, sp.SORT_HYBRID_LSD)
        check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(2.0)], mode="bvh", sample=1024)
        sp.splats_set_option(sp.OPT_SORT, sp.SORT_HYBRID)
        sc, _ = check_scene(s, color, depth, cam, W, H, 1.0, [synth.orbit_camera(2.0)], mode="bvh", sample=4096)
        assert sc["N"] == W * H > (1 << 20)
        for (w, h) in ((1500, 800), (1400, 700), (900, 500), (640, 360)):
            c2, d2, cam2 = synth.dense_frame(w, h, seed=w)
            check_scene(s, c2, d2, cam2, w, h, 1.0, [synth.orbit_camera(-2.0)], mode="bvh", sample=2048)


def test_repeated_updates_and_size_changes():
    # frame-parity double buffering: A, B (other size), A again must reproduce A
    cfg = synth.make_config(0)
    colorA, depthA = synth.source_frame(cfg, 0)
    colorB, depthB, camB = synth.random_frame(100, 37, seed=77, fill=0.5)
    dst = synth.orbit_camera(7.0)
    with Session(128, 64) as s:
        s.update(colorA, depthA, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
        a1 = s.render(dst, 64, 64)
        scB, _ = check_scene(s, colorB, depthB, camB, 100, 37, 2.0, [dst], [(80, 40)], mode="brute")
        scA, _ = check_scene(s, colorA, depthA, cfg.src_cams[0], cfg.W, cfg.H, 1.0, [dst], mode="brute")
        a2 = s.render(dst, 64, 64)
        assert np.array_equal(a1, a2)


def test_host_buffer_entry_points_match_device_ones():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
        a = s.render(cfg.dst_cams[0], 64, 64)
        hc = torch.from_numpy(color).pin_memory()
        hd = torch.from_numpy(depth).pin_memory()
        ho = torch.empty((64, 64, 4), dtype=torch.float32).pin_memory()
        sp.splats_update_host(hc, hd, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
        sp.splats_render_host(cfg.dst_cams[0], 64, 64, ho)
        sp.splats_synchronize()
        assert np.array_equal(ho.numpy(), a)


def test_host_pipeline_many_frames_in_flight():
    # more updates / renders in flight than staging buffers (2 in, 3 out): every image must be
    # the one its own frame and camera give, whatever the copy streams overlap
    frames = [synth.random_frame(96, 54, seed=100 + i, fill=0.5 + 0.05 * i) for i in range(5)]
    cams = [synth.orbit_camera(2.0 * j) for j in range(4)]
    with Session(96, 54) as s:
        ref = []
        for color, depth, cam in frames:
            s.update(color, depth, cam, 96, 54, 1.5)
            ref.append([s.render(c, 96, 54) for c in cams])
        hc = [torch.from_numpy(f[0]).pin_memory() for f in frames]
        hd = [torch.from_numpy(f[1]).pin_memory() for f in frames]
        ho = [[torch.empty((54, 96, 4), dtype=torch.float32).pin_memory() for _ in cams] for _ in frames]
        for i, (color, depth, cam) in enumerate(frames):
            sp.splats_update_host(hc[i], hd[i], cam, 96, 54, 1.5)
            for j, c in enumerate(cams):
                sp.splats_render_host(c, 96, 54, ho[i][j])
        sp.splats_synchronize()
        for i in range(len(frames)):
            for j in range(len(cams)):
                assert np.array_equal(ho[i][j].numpy(), ref[i][j]), (i, j)


def test_error_codes():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    cam = cfg.src_cams[0]
    with pytest.raises(sp.SplatsError) as e:
        sp.splats_update(torch.zeros(16, device="cuda"), torch.zeros(4, device="cuda"), cam, 2, 2, 1.0)
    assert e.value.code == -4   # no context
    with Session(64, 64) as s:
        out = torch.empty((64, 64, 4), device="cuda")
        with pytest.raises(sp.SplatsError) as e:
            sp.splats_render(cam, 64, 64, out)
        assert e.value.code == -2   # no BVH yet
        dc, dd = torch.from_numpy(color).cuda(), torch.from_numpy(depth).cuda()
        for bad in (0.0, -1.0, float("nan"), float("inf")):
            with pytest.raises(sp.SplatsError) as e:
                sp.splats_update(dc, dd, cam, 64, 64, bad)
            assert e.value.code == -1
        badcam = cam.copy(); badcam[4] = np.nan
        with pytest.raises(sp.SplatsError) as e:
            sp.splats_update(dc, dd, badcam, 64, 64, 1.0)
        assert e.value.code == -1
        with pytest.raises(sp.SplatsError) as e:
            sp._check(sp.lib().splats_update(dc.data_ptr(), dd.data_ptr(), None, 64, 64, 1.0))
        assert e.value.code == -1
        big = torch.zeros(65 * 64 * 4, device="cuda")
        with pytest.raises(sp.SplatsError) as e:
            sp.splats_update(big, big, cam, 65, 64, 1.0)   # beyond capacity
        assert e.value.code == -1
        with pytest.raises(sp.SplatsError) as e:
            sp.splats_create(8, 8)                          # context already exists
        assert e.value.code == -4
        sp.splats_update(dc, dd, cam, 64, 64, 1.0)          # still usable after the errors
        sp.splats_render(cam, 64, 64, out)
        torch.cuda.synchronize()
        assert "context" in sp.splats_last_error() or sp.splats_last_error() != ""


def test_rgba8_output_device_and_host():
    # splats_render_rgba8 / splats_render_host_rgba8: the composited image rounded to 8 bit per channel
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    c2, d2, cam2 = synth.random_frame(130, 50, seed=8, fill=0.6)
    sc2 = oracle.build_scene(c2, d2, cam2, 130, 50, 2.0)
    with Session(130, 64) as s:
        for (scn, col, dep, cam, W, H, rs, dst, W2, H2) in ((sc, color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, cfg.dst_cams[0], 64, 64),
                                                            (sc2, c2, d2, cam2, 130, 50, 2.0, synth.orbit_camera(7.0), 97, 33)):
            s.update(col, dep, cam, W, H, rs)
            want = oracle.quantise_image(oracle.render(scn, dst, W2, H2, "brute"))
            out = torch.full((H2, W2), 0x5a5a5a5a, dtype=torch.int32, device="cuda")
            sp.splats_render_rgba8(dst, W2, H2, out)
            torch.cuda.synchronize()
            np.testing.assert_array_equal(out.cpu().numpy().view(np.uint32), want)
            host = torch.zeros((H2, W2), dtype=torch.int32).pin_memory()
            sp.splats_render_host_rgba8(dst, W2, H2, host)
            sp.splats_synchronize()
            np.testing.assert_array_equal(host.numpy().view(np.uint32), want)
            assert (want != 0).mean() > 0.02


def test_overlapping_renders_option():
    # SPLATS_OPT_OVERLAP: consecutive renders of one BVH into disjoint images may run concurrently.
    # Eleven renders in a row (the ninth is serialised), two of them into the same buffer, an
    # update in between, first-hit / rgba8 / points mixed in: every image equals the serial result.
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    c2, d2, cam2 = synth.random_frame(300, 200, seed=12, fill=0.7)
    sc2 = oracle.build_scene(c2, d2, cam2, 300, 200, 2.0)
    W, H = cfg.W, cfg.H
    cams = [synth.orbit_camera(2.0 * i, 1.0 * i) for i in range(11)]
    with Session(W, H) as s:
        sp.splats_set_option(sp.OPT_OVERLAP, 1)
        s.update(color, depth, cfg.src_cams[0], W, H, 1.0)
        outs = [torch.full((H, W, 4), -7.0, dtype=torch.float32, device="cuda") for _ in range(11)]
        for i, cam in enumerate(cams):
            sp.splats_render(cam, W, H, outs[i])
        # stream-ordered copies of EARLIER images right behind the last render, no device-wide
        # synchronisation: completion must be in launch order for them to see finished images
        early = [torch.empty((H, W, 4), dtype=torch.float32).pin_memory() for _ in range(3)]
        for i in range(3):
            early[i].copy_(outs[7 + i], non_blocking=True)
        torch.cuda.current_stream().synchronize()
        early = [e.clone() for e in early]
        shared = torch.full((H, W, 4), -7.0, dtype=torch.float32, device="cuda")
        sp.splats_render(cams[0], W, H, shared)
        sp.splats_render(cams[5], W, H, shared)             # same image twice: the second one must win
        fh = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
        sp.splats_render_first_hit(cams[3], W, H, fh)
        o8 = torch.empty((H, W), dtype=torch.int32, device="cuda")
        sp.splats_render_rgba8(cams[4], W, H, o8)
        pts = torch.empty((H, W, 4), dtype=torch.float32, device="cuda")
        sp.splats_render_points(cams[2], W, H, 2, pts)
        # a new frame while the renders above may still be in flight, then renders of the new BVH
        dc2, dd2 = torch.from_numpy(c2).cuda(), torch.from_numpy(d2).cuda()
        sp.splats_update(dc2, dd2, cam2, 300, 200, 2.0)
        new = [torch.empty((120, 160, 4), dtype=torch.float32, device="cuda") for _ in range(3)]
        for i in range(3):
            sp.splats_render(cams[i + 1], 160, 120, new[i])
        torch.cuda.synchronize()
        for i in (0, 3, 4, 7, 10):
            assert_rgba_close(outs[i].cpu().numpy(), oracle.render(sc, cams[i], W, H, "bvh"), f"render {i}")
        for i in range(3):
            assert torch.equal(early[i], outs[7 + i].cpu()), f"stream-ordered copy of render {7 + i} saw an unfinished image"
        ref5 = oracle.render(sc, cams[5], W, H, "bvh")
        assert_rgba_close(shared.cpu().numpy(), ref5, "aliased image")
        assert np.array_equal(fh.cpu().numpy(), oracle.render(sc, cams[3], W, H, "bvh", first_hit=True))
        np.testing.assert_array_equal(o8.cpu().numpy().view(np.uint32), oracle.quantise_image(oracle.render(sc, cams[4], W, H, "bvh")))
        assert np.array_equal(pts.cpu().numpy(), oracle.render_points(sc, cams[2], W, H, 2))
        for i in range(3):
            assert_rgba_close(new[i].cpu().numpy(), oracle.render(sc2, cams[i + 1], 160, 120, "bvh"), f"new frame render {i}")
        # serial and overlapped executions give identical bits
        sp.splats_set_option(sp.OPT_OVERLAP, 0)
        serial = torch.empty((120, 160, 4), dtype=torch.float32, device="cuda")
        sp.splats_render(cams[2], 160, 120, serial)
        torch.cuda.synchronize()
        assert torch.equal(serial, new[1])


@pytest.mark.parametrize("seed", range(10))
def test_seeded_fuzz_whole_path(seed):
    # random sizes, fills, radii, source kinds (frame / packed) and options; everything bit-exact
    rng = np.random.default_rng(1000 + seed)
    W, H = int(rng.integers(1, 400)), int(rng.integers(1, 300))
    fill = float(rng.choice([0.02, 0.3, 0.7, 1.0]))
    r_scale = float(rng.choice([0.5, 1.0, 1.0, 2.0, 3.5]))
    radius = [(0, 0.0), (0, 0.0), (1, 0.006), (2, 0.3)][int(rng.integers(4))]
    color, depth, cam = synth.random_frame(W, H, seed=seed, fill=fill, cam=synth.orbit_camera(float(rng.uniform(-40, 40)), float(rng.uniform(-20, 20))))
    if seed % 3 == 0:
        depth[depth > 0] = np.float32(3.0 + 0.01 * (seed % 5))        # coplanar: many equal codes / equal t
    W2, H2 = int(rng.integers(1, 200)), int(rng.integers(1, 150))
    dst = synth.orbit_camera(float(rng.uniform(-30, 30)), float(rng.uniform(-15, 15)), float(rng.uniform(2.0, 5.0)))
    with Session(max(W, 200), max(H, 150)) as s:
        sp.splats_set_option(sp.OPT_OVERLAP, seed % 2)
        sp.splats_set_option(sp.OPT_SORT, [sp.SORT_HYBRID, sp.SORT_HYBRID_LSD, sp.SORT_LSD8][seed % 3])
        sc, _ = check_scene(s, color, depth, cam, W, H, r_scale, [dst, cam], [(W2, H2), (W2, H2)], mode="bvh", radius=radius)
        fh = s.render(dst, W2, H2, first_hit=True)
        assert np.array_equal(fh, oracle.render(sc, dst, W2, H2, "bvh", first_hit=True))
        pts = torch.empty((H2, W2, 4), dtype=torch.float32, device="cuda")
        sp.splats_render_points(dst, W2, H2, 1 + seed % 3, pts)
        assert np.array_equal(pts.cpu().numpy(), oracle.render_points(sc, dst, W2, H2, 1 + seed % 3))
        # the same frame through the wire format
        quant = np.array([-4, -4, -4, 5, 5, 5, 0.05], np.float32)
        rs, rc = oracle.pack(color, depth, cam, W, H, r_scale, quant, radius[0], radius[1])
        scp = oracle.build_scene_packed(rs, rc, quant)
        ws = torch.from_numpy(np.ascontiguousarray(rs.view(np.int64) if len(rs) else np.zeros(1, np.int64))).cuda()
        cs = torch.from_numpy(np.ascontiguousarray(rc.view(np.int32) if len(rc) else np.zeros(1, np.int32))).cuda()
        sp.splats_update_packed(ws, cs, len(rs), quant)
        assert_bvh_bit_exact(scp)
        assert_rgba_close(s.render(dst, W2, H2), oracle.render(scp, dst, W2, H2, "bvh"), "packed")
        sp.splats_set_radius(0, 0.0)


def test_decoupled_build_begin_commit():
    # splats_update_begin / splats_update_commit: the next BVH is built on the library's stream
    # while renders of the current one run; every image and every BVH equals the sequential result.
    cfg = synth.make_config(1)
    frames = [synth.source_frame(cfg, 0) + (cfg.src_cams[0], cfg.W, cfg.H, 1.0)]
    for b, (W, H, rs) in enumerate(((300, 200, 2.0), (512, 512, 1.0), (64, 64, 1.0))):
        c, d, cam = synth.random_frame(W, H, seed=60 + b, fill=0.6)
        frames.append((c, d, cam, W, H, rs))
    scenes = [oracle.build_scene(c, d, cam, W, H, rs) for (c, d, cam, W, H, rs) in frames]
    dev = [(torch.from_numpy(c).cuda(), torch.from_numpy(d).cuda()) for (c, d, *_ ) in frames]
    cams = [synth.orbit_camera(3.0 * i, 2.0 * i) for i in range(4)]
    with Session(512, 512) as s:
        sp.splats_set_option(sp.OPT_OVERLAP, 1)
        with pytest.raises(sp.SplatsError):
            sp.splats_update_commit()                                   # nothing pending
        c0, d0, cam0, W0, H0, rs0 = frames[0]
        sp.splats_update(dev[0][0], dev[0][1], cam0, W0, H0, rs0)
        outs = []
        reuse = torch.full((120, 160, 4), -7.0, dtype=torch.float32, device="cuda")
        for k in range(len(frames)):
            nxt = (k + 1) % len(frames)
            cn, dn, camn, Wn, Hn, rsn = frames[nxt]
            sp.splats_update_begin(dev[nxt][0], dev[nxt][1], camn, Wn, Hn, rsn)     # builds BVH k+1 ...
            with pytest.raises(sp.SplatsError):
                sp.splats_update_begin(dev[nxt][0], dev[nxt][1], camn, Wn, Hn, rsn)
            with pytest.raises(sp.SplatsError):
                sp.splats_update(dev[nxt][0], dev[nxt][1], camn, Wn, Hn, rsn)
            imgs = [torch.full((120, 160, 4), -7.0, dtype=torch.float32, device="cuda") for _ in cams]
            for cam, img in zip(cams, imgs):                                           # ... while BVH k is rendered
                sp.splats_render(cam, 160, 120, img)
            outs.append(imgs)
            sp.splats_update_commit()
            # the same image buffer is rendered into from the old BVH (possibly still in flight) and,
            # right after the commit, from the new one: the second write must win
            sp.splats_render(cams[0], 160, 120, reuse)
            if k == 0:
                first_reuse_scene = nxt
            if k == 1:
                torch.cuda.synchronize()
                assert_bvh_bit_exact(scenes[nxt])                                      # the committed BVH is the new one
        sp.splats_synchronize()
        torch.cuda.synchronize()
        for k, imgs in enumerate(outs):
            for cam, img in zip(cams, imgs):
                assert_rgba_close(img.cpu().numpy(), oracle.render(scenes[k], cam, 160, 120, "bvh"), f"step {k}")
        # after the loop the current BVH is frame 0 again
        assert_bvh_bit_exact(scenes[0])
        assert_rgba_close(reuse.cpu().numpy(), oracle.render(scenes[0], cams[0], 160, 120, "bvh"), "reused image")


def test_exact_nodes_option_changes_nothing():
    # SPLATS_OPT_EXACT_NODES only adds the 64-byte exact records: keys, topology, the quantised
    # traversal records and the images are the same with and without it; without it the exact boxes
    # cannot be exported
    cfg = synth.make_config(1)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    res = {}
    for exact in (False, True):
        with Session(cfg.W, cfg.H, exact_nodes=exact) as s:
            s.update(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
            assert_bvh_bit_exact(sc, exact=exact)
            if not exact:
                with pytest.raises(sp.SplatsError):
                    sp.splats_export()
                with pytest.raises(sp.SplatsError):
                    sp.splats_export_child_boxes()
            res[exact] = (sp.splats_export_qnodes()["qnodes"].cpu().numpy(), s.render(cfg.dst_cams[1], cfg.W, cfg.H))
    assert np.array_equal(res[False][0], res[True][0])
    assert np.array_equal(res[False][1], res[True][1])


def test_quantised_boxes_contain_the_exact_ones():
    # decode the traversal records in float64 and compare with the oracle's exact boxes: never smaller,
    # at most one code step larger per plane (independent of the oracle's float32 statement, oracle.quantise_child_boxes)
    W, H = 200, 120
    color, depth, _ = synth.random_frame(W, H, 5, fill=0.8)
    cam = synth.orbit_camera(20.0)
    sc = oracle.build_scene(color, depth, cam, W, H, 1.5)
    with Session(W, H) as s:
        s.update(color, depth, cam, W, H, 1.5)
        q = sp.splats_export_qnodes()
    rec = q["qnodes"].cpu().numpy().view(np.uint32)
    fr = q["frame"].cpu().numpy().astype(np.float64)
    qlo = fr[0:3] - fr[6]
    step = ((fr[3:6] + fr[6]) - qlo) / 65535.0
    w = rec[:, 0:6].reshape(-1, 2, 3)
    lo = qlo + (w & 0xffff) * step
    hi = qlo + (w >> 16) * step
    want = sc["aabbs"][sc["children"]].astype(np.float64)
    eps = 1e-6 * np.abs(want).max()
    assert np.all(lo <= want[:, :, 0:3] + eps) and np.all(hi >= want[:, :, 3:6] - eps)
    assert np.all(lo >= want[:, :, 0:3] - step - eps) and np.all(hi <= want[:, :, 3:6] + step + eps)


def test_alternating_frames_under_overlap_stress():
    # ADVICE (round 1): kernels that skip griddepcontrol.wait read through the non-coherent path what an earlier
    # grid produced.  Two frames of very different N alternate for ten updates, three renders behind each, all
    # enqueued back to back with SPLATS_OPT_OVERLAP on and no synchronisation: the BVH sets, key buffers, frame
    # states and status words are reused every other update, so a stale line or a kernel running ahead of its
    # producer shows up as a wrong image or a wrong tree at the end.
    cfg = synth.make_config(1)
    W, H = cfg.W, cfg.H
    colA, depA = synth.source_frame(cfg, 0)
    camA = cfg.src_cams[0]
    colB, depB, camB = synth.random_frame(W, H, seed=9, fill=0.35)
    scenes = [oracle.build_scene(colA, depA, camA, W, H, 1.0), oracle.build_scene(colB, depB, camB, W, H, 1.0)]
    assert scenes[1]["N"] > 3 * scenes[0]["N"]
    cams = [synth.orbit_camera(3.0), synth.orbit_camera(-6.0, 2.0), synth.orbit_camera(11.0)]
    rng = np.random.default_rng(3)
    px = np.sort(rng.choice(W * H, size=30_000, replace=False)).astype(np.int64)
    refs = [[oracle.render(sc, cam, W, H, "bvh", pixels=px) for cam in cams] for sc in scenes]
    frames = [(torch.from_numpy(colA).cuda(), torch.from_numpy(depA).cuda(), camA),
              (torch.from_numpy(colB).cuda(), torch.from_numpy(depB).cuda(), camB)]
    n_updates = 10
    with Session(W, H, exact_nodes=False):
        sp.splats_set_option(sp.OPT_OVERLAP, 1)
        outs = [[torch.full((H, W, 4), -7.0, dtype=torch.float32, device="cuda") for _ in cams] for _ in range(n_updates)]
        for it in range(n_updates):
            dc, dd, cam = frames[it & 1]
            sp.splats_update(dc, dd, cam, W, H, 1.0)
            for j, c in enumerate(cams):
                sp.splats_render(c, W, H, outs[it][j])
        torch.cuda.synchronize()
        assert_bvh_bit_exact(scenes[(n_updates - 1) & 1], exact=False)
        for it in range(n_updates):
            for j in range(len(cams)):
                got = outs[it][j].cpu().numpy().reshape(-1, 4)[px]
                assert_rgba_close(got, refs[it & 1][j], f"update {it}, camera {j}")
