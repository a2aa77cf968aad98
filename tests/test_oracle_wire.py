"""Pins for the wire format of SURVEY.md sec. 8(f) row 2 ("quantize the object space
coordinate and pack it together with the radius into 64 bits", compaction of zero-radius samples;
PAPER.md:103 "32 bits per color and 64 bits per object space sample").  The bit split is this
repository's reading; these tests pin the oracle's pack / decode to it by
hand-worked words, error bounds and invariants."""
import numpy as np
import pytest

import oracle
import synth

UNIT = [0, 0, 0, 1, 1, 1, 0.5]


def _one_pixel(t, cam=None, color=(0.25, 0.5, 1.0, 0.5)):
    cam = synth.orbit_camera(0.0) if cam is None else cam
    depth = np.array([[t]], np.float32)
    col = np.array([[color]], np.float32)
    return col, depth, cam


def test_hand_worked_sample_word_and_colour_word():
    # 1x1 image: the only ray is the camera axis; put the eye at (0.5, 0.25, 2.75) looking down -z,
    # so that depth 2 lands on p = (0.5, 0.25, 0.75); constant radius 0.25 = r_max / 2.
    cam = np.array([0.5, 0.25, 2.75, 1, 0, 0, 0, 1, 0, 0, 0, -1, 0.5], np.float32)
    col, depth, _ = _one_pixel(2.0)
    s, c8 = oracle.pack(col, depth, cam, 1, 1, 1.0, UNIT, oracle.RADIUS_CONSTANT, 0.25)
    # x = 0.5 -> 32768, y = 0.25 -> 16384, z = 0.75 -> 49152, r: ceil(0.5 * 65535) = 32768
    assert s.tolist() == [(32768 << 48) | (49152 << 32) | (16384 << 16) | 32768]
    # 0.25 -> 64 (63.75 + .5 = 64.25), 0.5 -> 128 (127.5 + .5 = 128.0), 1.0 -> 255, alpha 0.5 -> 128
    assert c8.tolist() == [64 | (128 << 8) | (255 << 16) | (128 << 24)]
    assert s.dtype.itemsize * 8 == 64 and c8.dtype.itemsize * 8 == 32
    sphere, rgba, valid = oracle.decode(s, c8, UNIT)
    cell = 1.0 / 65536
    np.testing.assert_allclose(sphere[0], [0.5 + cell / 2, 0.25 + cell / 2, 0.75 + cell / 2, 32768 * 0.5 / 65535], rtol=1e-7)
    np.testing.assert_array_equal(rgba[0], np.array([64, 128, 255, 128], np.float32) / np.float32(255))
    assert valid.tolist() == [1]


def test_position_error_is_at_most_half_a_cell_and_radius_never_shrinks():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    quant = np.array([-0.1, -0.2, -0.3, 1.2, 1.1, 1.4, 0.1], np.float32)
    s, c8 = oracle.pack(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, quant)
    sphere, valid, n = oracle.unproject(depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    assert len(s) == n > 100
    exact = sphere[valid == 1]                         # compaction keeps pixel order
    dec, rgba, dv = oracle.decode(s, c8, quant)
    assert dv.all()
    cell = (quant[3:6] - quant[:3]).astype(np.float64) / 65536
    err = np.abs(dec[:, :3].astype(np.float64) - exact[:, :3])
    assert np.all(err <= cell / 2 * (1 + 1e-3) + 1e-7) and err.max() > cell.min() / 4
    rstep = 0.1 / 65535
    assert np.all(dec[:, 3] >= exact[:, 3]) and np.all(dec[:, 3] - exact[:, 3] <= rstep * (1 + 1e-3))
    # colours: nearest of 256 levels
    src = color.reshape(-1, 4)[valid == 1]
    assert np.abs(rgba.astype(np.float64) - np.clip(src, 0, 1)).max() <= 0.5 / 255 + 1e-7


def test_corners_clamp_and_zero_radius_is_dropped():
    cam = np.array([0.0, 0.0, 2.0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 0.5], np.float32)
    col, depth, _ = _one_pixel(2.0)            # p = (0, 0, 0) = lo corner
    s, _ = oracle.pack(col, depth, cam, 1, 1, 1.0, UNIT, oracle.RADIUS_CONSTANT, 9.0)   # r > r_max
    assert s.tolist() == [65535 << 48]
    col, depth, _ = _one_pixel(1.0)            # p = (0, 0, 1): z = hi -> clamps to the last cell
    s, _ = oracle.pack(col, depth, cam, 1, 1, 1.0, UNIT, oracle.RADIUS_CONSTANT, 1e-9)  # tiny radius -> 1, not 0
    assert s.tolist() == [(1 << 48) | (65535 << 32)]
    col, depth, _ = _one_pixel(5.0)            # p = (0, 0, -3): outside the box -> clamps to 0
    s, _ = oracle.pack(col, depth, cam, 1, 1, 1.0, UNIT, oracle.RADIUS_CONSTANT, 0.5)
    assert s.tolist() == [65535 << 48]
    # opacity radius with floor 0 and alpha 0 gives r = 0: "we set the radius to zero ... send only
    # those object space samples with non-zero radius"
    col, depth, _ = _one_pixel(1.5, color=(0, 0, 0, 0))
    s, c8 = oracle.pack(col, depth, cam, 1, 1, 1.0, UNIT, oracle.RADIUS_OPACITY, 0.0)
    assert len(s) == 0 and len(c8) == 0
    # a received word with radius field 0 is dropped by the client
    sphere, rgba, valid = oracle.decode([12345, (7 << 48) | 5], [0, 0xffffffff], UNIT)
    assert valid.tolist() == [0, 1]
    sc = oracle.build_scene_packed([12345, (7 << 48) | 5], [0, 0xffffffff], UNIT)
    assert sc["N"] == 1 and sc["sorted_ids"].tolist() == [1] and np.all(sc["rgba_sorted"] == 1.0)


def test_compaction_keeps_pixel_order_and_count():
    color, depth, cam = synth.random_frame(37, 21, seed=3, fill=0.4)
    quant = [-3, -3, -3, 4, 4, 4, 0.05]
    s, c8 = oracle.pack(color, depth, cam, 37, 21, 1.0, quant)
    v = depth.reshape(-1) > 0
    assert len(s) == v.sum()
    # every pixel packed on its own gives the same word: compaction only removes and never reorders
    idx = np.flatnonzero(v)
    for j in (0, 1, len(idx) // 2, len(idx) - 1):
        d1 = np.zeros_like(depth); d1.reshape(-1)[idx[j]] = depth.reshape(-1)[idx[j]]
        s1, c1 = oracle.pack(color, d1, cam, 37, 21, 1.0, quant)
        assert s1.tolist() == [s[j]] and c1.tolist() == [c8[j]]


def test_scene_from_packed_samples_renders_like_the_float_scene():
    # the decoded scene is the float scene moved by <= half a cell: same tree size, images close
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    quant = [0, 0, 0, 1, 1, 1, 0.1]
    s, c8 = oracle.pack(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, quant)
    scp = oracle.build_scene_packed(s, c8, quant)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    assert scp["N"] == sc["N"] and scp["children"].shape == sc["children"].shape
    a = oracle.render(scp, cfg.dst_cams[0], 64, 64, "brute")
    b = oracle.render(scp, cfg.dst_cams[0], 64, 64, "bvh")
    assert np.array_equal(a, b)
    ref = oracle.render(sc, cfg.dst_cams[0], 64, 64, "brute")
    assert ((a[..., 3] > 0) == (ref[..., 3] > 0)).mean() > 0.99


def test_image_quantisation_hand_values():
    # the display format of splats_render_rgba8 = the wire's colour rounding, per channel
    img = np.array([[[0.25, 0.5, 1.0, 0.5], [0, 0, 0, 0]], [[2.0, -1.0, 0.999, 0.002], [1 / 255, 0.5 / 255, 0.49 / 255, 254.5 / 255]]], np.float32)
    q = oracle.quantise_image(img)
    assert q.shape == (2, 2) and q.dtype == np.uint32
    assert q.tolist() == [[0x80FF8040, 0], [0x01FF00FF, (255 << 24) | (0 << 16) | (1 << 8) | 1]]
