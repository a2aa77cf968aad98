"""Pins for the point-primitive comparison renderer (PAPER.md:37,55,67,
101): hand-placed points, a float64 re-projection written here, and the paper's qualitative claim."""
import numpy as np
import pytest

import oracle
import synth

CAM = np.array([0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 0.5], np.float32)   # at the origin, looking down -z, tan = 0.5


def _scene(points, cols=None, ids=None):
    pts = np.asarray(points, np.float32).reshape(-1, 3)
    n = len(pts)
    sphere = np.concatenate([pts, np.full((n, 1), 0.01, np.float32)], axis=1)
    cols = np.tile(np.array([[0.2, 0.4, 0.6, 0.8]], np.float32), (n, 1)) if cols is None else np.asarray(cols, np.float32)
    ids = np.arange(n, dtype=np.uint32) if ids is None else np.asarray(ids, np.uint32)
    return dict(N=n, sphere_sorted=np.ascontiguousarray(sphere), rgba_sorted=np.ascontiguousarray(cols), sorted_ids=ids)


def test_point_on_the_axis_covers_the_pixels_around_the_image_centre():
    sc = _scene([[0, 0, -3]])
    for W, H, s, xs, ys in ((9, 9, 1, [4], [4]), (9, 9, 3, [3, 4, 5], [3, 4, 5]), (8, 8, 2, [3, 4], [3, 4]),
                            (8, 8, 1, [4], [4]), (9, 9, 2, [4, 5], [4, 5])):
        out = oracle.render_points(sc, CAM, W, H, s)
        yy, xx = np.nonzero(out[..., 3])
        assert sorted(set(xx)) == xs and sorted(set(yy)) == ys and len(xx) == s * s
        assert np.array_equal(out[ys[0], xs[0]], sc["rgba_sorted"][0])


def test_window_coordinates_hand_worked():
    # z = -2, tan = 0.5: the image plane half extent at that depth is 1; x = 0.5 -> ndc 0.5 ->
    # window x = (0.5 + 1) * 8 / 2 = 6 -> size 1 is odd: pixel floor(6) = 6 (centre 6.5 in (5.5, 6.5])
    # y = 0.25 -> ndc 0.25 -> window y = (1 - 0.25) * 4 = 3 -> pixel 3
    out = oracle.render_points(_scene([[0.5, 0.25, -2]]), CAM, 8, 8, 1)
    assert np.argwhere(out[..., 3] > 0).tolist() == [[3, 6]]
    # x = 0.4 -> window x = 5.6 -> pixel 5; size 2 (even): centre floor(5.6 + .5) = 6 -> pixels 5, 6
    out = oracle.render_points(_scene([[0.4, 0.25, -2]]), CAM, 8, 8, 1)
    assert np.argwhere(out[..., 3] > 0).tolist() == [[3, 5]]
    out = oracle.render_points(_scene([[0.4, 0.25, -2]]), CAM, 8, 8, 2)
    assert sorted(set(np.nonzero(out[..., 3])[1])) == [5, 6] and sorted(set(np.nonzero(out[..., 3])[0])) == [2, 3]


def test_nearest_point_wins_and_ties_go_to_the_smaller_id():
    red, blue = [0.5, 0, 0, 0.5], [0, 0, 0.9, 1.0]
    for order in ((0, 1), (1, 0)):
        pts = [[0, 0, -3], [0, 0, -2]]
        cols = [red, blue]
        sc = _scene([pts[i] for i in order], [cols[i] for i in order], list(order))
        out = oracle.render_points(sc, CAM, 5, 5, 1)
        assert np.array_equal(out[2, 2], np.asarray(blue, np.float32))       # z = -2 is nearer; no blending
    for ids, want in (([7, 3], blue), ([3, 7], red)):
        out = oracle.render_points(_scene([[0, 0, -2], [0, 0, -2]], [red, blue], ids), CAM, 5, 5, 1)
        assert np.array_equal(out[2, 2], np.asarray(want, np.float32))


def test_points_behind_the_eye_or_off_screen_are_dropped():
    sc = _scene([[0, 0, 3], [0, 0, 0], [50, 0, -2], [0, -50, -2], [1e30, 0, -1]])
    assert np.all(oracle.render_points(sc, CAM, 16, 16, 3) == 0)
    # a point just outside still contributes the part of its square that is inside
    out = oracle.render_points(_scene([[1.05, 0, -2]]), CAM, 8, 8, 3)
    assert (out[..., 3] > 0).sum() == 3 and set(np.nonzero(out[..., 3])[1]) == {7}


def test_against_a_float64_projection_written_here():
    rng = np.random.default_rng(5)
    cam = synth.orbit_camera(20.0, 10.0, 3.0)
    pts = rng.uniform(0.1, 0.9, size=(400, 3))
    W, H, s = 64, 48, 3
    e, R, U, F, tau = cam[0:3].astype(np.float64), cam[3:6], cam[6:9], cam[9:12], float(cam[12])
    v = pts.astype(np.float32).astype(np.float64) - e
    zc = v @ F; wx = ((v @ R) / (zc * tau * W / H) + 1) * W / 2; wy = (1 - (v @ U) / (zc * tau)) * H / 2
    zbuf = np.full((H, W), np.inf); own = np.full((H, W), -1)
    margin = np.minimum(np.abs((wx - s / 2 - 0.5) - np.round(wx - s / 2 - 0.5)), np.abs((wy - s / 2 - 0.5) - np.round(wy - s / 2 - 0.5)))
    keep = margin > 1e-3                     # points whose square edge sits on a pixel centre are left out
    for i in np.flatnonzero(keep):
        x0, y0 = int(np.floor(wx[i] - s / 2 - 0.5)) + 1, int(np.floor(wy[i] - s / 2 - 0.5)) + 1
        for y in range(max(y0, 0), min(y0 + s, H)):
            for x in range(max(x0, 0), min(x0 + s, W)):
                if zc[i] < zbuf[y, x]:
                    zbuf[y, x], own[y, x] = zc[i], i
    cols = rng.uniform(0.1, 1, size=(400, 4)).astype(np.float32)
    out = oracle.render_points(_scene(pts[keep], cols[keep], np.flatnonzero(keep)), cam, W, H, s)
    want = np.where(own[..., None] >= 0, cols[np.maximum(own, 0)], 0).astype(np.float32)
    assert (own >= 0).mean() > 0.1 and np.array_equal(out, want)


def test_identity_camera_with_one_pixel_points_reproduces_the_source_image():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    out = oracle.render_points(sc, cfg.src_cams[0], cfg.W, cfg.H, 1)
    v = depth > 0
    assert np.array_equal(out[v], color[v]) and np.all(out[~v] == 0)


def test_fixed_size_points_leave_holes_when_the_camera_moves_in():
    # with rasterisation "the point primitives' size is fixed to a certain number of
    # pixels, and this causes a variety of artifacts"; solids "closer to the viewer will cover more
    # pixels".  Dolly to half the distance: one-pixel points cover about a quarter of what the
    # ray-traced spheres cover.
    cfg = synth.make_config(0, W=96, H=96)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0)
    near = synth.orbit_camera(0.0, 0.0, synth.DIAG)
    pts = (oracle.render_points(sc, near, 96, 96, 1)[..., 3] > 0).sum()
    sph = (oracle.render(sc, near, 96, 96, "bvh")[..., 3] > 0).sum()
    assert sc["N"] * 0.9 <= pts <= sc["N"] and sph > 2.5 * pts
