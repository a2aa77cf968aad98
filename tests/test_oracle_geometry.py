"""Pins for oracle steps O1-O4 (unprojection Eq. 1, radius, validity, Morton).

Each check is against something other than the oracle's own formula: hand-worked
values, geometric invariants evaluated in float64, or a differently-formulated
bit interleave."""
import math

import numpy as np
import pytest

import oracle
import synth

IDENT = np.array([0, 0, 0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 1.0], np.float32)  # eye 0, R=x, U=y, F=-z, tan=1


def test_pixel_ray_hand_worked_2x2():
    # W=H=2, fov 90: pixel centres at ndc (+-0.5, +-0.5); row 0 is the top row.
    d, ln = oracle.pixel_ray(IDENT, 2, 2, 0, 0)
    assert ln == pytest.approx(math.sqrt(1.5), rel=1e-6)
    np.testing.assert_allclose(d, np.array([-0.5, 0.5, -1.0]) / math.sqrt(1.5), rtol=1e-6)
    d, _ = oracle.pixel_ray(IDENT, 2, 2, 1, 1)
    np.testing.assert_allclose(d, np.array([0.5, -0.5, -1.0]) / math.sqrt(1.5), rtol=1e-6)


def test_pixel_ray_aspect_hand_worked_4x2():
    # W=4,H=2: horizontal half-extent = tan * W/H = 2; pixel 0 centre at ndc -0.75 -> u = -1.5
    d, ln = oracle.pixel_ray(IDENT, 4, 2, 0, 1)
    v = np.array([-1.5, -0.5, -1.0])
    np.testing.assert_allclose(d, v / np.linalg.norm(v), rtol=1e-6)
    assert ln == pytest.approx(np.linalg.norm(v), rel=1e-6)


def test_pixel_ray_odd_centre_is_forward():
    cam = synth.orbit_camera(33.0, 12.0)
    d, ln = oracle.pixel_ray(cam, 7, 5, 3, 2)
    np.testing.assert_allclose(d, cam[9:12], atol=2e-7)
    assert ln == pytest.approx(1.0, abs=2e-7)


def test_pixel_ray_unit_and_mirror():
    cam = synth.orbit_camera(10.0, -7.0)
    W, H = 16, 10
    for (x, y) in [(0, 0), (5, 3), (15, 9), (8, 4)]:
        d, _ = oracle.pixel_ray(cam, W, H, x, y)
        assert abs(np.linalg.norm(d.astype(np.float64)) - 1.0) < 2e-7
        dm, _ = oracle.pixel_ray(cam, W, H, W - 1 - x, H - 1 - y)
        # mirrored pixel: components along R and U flip sign, along F stay
        R, U, F = cam[3:6].astype(np.float64), cam[6:9].astype(np.float64), cam[9:12].astype(np.float64)
        assert np.dot(d, R) == pytest.approx(-np.dot(dm, R), abs=1e-6)
        assert np.dot(d, U) == pytest.approx(-np.dot(dm, U), abs=1e-6)
        assert np.dot(d, F) == pytest.approx(np.dot(dm, F), abs=1e-6)


def _project(cam, W, H, c):
    """float64 pinhole projection of point c -> continuous pixel coordinates."""
    cam = cam.astype(np.float64)
    e, R, U, F, tau = cam[0:3], cam[3:6], cam[6:9], cam[9:12], cam[12]
    v = c.astype(np.float64) - e
    z = v @ F
    nx = (v @ R) / z / (tau * W / H)
    ny = (v @ U) / z / tau
    return (nx + 1) * W / 2, (1 - ny) * H / 2, z


def test_unproject_roundtrip_and_distance():
    # Eq. 1: p = o + d t  =>  |p - o| = t and p projects back to its own pixel centre.
    cam = synth.orbit_camera(20.0, 5.0)
    W, H = 48, 27
    rng = np.random.default_rng(1)
    depth = rng.uniform(1.0, 6.0, (H, W)).astype(np.float32)
    sphere, valid, n = oracle.unproject(depth, cam, W, H, 1.0)
    assert n == W * H and valid.all()
    for p in rng.integers(0, W * H, 200):
        x, y = p % W, p // W
        c = sphere[p, :3]
        assert np.linalg.norm(c.astype(np.float64) - cam[:3]) == pytest.approx(depth.reshape(-1)[p], rel=3e-7)
        px, py, _ = _project(cam, W, H, c)
        assert px == pytest.approx(x + 0.5, abs=1e-3)
        assert py == pytest.approx(y + 0.5, abs=1e-3)


def test_radius_is_half_diagonal_of_pixel_footprint():
    # north_star: "radius is its one-pixel footprint at its depth".  Geometric route: the
    # footprint side at view depth z is the distance between the unprojections of two
    # horizontally adjacent pixel centres at that same z; r = side * sqrt(2)/2 * r_scale.
    cam = synth.orbit_camera(-15.0, 8.0)
    W, H = 64, 36
    cam64 = cam.astype(np.float64)
    for r_scale in (1.0, 2.0, 0.5):
        depth = np.full((H, W), 3.0, np.float32)
        sphere, _, _ = oracle.unproject(depth, cam, W, H, r_scale)
        for (x, y) in [(10, 10), (40, 30), (63, 0)]:
            p = y * W + x
            _, _, z = _project(cam, W, H, sphere[p, :3])
            side = z * 2 * cam64[12] / H
            assert sphere[p, 3] == pytest.approx(r_scale * side * math.sqrt(0.5), rel=2e-6)
            # and via a neighbour's ray at the same view depth
            q = p - 1 if x else p + 1
            d0 = sphere[p, :3].astype(np.float64) - cam64[:3]
            d1 = sphere[q, :3].astype(np.float64) - cam64[:3]
            d1 *= (d0 @ cam64[9:12]) / (d1 @ cam64[9:12])
            assert np.linalg.norm(d0 - d1) == pytest.approx(side, rel=1e-4)


def test_radius_monotone_in_depth():
    # "solids that are closer to the viewer will cover more pixels" -- with a
    # footprint radius that grows linearly with view depth the *projected* size is constant.
    cam = synth.orbit_camera(0.0)
    W, H = 8, 8
    rs = []
    for t in (1.0, 2.0, 4.0, 8.0):
        sphere, _, _ = oracle.unproject(np.full((H, W), t, np.float32), cam, W, H, 1.0)
        rs.append(sphere[27, 3])
    assert rs[0] < rs[1] < rs[2] < rs[3]
    assert rs[3] / rs[0] == pytest.approx(8.0, rel=1e-6)


def test_invalid_depths_dropped():
    cam = synth.orbit_camera(0.0)
    depth = np.array([[1.0, 0.0, -2.0, np.nan], [np.inf, -np.inf, 1e-30, 3.0]], np.float32)
    sphere, valid, n = oracle.unproject(depth, cam, 4, 2, 1.0)
    assert valid.tolist() == [1, 0, 0, 0, 0, 0, 1, 1]
    assert n == 3
    assert np.all(sphere[valid == 0] == 0)


# ----------------------------------------------------------------------------- Morton
def _interleave_strings(qx, qy, qz):
    bx, by, bz = format(qx, "021b"), format(qy, "021b"), format(qz, "021b")
    return int("".join(a + b + c for a, b, c in zip(bx, by, bz)), 2)


def test_morton_corners_and_axis_slots():
    lo = np.zeros(3, np.float32)
    hi = np.ones(3, np.float32)
    assert oracle.morton_point(lo, lo, hi) == 0
    assert oracle.morton_point(hi, lo, hi) == 2 ** 63 - 1
    h = 2.0 ** -21
    assert oracle.morton_point([1.5 * h, 0, 0], lo, hi) == 4   # bit 0 of q_x -> code bit 2
    assert oracle.morton_point([0, 1.5 * h, 0], lo, hi) == 2   # q_y -> bit 1
    assert oracle.morton_point([0, 0, 1.5 * h], lo, hi) == 1   # q_z -> bit 0
    assert oracle.morton_point([1, 0, 0], lo, hi) == 0x4924924924924924
    assert oracle.morton_point([0, 1, 0], lo, hi) == 0x2492492492492492
    assert oracle.morton_point([0, 0, 1], lo, hi) == 0x1249249249249249
    assert oracle.morton_point([0.5, 0.5, 0.5], lo, hi) == 7 << 60


def test_morton_vs_string_interleave():
    rng = np.random.default_rng(7)
    lo = np.array([-1.0, 2.0, 0.25], np.float32)
    hi = np.array([3.0, 2.5, 8.25], np.float32)   # power-of-two extents: quantisation is exact
    for _ in range(300):
        q = rng.integers(0, 2 ** 21, 3)
        c = lo.astype(np.float64) + (hi - lo).astype(np.float64) * (q + 0.5) / 2.0 ** 21
        c32 = c.astype(np.float32)
        # keep only points whose float32 rounding did not leave the cell
        qq = np.floor((c32.astype(np.float64) - lo) / (hi - lo) * 2 ** 21).astype(np.int64)
        assert oracle.morton_point(c32, lo, hi) == _interleave_strings(int(qq[0]), int(qq[1]), int(qq[2]))


def test_morton_zero_extent_axis():
    lo = np.array([0.0, 5.0, 0.0], np.float32)
    hi = np.array([1.0, 5.0, 1.0], np.float32)
    code = oracle.morton_point([1.0, 5.0, 1.0], lo, hi)
    assert code == _interleave_strings(2 ** 21 - 1, 0, 2 ** 21 - 1)


def test_bounds_are_of_centres_and_codes_span_range():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
    v = sc["valid"] == 1
    np.testing.assert_array_equal(sc["lo"], sc["sphere"][v, :3].min(axis=0))
    np.testing.assert_array_equal(sc["hi"], sc["sphere"][v, :3].max(axis=0))
    # the extreme centres quantise to 0 / 2^21-1 on their axis
    for k, shift in ((0, 2), (1, 1), (2, 0)):
        axis_bits = [(int(c) >> shift) & 0x1249249249249249 for c in sc["codes"]]
        assert min(axis_bits) == 0
        assert max(axis_bits) == 0x1249249249249249
    assert sc["ids"].tolist() == np.nonzero(v)[0].tolist()
