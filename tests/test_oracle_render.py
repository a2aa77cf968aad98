"""Pins for oracle steps O8-O9: sphere entry t, compositing, identity reprojection,
BVH-walk == brute force (BASELINE.json north_star lists exactly these four)."""
import math

import numpy as np
import pytest

import oracle
import synth

O = np.zeros(3, np.float32)
DZ = np.array([0, 0, -1], np.float32)


def test_single_sphere_on_axis_exact():
    # closed form t = z0 - r (values exactly representable)
    hit, t = oracle.ray_sphere(O, DZ, [0, 0, -4, 0.5])
    assert hit and t == 3.5
    hit, t = oracle.ray_sphere([1, 2, 3], [1, 0, 0], [9, 2, 3, 2])
    assert hit and t == 6.0


def test_single_sphere_off_axis_closed_form():
    # t = b - sqrt(r^2 - l^2): 3-4-5 triangle, l = 0.3, r = 0.5 -> sqrt = 0.4
    hit, t = oracle.ray_sphere(O, DZ, [0.3, 0, -4, 0.5])
    assert hit and t == pytest.approx(3.6, abs=1e-6)
    rng = np.random.default_rng(0)
    for _ in range(200):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        b = rng.uniform(2, 5); r = rng.uniform(1e-3, 4e-3)
        perp = np.cross(d, rng.normal(size=3)); perp /= np.linalg.norm(perp)
        l = rng.uniform(0, 0.95) * r
        c = b * d + l * perp
        hit, t = oracle.ray_sphere(O, d.astype(np.float32), [*c, r])
        assert hit
        assert t == pytest.approx(b - math.sqrt(r * r - l * l), abs=3e-6)


def test_sphere_misses():
    assert not oracle.ray_sphere(O, DZ, [0.5, 0, -4, 0.5])[0]      # tangent: disc == 0 -> miss
    assert not oracle.ray_sphere(O, DZ, [0.6, 0, -4, 0.5])[0]      # passes beside
    assert not oracle.ray_sphere(O, DZ, [0, 0, 4, 0.5])[0]         # behind the eye
    assert not oracle.ray_sphere(O, DZ, [0, 0, -0.2, 0.5])[0]      # eye inside: entry t < 0
    hit, t = oracle.ray_sphere(O, DZ, [0, 0, -0.5, 0.5])           # eye on the surface: t = +0 accepted
    assert hit and t == 0.0


@pytest.mark.parametrize("alpha,n_expected", [(0.05, 90), (0.5, 7), (0.25, 17), (0.995, 1)])
def test_alpha_stack_closed_form(alpha, n_expected):
    # n equal splats of opacity alpha, premultiplied colour alpha*rgb:
    # A_n = 1-(1-alpha)^n, C = rgb*A_n, stops at n* = ceil(ln 0.01 / ln(1-alpha))
    assert n_expected == math.ceil(math.log(0.01) / math.log(1 - alpha) - 1e-12)
    n = 200
    rgb = np.array([0.2, 0.5, 0.9])
    rgba = np.tile(np.concatenate([rgb * alpha, [alpha]]), (n, 1)).astype(np.float32)
    t = np.linspace(5.0, 1.0, n).astype(np.float32)       # given back to front: must be sorted
    out, used = oracle.composite(t, np.arange(n), rgba)
    assert used == n_expected
    A = 1 - (1 - alpha) ** n_expected
    assert out[3] == pytest.approx(A, abs=2e-6)
    np.testing.assert_allclose(out[:3], rgb * A, atol=2e-6)
    assert out[3] >= 0.99


def test_half_alpha_exact_binary_fractions():
    rgba = np.tile(np.array([0.5, 0.25, 0.0, 0.5], np.float32), (10, 1))
    out, used = oracle.composite(np.arange(10, dtype=np.float32), np.arange(10), rgba)
    assert used == 7 and out[3] == 1 - 2.0 ** -7 and out[0] == out[3] and out[1] == out[3] / 2


def test_composite_orders_by_t_then_id():
    red = [0.6, 0, 0, 0.6]
    blue = [0, 0, 0.6, 0.6]
    out, _ = oracle.composite([2.0, 1.0], [0, 1], [red, blue])      # blue is nearer
    np.testing.assert_allclose(out, [0.24, 0, 0.6, 0.84], atol=1e-6)
    out, _ = oracle.composite([1.0, 1.0], [7, 3], [red, blue])      # equal t: lower id (blue) first
    np.testing.assert_allclose(out, [0.24, 0, 0.6, 0.84], atol=1e-6)
    out, _ = oracle.composite([1.0, 1.0], [3, 7], [red, blue])      # red first
    np.testing.assert_allclose(out, [0.6, 0, 0.24, 0.84], atol=1e-6)


def test_single_hit_reproduces_colour_bit_exactly():
    col = np.array([[0.123456789, 0.3333333, 0.9876543, 0.7]], np.float32)
    out, used = oracle.composite([1.0], [0], col)
    assert used == 1 and np.array_equal(out, col[0])


def _scene(kind):
    if kind == "config0":
        cfg = synth.make_config(0)
        color, depth = synth.source_frame(cfg, 0)
        return color, depth, cfg.src_cams[0], cfg.W, cfg.H
    if kind == "wide":
        color, depth, cam = synth.random_frame(48, 27, 11, 0.6)
        return color, depth, cam, 48, 27
    color, depth, cam = synth.random_frame(33, 31, 12, 0.9)
    return color, depth, cam, 33, 31


@pytest.mark.parametrize("kind", ["config0", "wide", "square"])
@pytest.mark.parametrize("r_scale", [1.0, 0.5])
def test_identity_camera_reproduces_source(kind, r_scale):
    # SURVEY.md sec. 8(c) closed form (iii): dst == src camera, r_scale <= 1 => every ray hits
    # only its own splat => out == color bit-exactly at valid pixels, 0 elsewhere.
    color, depth, cam, W, H = _scene(kind)
    sc = oracle.build_scene(color, depth, cam, W, H, r_scale)
    for mode in ("brute", "bvh"):
        out, used = oracle.render(sc, cam, W, H, mode, return_hits=True)
        v = (sc["valid"] == 1).reshape(H, W)
        assert np.array_equal(out[v], color[v])
        assert np.all(out[~v] == 0)
        assert np.all(used[v] == 1) and np.all(used[~v] == 0)


@pytest.mark.parametrize("kind,r_scale", [("config0", 1.0), ("wide", 2.0), ("square", 3.0)])
def test_bvh_walk_equals_brute_force(kind, r_scale):
    color, depth, cam, W, H = _scene(kind)
    sc = oracle.build_scene(color, depth, cam, W, H, r_scale)
    cams = [synth.orbit_camera(5.0), synth.orbit_camera(-20.0, 10.0, 2.5), synth.orbit_camera(15.0, shift_right=0.4)]
    for dst in cams:
        for (W2, H2) in ((W, H), (40, 30)):
            a, ua = oracle.render(sc, dst, W2, H2, "brute", return_hits=True)
            b, ub = oracle.render(sc, dst, W2, H2, "bvh", return_hits=True)
            assert np.array_equal(a, b) and np.array_equal(ua, ub)
            assert (a[..., 3] > 0).any()


def test_low_alpha_stack_through_renderer():
    # 100 coaxial splats of alpha 0.05 along the central ray: needs 90 hits (closed form (ii)).
    W = H = 1
    cam = synth.orbit_camera(0.0)
    n = 100
    sphere = np.zeros((n, 4), np.float32)
    e, F = cam[:3].astype(np.float64), cam[9:12].astype(np.float64)
    for i in range(n):
        sphere[i, :3] = e + F * (2.0 + 0.01 * i)
        sphere[i, 3] = 0.004
    rgba = np.tile(np.array([0.01, 0.02, 0.03, 0.05], np.float32), (n, 1))
    sc = dict(N=n, sphere_sorted=sphere, rgba_sorted=rgba, sorted_ids=np.arange(n, dtype=np.uint32))
    out, used = oracle.render(sc, cam, W, H, "brute", return_hits=True)
    assert used[0, 0] == 90
    assert out[0, 0, 3] == pytest.approx(1 - 0.95 ** 90, abs=2e-6)


def test_empty_scene_renders_zeros():
    depth = np.zeros((4, 4), np.float32)
    color = np.ones((4, 4, 4), np.float32)
    cam = synth.orbit_camera(0.0)
    sc = oracle.build_scene(color, depth, cam, 4, 4, 1.0)
    assert sc["N"] == 0
    for mode in ("brute", "bvh"):
        assert np.all(oracle.render(sc, cam, 4, 4, mode) == 0)


def test_single_splat_scene():
    depth = np.zeros((3, 3), np.float32)
    depth[1, 1] = 2.0
    color = np.full((3, 3, 4), 0.5, np.float32)
    cam = synth.orbit_camera(0.0)
    sc = oracle.build_scene(color, depth, cam, 3, 3, 1.0)
    assert sc["N"] == 1 and sc["parents"].tolist() == [-1]
    for mode in ("brute", "bvh"):
        out = oracle.render(sc, cam, 3, 3, mode)
        assert np.array_equal(out[1, 1], color[1, 1]) and out[..., 3].sum() == 0.5


# ------------------------------------------------------------------ first-hit query
def _coaxial(ts, ids, cols, radius=0.004):
    """Spheres centred on the central ray of a 1x1 image at distances ts (array order as given)."""
    cam = synth.orbit_camera(0.0)
    e, F = cam[:3].astype(np.float64), cam[9:12].astype(np.float64)
    sphere = np.array([[*(e + F * t), radius] for t in ts], np.float32)
    return cam, dict(N=len(ts), sphere_sorted=sphere, rgba_sorted=np.asarray(cols, np.float32),
                     sorted_ids=np.asarray(ids, np.uint32))


def test_first_hit_takes_the_nearest_sphere_and_copies_its_colour():
    # "a simple first-hit ray tracing query ... no shading other than the constant
    # sample color": whatever the array order, the nearest entry point wins and nothing behind
    # it contributes, even when it is almost transparent.
    cols = [[0.6, 0.0, 0.0, 0.6], [0.0, 0.02, 0.0, 0.05], [0.0, 0.0, 0.9, 1.0]]
    for order in ([0, 1, 2], [2, 1, 0], [1, 2, 0]):
        ts = [3.0, 2.0, 4.0]
        cam, sc = _coaxial([ts[i] for i in order], order, [cols[i] for i in order])
        for mode in ("brute",):
            out, used = oracle.render(sc, cam, 1, 1, mode, return_hits=True, first_hit=True)
            assert used[0, 0] == 1
            assert np.array_equal(out[0, 0], np.asarray(cols[1], np.float32))
        # compositing the same stack gives something else: all three contribute
        allhit = oracle.render(sc, cam, 1, 1, "brute")
        assert allhit[0, 0, 3] > 0.99 and allhit[0, 0, 2] > 0.3


def test_first_hit_equal_t_is_decided_by_id():
    cols = [[0.5, 0, 0, 0.5], [0, 0.5, 0, 0.5]]
    for ids, want in (([7, 3], 1), ([3, 7], 0)):
        cam, sc = _coaxial([2.5, 2.5], ids, cols)
        out = oracle.render(sc, cam, 1, 1, "brute", first_hit=True)
        assert np.array_equal(out[0, 0], np.asarray(cols[want], np.float32))


@pytest.mark.parametrize("kind,r_scale", [("config0", 1.0), ("wide", 2.0), ("square", 3.0)])
def test_first_hit_equals_compositing_of_opaque_splats_and_walk_equals_brute(kind, r_scale):
    # With every alpha = 1 the first composited hit already reaches A >= 0.99, so the all-hit
    # renderer degenerates to the first-hit query: the two independent code paths must agree.
    color, depth, cam, W, H = _scene(kind)
    opaque = color.copy()
    opaque[..., 3] = 1.0
    sc = oracle.build_scene(opaque, depth, cam, W, H, r_scale)
    sc_t = oracle.build_scene(color, depth, cam, W, H, r_scale)   # translucent colours, same geometry
    for dst in (synth.orbit_camera(5.0), synth.orbit_camera(-20.0, 10.0, 2.5)):
        a = oracle.render(sc, dst, W, H, "brute")
        f, used = oracle.render(sc, dst, W, H, "brute", first_hit=True, return_hits=True)
        assert np.array_equal(a, f) and (a[..., 3] > 0).any()
        assert set(np.unique(used)) <= {0, 1}
        fb = oracle.render(sc_t, dst, W, H, "brute", first_hit=True)
        fw = oracle.render(sc_t, dst, W, H, "bvh", first_hit=True)
        assert np.array_equal(fb, fw)
        # same geometry => same winner: the translucent image is the opaque one with the alpha swapped in
        hit = f[..., 3] > 0
        assert np.array_equal(fb[..., 3] > 0, hit)


def test_first_hit_identity_camera_reproduces_source():
    color, depth, cam, W, H = _scene("config0")
    sc = oracle.build_scene(color, depth, cam, W, H, 1.0)
    out = oracle.render(sc, cam, W, H, "bvh", first_hit=True)
    v = (sc["valid"] == 1).reshape(H, W)
    assert np.array_equal(out[v], color[v]) and np.all(out[~v] == 0)
