"""Pins for the server-side ray marcher of the oracle (
recipe = BASELINE.json's server pass): closed forms on hand-made volumes and the independent
float64 generator in synth/ (written before, sharing no code)."""
import numpy as np
import pytest

import oracle
import synth

# eye on the +z axis of the unit cube's centre, looking down -z
def _cam(dist, tan=0.5):
    return np.array([0.5, 0.5, 0.5 + dist, 1, 0, 0, 0, 1, 0, 0, 0, -1, tan], np.float32)


ONE_TENT = oracle.make_transfer([(0.35, 0.8, (1.0, 0.5, 0.25))], shade=0.0)


def test_empty_volume_and_rays_that_miss_the_cube():
    vol = np.zeros((8, 8, 8), np.float32)
    c, d = oracle.march(vol, _cam(3.0), 9, 7)
    assert np.all(c == 0) and np.all(d == 0)
    full = np.full((8, 8, 8), 0.35, np.float32)
    c, d = oracle.march(full, _cam(3.0, tan=1.0), 9, 9, ONE_TENT)     # wide view: the corner rays pass beside the cube
    assert d[4, 4] > 0 and d[0, 0] == 0 and np.all(c[0, 0] == 0)
    away = _cam(3.0); away[9:12] = (0, 0, 1)                            # looking away
    c, d = oracle.march(full, away, 5, 5, ONE_TENT)
    assert np.all(d == 0) and np.all(c == 0)


def test_uniform_volume_closed_form_on_the_central_ray():
    # density 0.35 everywhere = the tent's peak: every sample has alpha 0.8.  Central ray enters the
    # cube at t0 = dist - 0.5; samples at t0 + (s + 1/2) * step, step = 0.5 / n.
    # A_k = 1 - 0.2^k: 0.8 >= 0.5 at the first sample -> depth = t0 + step / 2;
    # 0.2^4 = 0.0016 > 0.001 >= 0.2^5 -> the march stops after 5 samples, A = 1 - 0.2^5
    n = 16
    vol = np.full((n, n, n), 0.35, np.float32)
    c, d = oracle.march(vol, _cam(2.0), 1, 1, ONE_TENT)
    step = 0.5 / n
    assert d[0, 0] == pytest.approx(1.5 + step / 2, abs=1e-6)
    A = 1 - 0.2 ** 5
    assert c[0, 0, 3] == pytest.approx(A, abs=1e-6)
    np.testing.assert_allclose(c[0, 0, :3], np.array([1.0, 0.5, 0.25]) * A, atol=1e-6)   # premultiplied
    # a higher depth threshold is reached one sample later: 0.96 >= 0.9 at s = 1
    tf = oracle.make_transfer([(0.35, 0.8, (1.0, 0.5, 0.25))], shade=0.0, depth_alpha=0.9)
    _, d2 = oracle.march(vol, _cam(2.0), 1, 1, tf)
    assert d2[0, 0] == pytest.approx(1.5 + 1.5 * step, abs=1e-6)
    # position shading: colour * (1 - shade + shade * P); on the central ray P = (0.5, 0.5, z)
    tf = oracle.make_transfer([(0.35, 0.8, (1.0, 1.0, 1.0))], shade=0.45, stop_alpha=0.5)     # one sample only
    c3, _ = oracle.march(vol, _cam(2.0), 1, 1, tf)
    z = 1.0 - step / 2
    np.testing.assert_allclose(c3[0, 0], [0.8 * 0.775, 0.8 * 0.775, 0.8 * (0.55 + 0.45 * z), 0.8], atol=1e-6)


def test_trilinear_reproduces_a_linear_ramp_and_depth_finds_the_iso_surface():
    # V(i, j, k) = z of the voxel centre: trilinear interpolation of a linear function is exact
    # inside the grid, so the density along the central ray is z = 2.5 - t; a narrow tent at iso
    # 0.40625 with alpha 1 at the peak: the first sample with |z - iso| < hw that carries the
    # accumulated alpha over 0.5 must lie within one step of the iso surface
    n = 64
    z = (np.arange(n, dtype=np.float32) + 0.5) / n
    vol = np.broadcast_to(z[:, None, None], (n, n, n)).copy()
    tf = oracle.make_transfer([(0.40625, 1.0, (1, 1, 1))], half_width=0.02, shade=0.0)
    c, d = oracle.march(vol, _cam(2.0), 1, 1, tf)
    t_iso = 2.5 - 0.40625
    assert abs(d[0, 0] - t_iso) <= 0.02 + 0.5 / n
    # the same march written out in float64: z = 2.5 - t, w = 1 - |z - iso| / hw
    step, A, t_half = 0.5 / n, 0.0, 0.0
    for s_ in range(2 * n):
        t = 1.5 + (s_ + 0.5) * step
        w = max(0.0, 1.0 - abs((2.5 - t) - 0.40625) / 0.02)
        A += (1 - A) * w
        if t_half == 0.0 and A >= 0.5:
            t_half = t
    assert 0.9 < A < 0.999 and c[0, 0, 3] == pytest.approx(A, abs=2e-5) and d[0, 0] == pytest.approx(t_half, abs=1e-6)
    # nearest-voxel values at voxel centres: a ray along a row of voxel centres sees V exactly
    rng = np.random.default_rng(0)
    vol = rng.uniform(0.5, 0.6, size=(4, 4, 4)).astype(np.float32)
    vol[:, 1, 2] = 0.35                                   # all voxels with x index 2, y index 1 (z any)
    eye = np.array([(2 + 0.5) / 4, (1 + 0.5) / 4, 3.0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 0.5], np.float32)
    c, d = oracle.march(vol, eye, 1, 1, ONE_TENT)
    assert d[0, 0] == pytest.approx(2.0 + 0.0625, abs=1e-6) and c[0, 0, 3] == pytest.approx(1 - 0.2 ** 5, abs=1e-6)


@pytest.mark.parametrize("ci,build", [(0, 0), (1, 0), (3, 9)])
def test_against_the_float64_generator(ci, build):
    # synth/gen.cpp marches the same recipe in double precision with its own code: colours must
    # agree to float32 accuracy, the valid set and the depths up to a few threshold flips
    cfg = synth.make_config(ci, W=160, H=90) if ci == 3 else synth.make_config(ci)
    vol = synth.volume(cfg)
    ref_c, ref_d = synth.source_frame(cfg, build)
    c, d = oracle.march(vol, cfg.src_cams[build], cfg.W, cfg.H)
    assert (ref_d > 0).sum() > 100
    flips = ((d > 0) != (ref_d > 0)).sum() + (np.abs(d - ref_d) > 1e-5).sum()
    assert flips <= max(2, 1e-3 * (ref_d > 0).sum())
    assert np.abs(c - ref_c).max() < 2e-3
    assert (np.abs(c - ref_c).max(axis=2) > 2e-4).mean() < 1e-3
