"""-m gpu: splats_march (the server's volume ray marcher) against the
oracle's marcher, bit for bit, and the whole server -> wire -> client chain on the GPU."""
import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_common import Session, assert_bvh_bit_exact, assert_rgba_close
from paper_2006_14726_b200 import binding as sp

pytestmark = pytest.mark.gpu


def _gpu_march(vol, cam, W, H, tf=None, otf=None):
    n = vol.shape[0]
    dv = torch.from_numpy(np.ascontiguousarray(vol, dtype=np.float32)).cuda()
    color = torch.full((H, W, 4), -7.0, dtype=torch.float32, device="cuda")
    depth = torch.full((H, W), -7.0, dtype=torch.float32, device="cuda")
    sp.splats_march(dv, n, tf if tf is not None else sp.make_transfer(oracle.BASELINE_TENTS), cam, W, H, color, depth)
    torch.cuda.synchronize()
    return color, depth


def _check(vol, cam, W, H, tents=None, **kw):
    tents = oracle.BASELINE_TENTS if tents is None else tents
    color, depth = _gpu_march(vol, cam, W, H, sp.make_transfer(tents, **kw))
    rc, rd = oracle.march(vol, cam, W, H, oracle.make_transfer(tents, **kw))
    np.testing.assert_array_equal(depth.cpu().numpy().view(np.uint32), rd.view(np.uint32))
    np.testing.assert_array_equal(color.cpu().numpy().view(np.uint32), rc.view(np.uint32))
    return color, depth, rc, rd


def test_config0_and_odd_views():
    cfg = synth.make_config(0)
    vol = synth.volume(cfg)
    with Session(256, 256):
        _, _, rc, rd = _check(vol, cfg.src_cams[0], cfg.W, cfg.H)
        assert (rd > 0).sum() > 100
        _check(vol, synth.orbit_camera(33.0, -20.0, 2.0), 97, 61)
        _check(vol, synth.orbit_camera(10.0, 5.0, 0.3), 50, 50)                 # eye inside the cube
        _check(vol, synth.orbit_camera(0.0, 0.0, 30.0), 33, 17)                 # far away: a few pixels
        _check(vol, cfg.src_cams[0], 64, 64, tents=[(0.5, 0.3, (1, 0, 0)), (0.35, 0.8, (0, 1, 0)), (0.7, 0.95, (0, 0, 1)), (0.2, 0.1, (1, 1, 1))],
               half_width=0.1, shade=0.0, depth_alpha=0.8, stop_alpha=0.95)     # four overlapping tents
        away = synth.orbit_camera(0.0).copy(); away[9:12] *= -1
        c, d, _, _ = _check(vol, away, 16, 16)
        assert (d == 0).all()
        with pytest.raises(sp.SplatsError):
            _gpu_march(vol, cfg.src_cams[0], 16, 16, sp.make_transfer(oracle.BASELINE_TENTS, half_width=0.0))


def test_hand_made_volumes():
    with Session(64, 64):
        cam = np.array([0.5, 0.5, 2.5, 1, 0, 0, 0, 1, 0, 0, 0, -1, 0.5], np.float32)
        _check(np.full((16, 16, 16), 0.35, np.float32), cam, 9, 9)
        _check(np.zeros((1, 1, 1), np.float32), cam, 4, 4)
        z = (np.arange(64, dtype=np.float32) + 0.5) / 64
        _check(np.broadcast_to(z[:, None, None], (64, 64, 64)).copy(), cam, 31, 33, tents=[(0.40625, 1.0, (1, 1, 1))], half_width=0.02)
        axis = np.array([0.5, 0.5, 3.0, 1, 0, 0, 0, 1, 0, 0, 0, -1, 1e-3], np.float32)   # near-parallel rays, d_x ~ 0
        _check(np.random.default_rng(0).uniform(0, 1, (8, 8, 8)).astype(np.float32), axis, 5, 5)


def test_config1_full_frame():
    cfg = synth.make_config(1)
    with Session(cfg.W, cfg.H):
        _, _, rc, rd = _check(synth.volume(cfg), cfg.src_cams[0], cfg.W, cfg.H)
        assert (rd > 0).sum() > 10_000


def test_config3_1080p_and_the_whole_chain_on_the_gpu():
    # server: march -> pack; client: update_packed -> render; every stage against the oracle's
    cfg = synth.make_config(3)
    vol = synth.volume(cfg)
    cam = cfg.src_cams[9]
    quant = np.array([0, 0, 0, 1, 1, 1, 0.02], np.float32)
    with Session(cfg.W, cfg.H) as s:
        color, depth, rc, rd = _check(vol, cam, cfg.W, cfg.H)
        samples = torch.empty(cfg.W * cfg.H, dtype=torch.int64, device="cuda")
        colours = torch.empty(cfg.W * cfg.H, dtype=torch.int32, device="cuda")
        count = torch.zeros(1, dtype=torch.int32, device="cuda")
        sp.splats_pack(color, depth, cam, cfg.W, cfg.H, 1.0, quant, samples, colours, count)
        n = int(count.item())
        rs, rcol = oracle.pack(rc, rd, cam, cfg.W, cfg.H, 1.0, quant)
        assert n == len(rs) > 100_000
        np.testing.assert_array_equal(samples[:n].cpu().numpy().view(np.uint64), rs)
        sp.splats_update_packed(samples, colours, n, quant)
        sc = oracle.build_scene_packed(rs, rcol, quant)
        assert_bvh_bit_exact(sc)
        dst = cfg.dst_cams[39]
        got = s.render(dst, cfg.W, cfg.H, first_hit=True)
        assert np.array_equal(got, oracle.render(sc, dst, cfg.W, cfg.H, "bvh", first_hit=True))
        rng = np.random.default_rng(3)
        px = rng.choice(cfg.W * cfg.H, size=100_000, replace=False).astype(np.int64)
        assert_rgba_close(s.render(dst, cfg.W, cfg.H).reshape(-1, 4)[px], oracle.render(sc, dst, cfg.W, cfg.H, "bvh", pixels=px), "chain")
