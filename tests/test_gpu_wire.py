"""-m gpu: the paper's wire format -- splats_pack
(server: Eq. 1 + radius + quantise + compact) and splats_update_packed (client: BVH from the
received samples) against the oracle, bit for bit."""
import math

import numpy as np
import pytest
import torch

import oracle
import synth
from gpu_common import Session, assert_bvh_bit_exact, assert_rgba_close
from paper_2006_14726_b200 import binding as sp

pytestmark = pytest.mark.gpu

BOX = np.array([0, 0, 0, 1, 1, 1, 0.05], np.float32)


def _gpu_pack(color, depth, cam, W, H, r_scale, quant):
    dc = torch.from_numpy(np.ascontiguousarray(color, dtype=np.float32)).cuda()
    dd = torch.from_numpy(np.ascontiguousarray(depth, dtype=np.float32)).cuda()
    samples = torch.full((W * H,), -1, dtype=torch.int64, device="cuda")
    colours = torch.full((W * H,), -1, dtype=torch.int32, device="cuda")
    count = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    sp.splats_pack(dc, dd, cam, W, H, r_scale, quant, samples, colours, count)
    torch.cuda.synchronize()
    n = int(count.item())
    return samples, colours, n


def _check_pack(color, depth, cam, W, H, r_scale, quant, radius=(0, 0.0)):
    sp.splats_set_radius(*radius)
    samples, colours, n = _gpu_pack(color, depth, cam, W, H, r_scale, quant)
    rs, rc = oracle.pack(color, depth, cam, W, H, r_scale, quant, radius[0], radius[1])
    assert n == len(rs)
    np.testing.assert_array_equal(samples[:n].cpu().numpy().view(np.uint64), rs)
    np.testing.assert_array_equal(colours[:n].cpu().numpy().view(np.uint32), rc)
    assert (samples[n:] == -1).all() and (colours[n:] == -1).all()      # nothing written past the count
    return samples, colours, n, rs, rc


def _check_packed_scene(s, samples, colours, n, rs, rc, quant, cams, sizes, mode="bvh"):
    sc = oracle.build_scene_packed(rs, rc, quant)
    sp.splats_update_packed(samples, colours, n, quant)
    assert_bvh_bit_exact(sc)
    for cam, (W2, H2) in zip(cams, sizes):
        got = s.render(cam, W2, H2)
        assert_rgba_close(got, oracle.render(sc, cam, W2, H2, mode), "all-hit")
        gf = s.render(cam, W2, H2, first_hit=True)
        assert np.array_equal(gf, oracle.render(sc, cam, W2, H2, mode, first_hit=True))
    return sc


def test_config0_pack_and_build_from_packed():
    cfg = synth.make_config(0)
    color, depth = synth.source_frame(cfg, 0)
    with Session(cfg.W, cfg.H) as s:
        samples, colours, n, rs, rc = _check_pack(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, BOX)
        _check_packed_scene(s, samples, colours, n, rs, rc, BOX, [cfg.dst_cams[0], cfg.src_cams[0]], [(64, 64), (48, 32)], "brute")


@pytest.mark.parametrize("W,H,fill,radius", [(97, 61, 0.7, (0, 0.0)), (130, 50, 0.3, (1, 0.01)), (33, 200, 1.0, (2, 0.25)),
                                               (2049, 3, 0.5, (2, 0.0))])
def test_pack_ragged_frames_and_radius_modes(W, H, fill, radius):
    color, depth, cam = synth.random_frame(W, H, seed=W + H, fill=fill)
    color[::7, ::5, 3] = 0.0                       # alpha 0: dropped by the opacity radius with floor 0
    quant = np.array([-3, -3, -3, 4, 4, 4, 0.02], np.float32)
    with Session(W, H) as s:
        samples, colours, n, rs, rc = _check_pack(color, depth, cam, W, H, 1.5, quant, radius)
        if radius == (2, 0.0):
            assert n < int((depth > 0).sum())
        _check_packed_scene(s, samples, colours, n, rs, rc, quant, [synth.orbit_camera(6.0)], [(80, 45)])
        sp.splats_set_radius(0, 0.0)


def test_received_buffer_with_dropped_words_and_tiny_counts():
    quant = BOX
    rng = np.random.default_rng(1)
    words = rng.integers(0, 2 ** 63, size=3000, dtype=np.int64).astype(np.uint64) | np.uint64(1 << 48)
    words[::11] &= np.uint64((1 << 48) - 1)        # radius field 0: not a legal sample, dropped
    words[5] = words[6] = words[7]                 # duplicates: equal codes, order by id
    cols = rng.integers(0, 2 ** 32, size=3000, dtype=np.int64).astype(np.uint32)
    with Session(64, 64) as s:
        for n in (3000, 2, 1, 0):
            ws = torch.from_numpy(words[:max(n, 1)].view(np.int64).copy()).cuda()
            cs = torch.from_numpy(cols[:max(n, 1)].view(np.int32).copy()).cuda()
            first = 1 if n == 1 else 0             # words[0] has radius field 0: use words[1] for n = 1
            if n == 1:
                ws, cs = ws.clone(), cs.clone()
                ws[0] = int(words[1].view(np.int64)); cs[0] = int(cols[1].view(np.int32))
            rs = words[first:first + n] if n == 1 else words[:n]
            rc = cols[first:first + n] if n == 1 else cols[:n]
            sc = _check_packed_scene(s, ws, cs, n, rs, rc, quant, [synth.orbit_camera(0.0, 0.0, 3.0)], [(32, 32)], "brute")
            assert sc["N"] == int(((rs >> np.uint64(48)) != 0).sum())
        big_w = torch.zeros(64 * 64 + 1, dtype=torch.int64, device="cuda")
        big_c = torch.zeros(64 * 64 + 1, dtype=torch.int32, device="cuda")
        with pytest.raises(sp.SplatsError):
            sp.splats_update_packed(big_w, big_c, 64 * 64 + 1, quant)       # beyond the capacity
        with pytest.raises(sp.SplatsError):
            sp.splats_update_packed(ws, cs, 1, [0, 0, 0, 1, 0, 1, 0.1])     # hi <= lo
        with pytest.raises(sp.SplatsError):
            sp.splats_update_packed(ws, cs, 1, [0, 0, 0, 1, 1, 1, 0.0])     # r_max <= 0


def test_all_invalid_frame_packs_to_nothing():
    depth = np.zeros((20, 30), np.float32)
    color = np.ones((20, 30, 4), np.float32)
    with Session(30, 20):
        samples, colours, n = _gpu_pack(color, depth, synth.orbit_camera(0.0), 30, 20, 1.0, BOX)
        assert n == 0 and (samples == -1).all()


def test_config2_paper_shape_constant_radius_round_trip():
    # 1024 x 1024 as in the paper's Table 1, constant radius of half a voxel's
    # diagonal: server packs, client builds from the packed buffer and renders.
    cfg = synth.make_config(2)
    color, depth = synth.source_frame(cfg, 0)
    half_diag = math.sqrt(3.0) / cfg.vol_n / 2
    quant = np.array([0, 0, 0, 1, 1, 1, 2 * half_diag], np.float32)
    with Session(cfg.W, cfg.H) as s:
        samples, colours, n, rs, rc = _check_pack(color, depth, cfg.src_cams[0], cfg.W, cfg.H, 1.0, quant, (1, half_diag))
        assert n == int((depth > 0).sum()) > 50_000
        sc = oracle.build_scene_packed(rs, rc, quant)
        sp.splats_update_packed(samples, colours, n, quant)
        assert_bvh_bit_exact(sc)
        cam = cfg.dst_cams[9]
        got = s.render(cam, cfg.W, cfg.H, first_hit=True)
        assert np.array_equal(got, oracle.render(sc, cam, cfg.W, cfg.H, "bvh", first_hit=True))
        rng = np.random.default_rng(0)
        px = rng.choice(cfg.W * cfg.H, size=100_000, replace=False).astype(np.int64)
        assert_rgba_close(s.render(cam, cfg.W, cfg.H).reshape(-1, 4)[px], oracle.render(sc, cam, cfg.W, cfg.H, "bvh", pixels=px), "all-hit")
        sp.splats_set_radius(0, 0.0)


def test_packed_host_entry_point_pipelined():
    # several received frames in flight through splats_update_packed_host + splats_render_host_rgba8
    cfg = synth.make_config(1)
    quant = BOX
    frames = []
    for b, (W, H) in enumerate(((512, 512), (300, 200), (512, 512), (64, 64))):
        color, depth, cam = synth.random_frame(W, H, seed=40 + b, fill=0.5) if b % 2 else (*synth.source_frame(cfg, 0), cfg.src_cams[0])
        rs, rc = oracle.pack(color, depth, cam, W, H, 1.0, quant)
        frames.append((rs, rc, torch.from_numpy(rs.view(np.int64).copy()).pin_memory(), torch.from_numpy(rc.view(np.int32).copy()).pin_memory()))
    dst = cfg.dst_cams[1]
    with Session(512, 512):
        outs = []
        for rs, rc, hs, hc in frames:
            sp.splats_update_packed_host(hs, hc, len(rs), quant)
            o = torch.zeros((120, 160), dtype=torch.int32).pin_memory()
            sp.splats_render_host_rgba8(dst, 160, 120, o)
            outs.append(o)
        sp.splats_synchronize()
        for (rs, rc, _, _), o in zip(frames, outs):
            sc = oracle.build_scene_packed(rs, rc, quant)
            want = oracle.quantise_image(oracle.render(sc, dst, 160, 120, "bvh"))
            np.testing.assert_array_equal(o.numpy().view(np.uint32), want)
        assert_bvh_bit_exact(oracle.build_scene_packed(frames[-1][0], frames[-1][1], quant))
