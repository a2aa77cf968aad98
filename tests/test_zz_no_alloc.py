"""-m gpu, collected last on purpose (the suite runs with pytest -x): splats_pack_noalloc -- the entry point
that allocates nothing (its scratch is a static __device__ array of the library, include/splats.h) -- against
the existing splats_pack on the same inputs, two calls in a row.  Packed words, colours and counts are integers:
compared for equality, as tests/test_gpu_wire.py does for splats_pack against the oracle."""
import numpy as np
import pytest
import torch

import synth
from paper_2006_14726_b200 import binding as sp

pytestmark = pytest.mark.gpu

QUANT = [0.0, 0.0, 0.0, 1.0, 1.0, 1.0, 0.05]


def _buffers(P):
    dev = torch.device("cuda", torch.cuda.current_device())
    return (torch.full((P,), -1, dtype=torch.int64, device=dev), torch.full((P,), -1, dtype=torch.int32, device=dev),
            torch.full((1,), -1, dtype=torch.int32, device=dev))


def _pack(fn, color, depth, cam, W, H, r_scale, **kw):
    dc, dd = torch.from_numpy(color).cuda(), torch.from_numpy(depth).cuda()
    samples, colors, count = _buffers(W * H)
    fn(dc, dd, cam, W, H, r_scale, QUANT, samples, colors, count, **kw)
    torch.cuda.synchronize()
    n = int(count.item())
    # everything, including the untouched tail (nothing is written past the count)
    return n, samples.cpu().numpy(), colors.cpu().numpy()


def test_pack_noalloc_matches_splats_pack_on_two_calls_in_a_row():
    cfg = synth.make_config(1)                       # 512 x 512 frame of a 128^3 volume
    colA, depA = synth.source_frame(cfg, 0)
    camA, WA, HA = cfg.src_cams[0], cfg.W, cfg.H
    colB, depB, camB = synth.random_frame(203, 97, seed=11, fill=0.7)   # smaller, ragged: the array keeps A's counts beyond B's tiles
    WB, HB = 203, 97

    # the existing path needs a context (its scratch is context memory) ...
    sp.splats_create(max(WA, WB), max(HA, HB))
    try:
        wantA = _pack(sp.splats_pack, colA, depA, camA, WA, HA, cfg.r_scale)
        wantB = _pack(sp.splats_pack, colB, depB, camB, WB, HB, 1.5)
        sp.splats_set_radius(sp.RADIUS_CONSTANT, 0.004)
        wantC = _pack(sp.splats_pack, colB, depB, camB, WB, HB, 1.5)
        sp.splats_set_radius(sp.RADIUS_FOOTPRINT, 0.0)
        # ... the new one does not: first call while the context exists,
        sp.splats_noalloc_setup()
        gotA = _pack(sp.splats_pack_noalloc, colA, depA, camA, WA, HA, cfg.r_scale)
    finally:
        sp.splats_destroy()
    # second and third call in a row with no context at all, on a smaller frame (stale counts in the array)
    gotB = _pack(sp.splats_pack_noalloc, colB, depB, camB, WB, HB, 1.5)
    gotC = _pack(sp.splats_pack_noalloc, colB, depB, camB, WB, HB, 1.5, radius_mode=sp.RADIUS_CONSTANT, radius_param=0.004)
    gotA2 = _pack(sp.splats_pack_noalloc, colA, depA, camA, WA, HA, cfg.r_scale)

    for got, want, what in ((gotA, wantA, "first call"), (gotB, wantB, "second call"), (gotC, wantC, "constant radius"),
                            (gotA2, wantA, "first frame again")):
        assert got[0] == want[0] and got[0] > 0, what
        np.testing.assert_array_equal(got[1], want[1], err_msg=what)
        np.testing.assert_array_equal(got[2], want[2], err_msg=what)


def test_pack_noalloc_on_its_own_stream():
    colB, depB, camB = synth.random_frame(640, 360, seed=5, fill=0.5)
    s = torch.cuda.Stream()
    dc, dd = torch.from_numpy(colB).cuda(), torch.from_numpy(depB).cuda()
    outs = []
    for stream in (None, s):
        samples, colors, count = _buffers(640 * 360)
        torch.cuda.synchronize()                      # calls share the array: never two in flight at once
        sp.splats_pack_noalloc(dc, dd, camB, 640, 360, 1.0, QUANT, samples, colors, count, stream=stream)
        torch.cuda.synchronize()
        outs.append((int(count.item()), samples.cpu().numpy(), colors.cpu().numpy()))
    assert outs[0][0] == outs[1][0] == int((depB > 0).sum())
    np.testing.assert_array_equal(outs[0][1], outs[1][1])
    np.testing.assert_array_equal(outs[0][2], outs[1][2])


def test_pack_noalloc_rejects_sizes_beyond_the_static_array():
    colB, depB, camB = synth.random_frame(64, 32, seed=1, fill=0.5)
    dc, dd = torch.from_numpy(colB).cuda(), torch.from_numpy(depB).cuda()
    samples, colors, count = _buffers(64 * 32)
    with pytest.raises(sp.SplatsError) as e:
        sp.splats_pack_noalloc(dc, dd, camB, 8192, 4096, 1.0, QUANT, samples, colors, count)   # 2 x the maximum
    assert e.value.code == -1 and "maximum" in str(e.value) and str(sp.NOALLOC_MAX_PIXELS) in str(e.value)
    torch.cuda.synchronize()
    assert int(count.item()) == -1                    # nothing was launched
    sp.splats_pack_noalloc(dc, dd, camB, 64, 32, 1.0, QUANT, samples, colors, count)           # and the next call is fine
    torch.cuda.synchronize()
    assert int(count.item()) == int((depB > 0).sum())
