"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C-ABI binding and
compare it with the oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2006_14726_b200 import binding as sp

RGBA_TOL = 1e-3          # BASELINE.json north_star: within 1e-3 absolute per channel ...
RGBA_BAD_FRACTION = 1e-4  # ... with at most 0.01 % of pixels beyond that


class Session:
    """One library context (the C ABI has a single global one)."""

    def __init__(self, max_W, max_H, exact_nodes=True):
        sp.splats_create(max_W, max_H)
        # the parity tests also want the exact float32 node boxes; the default (tiled) build carries only
        # the quantised ones, so with this option the update runs the exact pyramid refit as well
        # (include/splats.h, SPLATS_OPT_EXACT_NODES); the traversal records are the same either way
        # (tests/test_gpu_parity.py::test_exact_nodes_option_changes_nothing)
        sp.splats_set_option(sp.OPT_EXACT_NODES, 1 if exact_nodes else 0)

    def close(self):
        sp.splats_destroy()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def update(self, color, depth, cam, W, H, r_scale):
        self.d_color = torch.from_numpy(np.ascontiguousarray(color, dtype=np.float32)).cuda()
        self.d_depth = torch.from_numpy(np.ascontiguousarray(depth, dtype=np.float32)).cuda()
        sp.splats_update(self.d_color, self.d_depth, cam, W, H, r_scale)

    def render(self, cam, W2, H2, first_hit=False):
        out = torch.full((H2, W2, 4), -7.0, dtype=torch.float32, device="cuda")
        (sp.splats_render_first_hit if first_hit else sp.splats_render)(cam, W2, H2, out)
        torch.cuda.synchronize()
        return out.cpu().numpy()


def assert_bvh_bit_exact(sc, exact=True):
    """Morton codes, sorted permutation, topology, AABBs (exact, and the quantised records the
    traversal reads), splats: bit-exact against the oracle."""
    ex = sp.splats_export(aabbs=exact)
    n = sc["N"]
    assert ex["N"] == n
    if n == 0:
        return ex
    np.testing.assert_array_equal(ex["keys"].cpu().numpy().view(np.uint64), sc["sorted_codes"])
    np.testing.assert_array_equal(ex["perm"].cpu().numpy().view(np.uint32), sc["sorted_ids"])
    np.testing.assert_array_equal(ex["children"].cpu().numpy(), sc["children"])
    np.testing.assert_array_equal(ex["parents"].cpu().numpy(), sc["parents"])
    q = sp.splats_export_qnodes()
    want_rec, want_frame = oracle.quantise_child_boxes(sc)   # O7b, pinned in tests/test_oracle_tree.py
    if n > 1:   # what the traversal reads, word by word
        np.testing.assert_array_equal(q["qnodes"].cpu().numpy().view(np.uint32), want_rec)
        np.testing.assert_array_equal(q["frame"].cpu().numpy().view(np.uint32), want_frame.view(np.uint32))
    if exact:
        np.testing.assert_array_equal(ex["node_aabbs"].cpu().numpy().view(np.uint32), sc["aabbs"].view(np.uint32))
        if n > 1:   # the exact child boxes of every record, one by one (not only their union)
            cb = sp.splats_export_child_boxes().cpu().numpy().view(np.uint32).reshape(n - 1, 2, 6)
            want = sc["aabbs"].view(np.uint32)[sc["children"]]          # (n-1, 2, 6): box of each child node / leaf
            np.testing.assert_array_equal(cb, want)
    es = sp.splats_export_splats()
    np.testing.assert_array_equal(es["sphere"].cpu().numpy().view(np.uint32), sc["sphere_sorted"].view(np.uint32))
    np.testing.assert_array_equal(es["rgba"].cpu().numpy().view(np.uint32), sc["rgba_sorted"].view(np.uint32))
    lo_hi = es["lo_hi"].cpu().numpy()
    np.testing.assert_array_equal(lo_hi[:3], sc["lo"])
    np.testing.assert_array_equal(lo_hi[3:], sc["hi"])
    return ex


def assert_rgba_close(got, ref, what=""):
    got = got.reshape(-1, 4)
    ref = ref.reshape(-1, 4)
    err = np.abs(got.astype(np.float64) - ref.astype(np.float64)).max(axis=1)
    bad = int((err > RGBA_TOL).sum())
    allowed = int(np.floor(RGBA_BAD_FRACTION * err.size))
    assert bad <= allowed, f"{what}: {bad} of {err.size} pixels beyond {RGBA_TOL} (allowed {allowed}), max err {err.max():.3g}"
    return float(err.max()), bad


def check_scene(sess, color, depth, cam, W, H, r_scale, dst_cams, dst_sizes=None, mode="bvh", sample=None, seed=0,
                radius=(0, 0.0)):
    """update + export parity + one render per destination camera.  radius = (mode, param) of
    splats_set_radius / oracle.build_scene."""
    sc = oracle.build_scene(color, depth, cam, W, H, r_scale, radius[0], radius[1])
    sp.splats_set_radius(radius[0], radius[1])
    sess.update(color, depth, cam, W, H, r_scale)
    assert_bvh_bit_exact(sc)
    stats = []
    for i, dst in enumerate(dst_cams):
        W2, H2 = (W, H) if dst_sizes is None else dst_sizes[i]
        got = sess.render(dst, W2, H2)
        if sample is None:
            ref = oracle.render(sc, dst, W2, H2, mode)
            stats.append(assert_rgba_close(got, ref, f"camera {i}"))
        else:
            rng = np.random.default_rng(seed + i)
            px = rng.choice(W2 * H2, size=min(sample, W2 * H2), replace=False).astype(np.int64)
            ref = oracle.render(sc, dst, W2, H2, mode, pixels=px)
            stats.append(assert_rgba_close(got.reshape(-1, 4)[px], ref, f"camera {i} (sampled)"))
    return sc, stats
