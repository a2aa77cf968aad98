"""Pins for oracle steps O5-O7: sort, binary radix tree (LBVH), refit."""
from pathlib import Path

import numpy as np
import pytest

import oracle
import synth

GOLDEN = Path(__file__).parent / "golden"


# Karras' per-node construction, restated from the published algorithm (direction,
# range by doubling + binary search, split by binary search, delta with index
# tie-break).  It is a different algorithm from the oracle's top-down bit split; the
# radix tree is unique, so both must give the same ranges, splits and node numbers.
def _clz(v, bits):
    return bits - int(v).bit_length()


def karras_tree(keys):
    n = len(keys)
    keys = [int(k) for k in keys]

    def delta(i, j):
        if j < 0 or j >= n:
            return -1
        if keys[i] == keys[j]:
            return 64 + _clz(i ^ j, 32)
        return _clz(keys[i] ^ keys[j], 64)

    children = np.zeros((n - 1, 2), np.int64)
    ranges = np.zeros((n - 1, 2), np.int64)
    for i in range(n - 1):
        d = 1 if delta(i, i + 1) > delta(i, i - 1) else -1
        dmin = delta(i, i - d)
        lmax = 2
        while delta(i, i + lmax * d) > dmin:
            lmax *= 2
        l, t = 0, lmax // 2
        while t >= 1:
            if delta(i, i + (l + t) * d) > dmin:
                l += t
            t //= 2
        j = i + l * d
        dnode = delta(i, j)
        s, t = 0, l
        while t > 1:
            t = (t + 1) // 2
            if delta(i, i + (s + t) * d) > dnode:
                s += t
        g = i + s * d + min(d, 0)
        lo, hi = min(i, j), max(i, j)
        children[i, 0] = (n - 1 + g) if lo == g else g
        children[i, 1] = (n - 1 + g + 1) if hi == g + 1 else g + 1
        ranges[i] = (lo, hi)
    return children, ranges


def _check_invariants(children, parents, ranges, n):
    assert children.shape == (n - 1, 2) and parents.shape == (2 * n - 1,)
    assert parents[0] == -1
    # every node except the root is the child of exactly one internal node
    counts = np.bincount(children.reshape(-1), minlength=2 * n - 1)
    assert counts[0] == 0 and np.all(counts[1:] == 1)
    for j in range(n - 1):
        for s in range(2):
            assert parents[children[j, s]] == j
    # contiguous ranges: children partition the parent's range at the split
    def rng(node):
        return (ranges[node, 0], ranges[node, 1]) if node < n - 1 else (node - (n - 1),) * 2
    assert tuple(ranges[0]) == (0, n - 1)
    for j in range(n - 1):
        (a, g), (g1, b) = rng(children[j, 0]), rng(children[j, 1])
        assert a == ranges[j, 0] and b == ranges[j, 1] and g1 == g + 1
        # Karras numbering
        if children[j, 0] < n - 1:
            assert children[j, 0] == g
        if children[j, 1] < n - 1:
            assert children[j, 1] == g + 1


def test_sort_is_stable_sort_by_code():
    rng = np.random.default_rng(3)
    for bits in (2, 8, 63):
        codes = rng.integers(0, 2 ** bits, 5000, dtype=np.uint64)
        order = oracle.sort_codes(codes)
        np.testing.assert_array_equal(order, np.argsort(codes, kind="stable"))
        s = codes[order]
        assert np.all(s[:-1] <= s[1:])
        ties = s[:-1] == s[1:]
        assert np.all(order[:-1][ties] < order[1:][ties])


def test_tree_hand_worked_8_keys():
    lines = [l.split() for l in (GOLDEN / "karras8.txt").read_text().splitlines() if l and not l.startswith("#")]
    keys = np.array([int(v) for v in lines[0][1:]], np.uint64)
    n = keys.size
    children, parents, ranges = oracle.tree(keys)
    dec = lambda s: int(s[1:]) + (n - 1 if s[0] == "L" else 0)
    for row in lines[1:]:
        j = int(row[0])
        assert tuple(ranges[j]) == (int(row[1]), int(row[2]))
        assert tuple(children[j]) == (dec(row[3]), dec(row[4]))
    _check_invariants(children, parents, ranges, n)


@pytest.mark.parametrize("bits", [3, 6, 63])
def test_tree_equals_karras_per_node(bits):
    rng = np.random.default_rng(100 + bits)
    for trial in range(150):
        n = int(rng.integers(2, 60))
        keys = np.sort(rng.integers(0, 2 ** bits, n, dtype=np.uint64))
        children, parents, ranges = oracle.tree(keys)
        kc, kr = karras_tree(keys)
        np.testing.assert_array_equal(children, kc)
        np.testing.assert_array_equal(ranges, kr)
        _check_invariants(children, parents, ranges, n)


def test_tree_all_duplicates_splits_on_position():
    keys = np.full(13, 42, np.uint64)
    children, parents, ranges = oracle.tree(keys)
    kc, kr = karras_tree(keys)
    np.testing.assert_array_equal(children, kc)
    # positions 0..12: highest differing bit of 0 and 12 is bit 3 -> split after 7
    assert tuple(children[0]) == (7, 8)
    _check_invariants(children, parents, ranges, 13)


def test_tree_n1_n2():
    children, parents, ranges = oracle.tree(np.array([5], np.uint64))
    assert children.shape == (0, 2) and parents.tolist() == [-1]
    children, parents, ranges = oracle.tree(np.array([5, 9], np.uint64))
    assert children.tolist() == [[1, 2]] and parents.tolist() == [-1, 0, 0]


def test_refit_is_exact_union_over_ranges():
    for cfg, frame in ((synth.make_config(0), None), (None, synth.random_frame(40, 25, 5, 0.6))):
        if cfg is not None:
            color, depth = synth.source_frame(cfg, 0)
            sc = oracle.build_scene(color, depth, cfg.src_cams[0], cfg.W, cfg.H, cfg.r_scale)
        else:
            color, depth, cam = frame
            sc = oracle.build_scene(color, depth, cam, 40, 25, 2.0)
        n = sc["N"]
        sp = sc["sphere_sorted"]
        leaf_lo = sp[:, :3] - sp[:, 3:4]
        leaf_hi = sp[:, :3] + sp[:, 3:4]
        np.testing.assert_array_equal(sc["aabbs"][n - 1:, :3], leaf_lo)
        np.testing.assert_array_equal(sc["aabbs"][n - 1:, 3:], leaf_hi)
        for j in range(n - 1):
            a, b = sc["ranges"][j]
            np.testing.assert_array_equal(sc["aabbs"][j, :3], leaf_lo[a:b + 1].min(axis=0))
            np.testing.assert_array_equal(sc["aabbs"][j, 3:], leaf_hi[a:b + 1].max(axis=0))
        _check_invariants(sc["children"], sc["parents"], sc["ranges"], n)
        # sorted order is by (code, id)
        key = sc["sorted_codes"].astype(object) * (2 ** 32) + sc["sorted_ids"].astype(object)
        assert all(key[i] < key[i + 1] for i in range(n - 1))


# ---- O7b: the 16-bit storage format of the child boxes (S13)
def _two_leaf_scene(c0, c1, r0, r1):
    """Two splats by hand: centres c0, c1 (c0 sorts first), radii r0, r1; one internal node, two leaves."""
    f32 = np.float32
    sph = np.array([[*c0, r0], [*c1, r1]], dtype=f32)
    lo, hi = sph[:, :3].min(0), sph[:, :3].max(0)
    aabbs = np.zeros((3, 6), f32)                       # node 0 = root, nodes 1, 2 = leaves
    for i in range(2):
        aabbs[1 + i, :3] = sph[i, :3] - sph[i, 3]
        aabbs[1 + i, 3:] = sph[i, :3] + sph[i, 3]
    aabbs[0, :3], aabbs[0, 3:] = aabbs[1:, :3].min(0), aabbs[1:, 3:].max(0)
    return dict(N=2, sphere_sorted=sph, lo=lo, hi=hi, aabbs=aabbs, children=np.array([[1, 2]], np.int32))


def test_quantised_boxes_hand_worked():
    # frame: lo = (0, 0, 0), hi = (3, 0, 0) + rmax = 1 -> qlo = -1, ext = (5, 2, 2), codes per unit = 13107, 32767.5, 32767.5
    sc = _two_leaf_scene((0.0, 0.0, 0.0), (3.0, 0.0, 0.0), 1.0, 0.5)
    rec, frame = oracle.quantise_child_boxes(sc)
    assert frame.tolist() == [0.0, 0.0, 0.0, 3.0, 0.0, 0.0, 1.0]
    w = rec[0]
    # left child: box [-1, 1]^3 -> x: 0 .. 2 * 13107 = 26214; y, z: 0 .. 65535 (the whole extent)
    assert (w[0] & 0xffff, w[0] >> 16) == (0, 26214)
    assert (w[1] & 0xffff, w[1] >> 16) == (0, 65535) and w[2] == w[1]
    # right child: box x [2.5, 3.5], y, z [-0.5, 0.5] -> x: floor(3.5 * 13107) = 45874 .. ceil(4.5 * 13107) = 58982;
    # y, z: floor(0.5 * 32767.5) = 16383 .. ceil(1.5 * 32767.5) = 49152
    assert (w[3] & 0xffff, w[3] >> 16) == (45874, 58982)
    assert (w[4] & 0xffff, w[4] >> 16) == (16383, 49152) and w[5] == w[4]
    assert (w[6], w[7]) == (0x80000000, 0x80000001)     # both children are leaves: sorted positions 0 and 1


def test_quantised_boxes_zero_extent_axis_and_n_below_two():
    sc = _two_leaf_scene((1.0, 2.0, 3.0), (2.0, 2.0, 3.0), 0.0, 0.0)   # radii 0: y and z have no extent at all
    rec, _ = oracle.quantise_child_boxes(sc)
    assert rec[0, 1] == 0 and rec[0, 2] == 0 and rec[0, 4] == 0 and rec[0, 5] == 0
    assert (rec[0, 0] & 0xffff, rec[0, 0] >> 16) == (0, 0) and (rec[0, 3] & 0xffff, rec[0, 3] >> 16) == (65535, 65535)
    one = dict(N=1, sphere_sorted=np.zeros((1, 4), np.float32), lo=np.zeros(3), hi=np.zeros(3), aabbs=np.zeros((1, 6), np.float32),
               children=np.zeros((0, 2), np.int32))
    assert oracle.quantise_child_boxes(one)[0].shape == (0, 8)


@pytest.mark.parametrize("seed,fill,r_scale", [(1, 0.7, 1.0), (2, 0.3, 2.5), (3, 1.0, 0.5)])
def test_quantised_boxes_contain_the_exact_ones_and_commute_with_the_union(seed, fill, r_scale):
    W, H = 96, 54
    color, depth, cam = synth.random_frame(W, H, seed, fill=fill)
    sc = oracle.build_scene(color, depth, cam, W, H, r_scale)
    n = sc["N"]
    rec, frame = oracle.quantise_child_boxes(sc)
    # (a) decoded in float64: never smaller than the exact box, at most one code step larger per plane
    fr = frame.astype(np.float64)
    qlo = fr[0:3] - fr[6]
    step = ((fr[3:6] + fr[6]) - qlo) / 65535.0
    w = rec[:, 0:6].reshape(-1, 2, 3)
    lo, hi = qlo + (w & 0xffff) * step, qlo + (w >> 16) * step
    want = sc["aabbs"][sc["children"]].astype(np.float64)
    eps = 1e-6 * np.abs(want).max()
    assert np.all(lo <= want[:, :, 0:3] + eps) and np.all(hi >= want[:, :, 3:6] - eps)
    assert np.all(lo >= want[:, :, 0:3] - step - eps) and np.all(hi <= want[:, :, 3:6] + step + eps)
    # (b) quantisation is monotone, so it commutes with the union: the code box of an internal child equals the
    # min / max of the code boxes stored in that child's own record (what a bottom-up build on codes relies on)
    ql, qh = (w & 0xffff).astype(np.int64), (w >> 16).astype(np.int64)
    ch = sc["children"]
    for j in range(n - 1):
        for side in range(2):
            c = int(ch[j, side])
            if c < n - 1:
                assert np.array_equal(ql[j, side], ql[c].min(axis=0)) and np.array_equal(qh[j, side], qh[c].max(axis=0))
    # (c) links: every node and every leaf is referenced exactly once
    links = rec[:, 6:8].reshape(-1)
    leaves = np.sort(links[links >= 0x80000000] & 0x7fffffff)
    inner = np.sort(links[links < 0x80000000])
    assert np.array_equal(leaves, np.arange(n)) and np.array_equal(inner, np.arange(1, n - 1))
