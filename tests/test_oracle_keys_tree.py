"""Pins P1-P5 for the CPU oracle: keys, sort, tree, groups (no GPU).

Each test checks the oracle against something other than itself: values the paper prints
(tests/golden/paper_examples.txt), the paper's own List 1, numpy's stable sort, a second tree
construction (tests/level_loop_tree.py, the paper's literal per-level loop) and structural invariants.
"""
import os

import numpy as np
import pytest

import bh_inputs
import oracle
from level_loop_tree import level_loop_tree, level_mask

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_examples.txt")


def _golden():
    rows = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = [x.strip() for x in line.split("|")]
        rows[f[0]] = f[1:]
    return rows


def list1_dilate(value: int) -> int:
    """PAPER.md:380-390, List 1, restated: the 10-bit dilate by shift-and-mask."""
    x = value & 0x03FF
    x = ((x << 16) + x) & 0xFF0000FF
    x = ((x << 8) + x) & 0x0F00F00F
    x = ((x << 4) + x) & 0xC30C30C3
    x = ((x << 2) + x) & 0x49249249
    return x & 0xFFFFFFFF


# ---------------------------------------------------------------- P1: dilate / key
def test_paper_mask_example():
    _, a, b, r = _golden()["mask_example"]
    assert int(a, 2) & int(b, 2) == int(r, 2)
    # the level mask of the tree construction is that operation: keep the top 3L bits of a 60-bit key
    k = np.uint64(0xFEDCBA987654321)
    assert int(k & level_mask(1)) == (int(k) >> 57) << 57
    assert int(level_mask(20)) == (1 << 60) - 1 and int(level_mask(0)) == 0


def test_paper_dilate_example():
    _, inp, full, printed = _golden()["dilate_example"]
    v = int(inp, 2)
    assert v == 0x13B
    want = int(full.replace(" ", ""), 2)
    assert want == 0x1009209
    assert oracle.dilate(v, 10) == want
    # the 5 triples that survived text extraction occur, in order, among the 10 of the full value
    it = iter(full.split())
    assert all(any(t == u for u in it) for t in printed.split())


def test_dilate_matches_list1_for_all_10_bit_values():
    for v in range(1024):
        assert oracle.dilate(v, 10) == list1_dilate(v)


def test_constants_match_paper():
    c = dict(x.split("=") for x in _golden()["constants"][1:])
    assert oracle.MAXLEVEL == int(c["max_level"]) and 3 * oracle.MAXLEVEL == int(c["key_bits_total"])
    assert oracle.NLEAF == int(c["nleaf"]) and oracle.NCRIT == int(c["ncrit"])


def _deinterleave(key):
    g = [0, 0, 0]
    for b in range(20):
        g[0] |= ((key >> (3 * b + 2)) & 1) << b
        g[1] |= ((key >> (3 * b + 1)) & 1) << b
        g[2] |= ((key >> (3 * b)) & 1) << b
    return g


def test_keys_cube_corners_and_roundtrip():
    # 8 corners of [0,1]^3 plus the centre: domain lo = 0, ext = 1 -> e = 1, side 2, scale 2^19
    pts = np.array([[x, y, z, 1.0] for x in (0, 1) for y in (0, 1) for z in (0, 1)] + [[0.5, 0.5, 0.5, 1.0]],
                   np.float32)
    lo, hi, e, ok = oracle.domain(pts)
    assert ok and e == 1 and np.all(lo == 0) and np.all(hi == 1)
    k = oracle.keys(pts, lo, e)
    for p, key in zip(pts, k):
        g = _deinterleave(int(key))
        assert g == [int(p[0] * 2 ** 19), int(p[1] * 2 ** 19), int(p[2] * 2 ** 19)]
    # octant order: x is the most significant bit of a triple, then y, then z (A4)
    top = [int(key) >> 57 for key in k[:8]]   # coordinate 2^19 -> bit 19 -> key bits 57..59 = level-1 triple
    assert top == [0, 1, 2, 3, 4, 5, 6, 7]
    assert int(k.max()) < (1 << 60)


def test_grid_coordinates_bounds_min_and_monotone():
    pm, _, _ = bh_inputs.make("c1", n=4096)
    lo, hi, e, ok = oracle.domain(pm)
    assert ok
    k = oracle.keys(pm, lo, e)
    g = np.array([_deinterleave(int(x)) for x in k])
    assert g.min() >= 0 and g.max() < 2 ** 20
    for ax in range(3):
        assert g[np.argmin(pm[:, ax]), ax] == 0           # particle at the per-axis minimum -> 0
        o = np.argsort(pm[:, ax], kind="stable")
        assert np.all(np.diff(g[o, ax]) >= 0)              # monotone in x
        # the definition, restated: trunc((x - lo) * 2^(20 - e)) in float32 then exact scaling
        d = (pm[:, ax] - lo[ax]).astype(np.float32)
        want = np.floor(d.astype(np.float64) * 2.0 ** (20 - e)).astype(np.int64)
        assert np.array_equal(g[:, ax], want)
    assert 2.0 ** e > float((hi - lo).max()) >= 2.0 ** (e - 1)


def test_domain_rejects_bad_input():
    pm, _, _ = bh_inputs.make("c1", n=64)
    for bad in (np.nan, np.inf):
        q = pm.copy(); q[5, 1] = bad
        assert not oracle.domain(q)[3]
    q = pm.copy(); q[7, 3] = 0.0
    assert not oracle.domain(q)[3]
    one = np.array([[1.0, 2.0, 3.0, 1.0]], np.float32)     # single particle: ext = 0 -> 1 -> e = 1
    assert oracle.domain(one)[2] == 1 and int(oracle.keys(one, one[0, :3], 1)[0]) == 0


# ---------------------------------------------------------------- P3: sort
def test_sort_is_numpy_stable_argsort():
    rng = np.random.default_rng(3)
    k = rng.integers(0, 1 << 60, 20000, dtype=np.uint64)
    k[::7] = k[3]          # many ties
    k[100:200] = 0
    perm = oracle.sort_perm(k)
    assert np.array_equal(perm, np.argsort(k, kind="stable").astype(np.uint32))
    assert np.all(np.diff(k[perm].astype(np.int64)) >= 0)
    assert np.array_equal(np.sort(perm), np.arange(k.size, dtype=np.uint32))


# ---------------------------------------------------------------- P4: tree
def _sorted_keys(pm):
    lo, hi, e, ok = oracle.domain(pm)
    k = oracle.keys(pm, lo, e)
    return k[oracle.sort_perm(k)]


def _check_tree_invariants(t, keys, nleaf=16):
    C, n = t.ncells, keys.shape[0]
    leaf = t.nchild == 0
    assert t.level[0] == 0 and t.pbegin[0] == 0 and t.pcount[0] == n and t.parent[0] == -1
    # every particle in exactly one leaf
    cover = np.zeros(n + 1, np.int64)
    np.add.at(cover, t.pbegin[leaf], 1)
    np.add.at(cover, t.pbegin[leaf] + t.pcount[leaf], -1)
    assert np.all(np.cumsum(cover)[:n] == 1) and t.pcount[leaf].sum() == n
    assert np.all((t.pcount[leaf] <= nleaf) | (t.level[leaf] == 20))
    assert np.all(t.pcount[~leaf] > nleaf) and np.all(t.level[~leaf] < 20)
    assert np.all((t.nchild[~leaf] >= 1) & (t.nchild[~leaf] <= 8))
    # level-major, ascending pbegin within a level
    for L in range(21):
        a, b = t.level_offset[L], t.level_offset[L + 1]
        assert np.all(t.level[a:b] == L) and np.all(np.diff(t.pbegin[a:b]) > 0)
    assert t.level_offset[21] == C
    # children consecutive, tile the parent's range, extend the parent's prefix
    nodes = np.nonzero(~leaf)[0]
    exp_cb = np.empty(nodes.size, np.int64)
    for L in range(20):
        sel = nodes[t.level[nodes] == L]
        exp = t.level_offset[L + 1] + np.concatenate([[0], np.cumsum(t.nchild[sel])[:-1]]) if sel.size else []
        assert np.array_equal(t.child_begin[sel], exp)
    for c in nodes[:: max(1, nodes.size // 2000)]:
        ch = np.arange(t.child_begin[c], t.child_begin[c] + t.nchild[c])
        assert np.all(t.parent[ch] == c) and np.all(t.level[ch] == t.level[c] + 1)
        assert t.pbegin[ch[0]] == t.pbegin[c] and np.all(t.pbegin[ch[1:]] == (t.pbegin[ch] + t.pcount[ch])[:-1])
        assert t.pbegin[ch[-1]] + t.pcount[ch[-1]] == t.pbegin[c] + t.pcount[c]
        assert np.all(t.prefix[ch] >> np.uint64(3) == t.prefix[c])
        assert np.all(np.diff(t.prefix[ch].astype(np.int64)) > 0)
    # prefix is the particles' key prefix
    for c in range(0, C, max(1, C // 3000)):
        sh = np.uint64(60 - 3 * int(t.level[c]))
        ks = keys[t.pbegin[c]: t.pbegin[c] + t.pcount[c]]
        assert np.all((ks >> sh if t.level[c] > 0 else ks * np.uint64(0)) == t.prefix[c])


@pytest.mark.parametrize("cfg,n", [("c1", 16384), ("c3", 30000), ("c1", 1000), ("c1", 17), ("c1", 16), ("c1", 1)])
def test_tree_two_constructions_agree_and_invariants(cfg, n):
    pm, _, _ = bh_inputs.make(cfg, n=n)
    ks = _sorted_keys(pm)
    t = oracle.build_tree(ks)
    ref = level_loop_tree(ks)
    for name in ("level_offset", "level", "prefix", "pbegin", "pcount", "child_begin", "nchild", "parent"):
        assert np.array_equal(getattr(t, name), ref[name]), name
    _check_tree_invariants(t, ks)


def test_tree_hand_built_cases():
    # N = 16 -> the root is a leaf;  N = 17 spread over octants -> root node + leaves
    ks = np.sort(np.arange(16, dtype=np.uint64) << np.uint64(56))
    t = oracle.build_tree(ks)
    assert t.ncells == 1 and t.nchild[0] == 0 and t.pcount[0] == 16
    ks = np.sort(np.concatenate([ks, [np.uint64(7) << np.uint64(57)]]))
    t = oracle.build_tree(ks)
    assert t.nchild[0] == 8 and t.ncells == 9 and np.all(t.level[1:] == 1)
    # 8 corners x 3 identical particles each: 24 > 16 -> root node with 8 leaves of 3
    corner = np.array([(o << 57) | ((1 << 57) - 1) * 0 for o in range(8)], dtype=np.uint64)
    ks = np.sort(np.repeat(corner, 3))
    t = oracle.build_tree(ks)
    assert t.ncells == 9 and np.all(t.pcount[1:] == 3) and np.all(t.nchild[1:] == 0)
    # 40 identical keys: a chain of 20 single-child nodes ending in a level-20 overflow leaf (A9)
    ks = np.full(40, 0x123456789ABCDEF, dtype=np.uint64)
    t = oracle.build_tree(ks)
    assert t.ncells == 21 and np.all(t.nchild[:20] == 1) and t.nchild[20] == 0
    assert t.level[20] == 20 and t.pcount[20] == 40
    ref = level_loop_tree(ks)
    assert np.array_equal(t.parent, ref["parent"]) and np.array_equal(t.child_begin, ref["child_begin"])


# ---------------------------------------------------------------- P5: groups
@pytest.mark.parametrize("cfg,n", [("c1", 16384), ("c3", 30000), ("c1", 50)])
def test_groups_partition(cfg, n):
    pm, _, _ = bh_inputs.make(cfg, n=n)
    ks = _sorted_keys(pm)
    t = oracle.make_groups(oracle.build_tree(ks))
    assert t.gbegin[0] == 0 and np.all(t.gbegin[1:] == (t.gbegin + t.gcount)[:-1])
    assert t.gbegin[-1] + t.gcount[-1] == n
    assert np.all((t.gcount >= 1) & (t.gcount <= 64))
    par = t.parent[t.gcell]
    assert np.all((par < 0) | (t.pcount[np.maximum(par, 0)] > 64))
    assert np.array_equal(t.pbegin[t.gcell], t.gbegin) and np.array_equal(t.pcount[t.gcell], t.gcount)


def test_groups_overflow_leaf_is_chunked():
    ks = np.full(150, 0x123456789ABCDEF, dtype=np.uint64)
    t = oracle.make_groups(oracle.build_tree(ks))
    assert list(t.gcount) == [64, 64, 22] and list(t.gbegin) == [0, 64, 128]
    assert np.all(t.gcell == 20)


# ---------------------------------------------------------------- A13: group boxes (the walk's targets, S7)
@pytest.mark.parametrize("cfg,n", [("c1", 16384), ("c3", 30000), ("c1", 50), ("c1", 1)])
def test_group_boxes_are_the_min_and_max_of_the_groups_particles(cfg, n):
    """orc_group_boxes against numpy's own min / max over each group's slice, the cell a group comes from (a group is all
    of one cell's particles unless it is a chunk of an overflow leaf: then the cell's box contains it) and the domain."""
    pm, vel, _ = bh_inputs.make(cfg, n=n)
    st = oracle.tree_build(pm, vel)
    t = st.tree
    assert t.gbox.shape == (t.ngroups, 6) and t.gbox.dtype == np.float32
    for g in range(t.ngroups):
        p = st.pos[t.gbegin[g]: t.gbegin[g] + t.gcount[g], :3]
        assert np.array_equal(t.gbox[g, :3], p.min(axis=0)) and np.array_equal(t.gbox[g, 3:], p.max(axis=0))
    whole = t.pcount[t.gcell] == t.gcount
    assert np.array_equal(t.gbox[whole], t.box[t.gcell[whole]])
    assert np.all(t.gbox[:, :3] >= t.box[t.gcell][:, :3]) and np.all(t.gbox[:, 3:] <= t.box[t.gcell][:, 3:])
    assert np.array_equal(t.gbox[:, :3].min(axis=0), st.pos[:, :3].min(axis=0)) and np.array_equal(t.gbox[:, 3:].max(axis=0), st.pos[:, :3].max(axis=0))


def test_group_boxes_of_overflow_chunks():
    """150 particles on one key: groups of 64, 64, 22 consecutive particles, each with its own box inside the leaf's."""
    rng = np.random.default_rng(3)
    pm = np.zeros((150, 4), np.float32)
    pm[:, :3] = (0.25 + rng.random((150, 3)) * 1e-9).astype(np.float32)      # one level-20 cell of the unit cube
    pm[:, 3] = 1.0 / 150
    far = np.array([[0.0, 0.0, 0.0, 1e-3], [1.0, 1.0, 1.0, 1e-3]], np.float32)  # fixes the domain to [0, 2)^3
    st = oracle.tree_build(np.concatenate([far[:1], pm, far[1:]]), None)
    t = st.tree
    big = np.nonzero(t.gcount == 64)[0]
    assert big.size == 2 and sorted(t.gcount.tolist()) == [1, 1, 22, 64, 64]
    for g in range(t.ngroups):
        p = st.pos[t.gbegin[g]: t.gbegin[g] + t.gcount[g], :3]
        assert np.array_equal(t.gbox[g, :3], p.min(axis=0)) and np.array_equal(t.gbox[g, 3:], p.max(axis=0))
