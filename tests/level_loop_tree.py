"""A second, independent construction of the sparse octree: the paper's literal per-level loop.

PAPER.md:63 (section 2.1, Fig.1): "For a given level, we mask the keys of non-flagged particles ...
Particles with identical masked keys are grouped together ... Cells containing up-to Nleaf particles
are marked as leaves, otherwise they are marked as nodes.  If a particle is assigned to a leaf the
particle is flagged as complete ... repeated for every single level in serial until all particles are
assigned to leaves or that the maximal depth of the tree is reached".
PAPER.md:65 (Fig.2): linking -- each cell "locates its parent and the first child ... by a binary
search of the appropriate Morton key in the array of tree-cells".

Written with numpy only; shares nothing with oracle/bh_oracle.cpp (which recurses on key runs).
Used by tests to pin the oracle's tree (P4).
"""
import numpy as np

MAXLEVEL = 20


def level_mask(level: int) -> np.uint64:
    bits = 3 * level
    return np.uint64(((1 << bits) - 1) << (60 - bits)) if level > 0 else np.uint64(0)


def level_loop_tree(keys_sorted: np.ndarray, nleaf: int = 16):
    keys = np.ascontiguousarray(keys_sorted, dtype=np.uint64)
    n = keys.shape[0]
    flagged = np.zeros(n, dtype=bool)
    lv_key, lv_begin, lv_count, lv_leaf = [], [], [], []
    for level in range(MAXLEVEL + 1):
        active = np.nonzero(~flagged)[0]
        if active.size == 0:
            break
        mk = keys[active] & level_mask(level)
        new = np.ones(active.size, dtype=bool)
        new[1:] = mk[1:] != mk[:-1]
        starts = np.nonzero(new)[0]
        counts = np.diff(np.append(starts, active.size))
        # a group of identical masked keys is contiguous in the particle array as well
        pbegin = active[starts]
        assert np.all(active[starts + counts - 1] - pbegin + 1 == counts)
        leaf = (counts <= nleaf) | (level == MAXLEVEL)
        lv_key.append(mk[starts])
        lv_begin.append(pbegin)
        lv_count.append(counts)
        lv_leaf.append(leaf)
        done = np.repeat(leaf, counts)
        flagged[active[done]] = True
    nlev = len(lv_key)
    sizes = [k.shape[0] for k in lv_key] + [0] * (MAXLEVEL + 1 - nlev)
    level_offset = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    C = int(level_offset[-1])
    level = np.concatenate([np.full(k.shape[0], L, np.int32) for L, k in enumerate(lv_key)])
    mkey = np.concatenate(lv_key)
    pbegin = np.concatenate(lv_begin).astype(np.int64)
    pcount = np.concatenate(lv_count).astype(np.int64)
    leaf = np.concatenate(lv_leaf)
    parent = np.full(C, -1, np.int64)
    child_begin = np.full(C, -1, np.int64)
    nchild = np.zeros(C, np.int32)
    # link (binary search by key, one level up / one level down)
    for L in range(nlev):
        lo, hi = int(level_offset[L]), int(level_offset[L + 1])
        if L > 0:
            plo, phi = int(level_offset[L - 1]), int(level_offset[L])
            pk = mkey[lo:hi] & level_mask(L - 1)
            idx = np.searchsorted(mkey[plo:phi], pk, side="left")
            assert np.all(mkey[plo:phi][idx] == pk)
            parent[lo:hi] = plo + idx
        if L + 1 < nlev:
            clo, chi = int(level_offset[L + 1]), int(level_offset[L + 2])
            ck = mkey[clo:chi] & level_mask(L)
            first = np.searchsorted(ck, mkey[lo:hi], side="left")
            last = np.searchsorted(ck, mkey[lo:hi], side="right")
            has = last > first
            child_begin[lo:hi] = np.where(has, clo + first, -1)
            nchild[lo:hi] = (last - first).astype(np.int32)
    assert np.all((nchild == 0) == leaf)
    prefix = np.array([int(k) >> (60 - 3 * int(L)) if L > 0 else 0 for k, L in zip(mkey, level)], dtype=np.uint64)
    return dict(level_offset=level_offset.astype(np.int64), level=level, prefix=prefix, pbegin=pbegin,
                pcount=pcount, child_begin=child_begin, nchild=nchild, parent=parent)
