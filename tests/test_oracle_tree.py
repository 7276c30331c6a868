"""Pins for the oracle's integer pipeline: cube, quantise, Morton keys, sort, tree (O1-O5).

Nothing here compares the oracle with itself: every expected value is a closed form, an invariant,
a library routine (numpy stable argsort) or a second, independently written builder that works on
UNSORTED integer coordinates by recursive partition (SURVEY.md §8(c) "What pins each part").
"""
import math

import numpy as np
import pytest

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import workloads as wl


# ------------------------------------------------------------------ O1 / O2 cube and quantiser
def test_cube_power_of_two_properties():
    for name, n in [("c1", 1024), ("c2", 4096), ("c4", 8192), ("c5", 4096)]:
        w = wl.make(name, n)
        lo, L, e = orc.cube(w.pos)
        ext = (w.pos.max(axis=0) - w.pos.min(axis=0)).max()
        assert np.array_equal(lo, w.pos.min(axis=0))
        assert L == 2.0 ** e and math.frexp(L)[0] == 0.5          # a power of two
        assert L / 2 <= ext < L                                     # smallest one above the extent
        q = orc.quantise(w.pos, lo, e)
        assert q.max() < 2 ** 21                                    # no clamp needed
        # truncation of an exactly scaled, once-rounded difference
        assert np.array_equal(q, np.floor((w.pos - lo) * 2.0 ** (21 - e)).astype(np.uint32))


def test_cube_hand_cases_exact():
    # extent exactly a power of two: L must be the NEXT power (strictly greater)
    pos = np.array([[0.0, 0.0, 0.0], [4.0, 1.0, 2.0]])
    lo, L, e = orc.cube(pos)
    assert (L, e) == (8.0, 3) and np.array_equal(lo, [0, 0, 0])
    q = orc.quantise(pos, lo, e)
    assert np.array_equal(q[1], [2 ** 20, 2 ** 18, 2 ** 19])
    # extent 3 -> L = 4; corner follows the minimum, also when negative
    pos = np.array([[-1.0, 5.0, 2.0], [2.0, 5.5, 2.25]])
    lo, L, e = orc.cube(pos)
    assert (L, e) == (4.0, 2) and np.array_equal(lo, [-1.0, 5.0, 2.0])
    assert np.array_equal(orc.quantise(pos, lo, e)[1], [3 * 2 ** 19, 2 ** 18, 2 ** 17])
    # all bodies coincident (or one body): E = 0 -> L = 1, every q = 0
    pos = np.full((5, 3), 7.25)
    lo, L, e = orc.cube(pos)
    assert (L, e) == (1.0, 0) and not orc.quantise(pos, lo, e).any()
    # tiny and huge scales stay exact powers of two
    lo, L, e = orc.cube(np.array([[0.0, 0, 0], [3e-200, 0, 0]]))
    assert L == 2.0 ** e and L / 2 <= 3e-200 < L
    lo, L, e = orc.cube(np.array([[0.0, 0, 0], [3e200, 0, 0]]))
    assert L == 2.0 ** e and L / 2 <= 3e200 < L


def test_cube_rejects_nonfinite():
    for bad in (np.nan, np.inf, -np.inf):
        pos = np.zeros((4, 3))
        pos[2, 1] = bad
        with pytest.raises(ValueError):
            orc.cube(pos)


# ------------------------------------------------------------------ O3 Morton keys
def _spread_mask(v):
    """Independent encoder: the classic magic-mask bit spreading, in numpy."""
    v = v.astype(np.uint64) & np.uint64(0x1FFFFF)
    v = (v | (v << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
    v = (v | (v << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
    v = (v | (v << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
    v = (v | (v << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
    v = (v | (v << np.uint64(2))) & np.uint64(0x1249249249249249)
    return v


def _decode(key):
    q = [0, 0, 0]
    for k in range(21):
        for a in range(3):
            q[a] |= ((key >> (3 * k + a)) & 1) << k
    return tuple(q)


def test_morton_closed_forms():
    assert orc.morton_key(0, 0, 0) == 0
    assert orc.morton_key(1, 0, 0) == 1
    assert orc.morton_key(0, 1, 0) == 2
    assert orc.morton_key(0, 0, 1) == 4
    assert orc.morton_key(2, 0, 0) == 8
    m = 2 ** 21 - 1
    assert orc.morton_key(m, m, m) == 2 ** 63 - 1
    assert orc.morton_key(m, 0, 0) == int("001" * 21, 2)
    assert orc.morton_key(0, 0, m) == int("100" * 21, 2)
    # the level-1 octant digit is (z,y,x) of the top bit
    assert orc.morton_key(2 ** 20, 0, 2 ** 20) >> 60 == 0b101


def test_morton_round_trip_and_spread_mask():
    rng = np.random.default_rng(5)
    q = rng.integers(0, 2 ** 21, size=(4000, 3), dtype=np.uint32)
    keys = np.array([orc.morton_key(int(a), int(b), int(c)) for a, b, c in q], dtype=np.uint64)
    ref = _spread_mask(q[:, 0]) | (_spread_mask(q[:, 1]) << np.uint64(1)) | (_spread_mask(q[:, 2]) << np.uint64(2))
    assert np.array_equal(keys, ref)
    for i in range(0, 4000, 97):
        assert _decode(int(keys[i])) == tuple(int(x) for x in q[i])
    # whole pipeline on real positions: key == spread(quantised coordinates)
    w = wl.make("c1")
    lo, L, e = orc.cube(w.pos)
    qq = orc.quantise(w.pos, lo, e)
    ref = _spread_mask(qq[:, 0]) | (_spread_mask(qq[:, 1]) << np.uint64(1)) | (_spread_mask(qq[:, 2]) << np.uint64(2))
    assert np.array_equal(orc.morton(w.pos, lo, e), ref)
    # Morton order is monotone along each axis when the others are fixed
    ks = [orc.morton_key(x, 5, 9) for x in range(64)]
    assert ks == sorted(ks)


# ------------------------------------------------------------------ O4 sort
def test_sort_matches_stable_argsort_with_ties():
    rng = np.random.default_rng(11)
    key = rng.integers(0, 50, size=5000).astype(np.uint64) << np.uint64(40)   # heavy ties
    key[::7] = np.uint64(2 ** 63 - 1)
    perm, skey = orc.sort(key)
    assert np.array_equal(perm, np.argsort(key, kind="stable").astype(np.uint32))
    assert np.array_equal(skey, key[perm])
    assert np.array_equal(np.sort(perm), np.arange(5000, dtype=np.uint32))    # a permutation
    assert (np.diff(skey.astype(np.float64)) >= 0).all()
    same = skey[1:] == skey[:-1]
    assert (perm[1:][same] > perm[:-1][same]).all()                           # ties by index


# ------------------------------------------------------------------ O5 tree
def _second_builder(q, C):
    """Independent builder: recursive top-down partition of UNSORTED integer coordinates by bit
    20-level, no keys and no sort.  Returns nodes in BFS order as tuples
    (level, prefix, count, parent, octant-mask) plus, per node, its set of body indices."""
    root = dict(level=0, prefix=0, idx=np.arange(q.shape[0]), parent=-1)
    nodes, queue = [], [root]
    while queue:                      # BFS, children pushed in octant order
        nxt = []
        for nd in queue:
            nd["id"] = len(nodes)
            nodes.append(nd)
        for nd in queue:
            nd["children"] = []
            nd["mask"] = 0
            if len(nd["idx"]) <= C or nd["level"] == 21:
                continue
            bit = 20 - nd["level"]
            sub = q[nd["idx"]]
            octant = ((sub[:, 0] >> bit) & 1) | (((sub[:, 1] >> bit) & 1) << 1) | (((sub[:, 2] >> bit) & 1) << 2)
            for o in range(8):
                sel = nd["idx"][octant == o]
                if len(sel):
                    ch = dict(level=nd["level"] + 1, prefix=nd["prefix"] * 8 + o, idx=sel, parent=nd["id"])
                    nd["children"].append(ch)
                    nd["mask"] |= 1 << o
                    nxt.append(ch)
        queue = nxt
    return nodes


@pytest.mark.parametrize("name,n,C", [("c1", 1024, 8), ("c1", 777, 1), ("c2", 3000, 16),
                                      ("c4", 6000, 16), ("c4", 2048, 2), ("c5", 5000, 32)])
def test_tree_equals_second_builder(name, n, C):
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    q = orc.quantise(w.pos, t.lo, t.e).astype(np.int64)
    nodes = _second_builder(q, C)
    assert t.M == len(nodes)
    assert t.depth == max(nd["level"] for nd in nodes)
    for nd in nodes:
        i = nd["id"]
        assert t.level[i] == nd["level"]
        assert t.count[i] == len(nd["idx"])
        assert t.parent[i] == nd["parent"]
        assert t.child_mask[i] == nd["mask"]
        assert t.first_child[i] == (nd["children"][0]["id"] if nd["children"] else -1)
        # the node's range of sorted bodies holds exactly the builder's bodies
        assert set(t.perm[t.begin[i]:t.begin[i] + t.count[i]].tolist()) == set(nd["idx"].tolist())
        if nd["level"]:
            assert int(t.skey[t.begin[i]]) >> (63 - 3 * nd["level"]) == nd["prefix"]


def test_tree_invariants():
    w = wl.make("c4", 20000)
    C = 16
    t = orc.build(w.pos, w.mass, C)
    leaf = t.first_child < 0
    assert (t.count[~leaf] > C).all() and (t.level[~leaf] < 21).all()
    assert ((t.count[leaf] <= C) | (t.level[leaf] == 21)).all()
    assert t.count[leaf].sum() == t.n
    assert (np.diff(t.level.astype(int)) >= 0).all()                 # ids level-monotone
    assert (t.child_mask[leaf] == 0).all()
    for i in np.flatnonzero(~leaf):
        k = bin(int(t.child_mask[i])).count("1")
        ch = np.arange(t.first_child[i], t.first_child[i] + k)
        assert (t.parent[ch] == i).all() and (t.level[ch] == t.level[i] + 1).all()
        assert t.begin[ch[0]] == t.begin[i] and t.count[ch].sum() == t.count[i]
        assert np.array_equal(t.begin[ch][1:], (t.begin[ch] + t.count[ch])[:-1])   # contiguous
        octs = [(int(t.skey[t.begin[c]]) >> (63 - 3 * int(t.level[c]))) & 7 for c in ch]
        assert octs == [o for o in range(8) if t.child_mask[i] >> o & 1]            # octant order
    assert t.M <= t.n + 21 * (t.n // (C + 1))                                      # hard bound


@pytest.mark.parametrize("k", [1, 2, 3])
def test_tree_lattice_closed_forms(k):
    """8^k bodies at the cell centres (i+1/2)/2^k of the unit cube: C=1 gives the complete octree of
    depth k, M=(8^(k+1)-1)/7; C=8 stops one level earlier, M=(8^k-1)/7."""
    g = (np.arange(2 ** k) + 0.5) / 2 ** k
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    rng = np.random.default_rng(k)
    pos = pos[rng.permutation(len(pos))]
    mass = np.full(len(pos), 1.0 / len(pos))
    t1 = orc.build(pos, mass, 1)
    assert t1.M == (8 ** (k + 1) - 1) // 7 and t1.depth == k
    assert (t1.count[t1.first_child < 0] == 1).all()
    t8 = orc.build(pos, mass, 8)
    assert t8.M == (8 ** k - 1) // 7 and t8.depth == k - 1
    assert (t8.count[t8.first_child < 0] == 8).all()
    # every node's monopole is the centre of its cell, exactly (power-of-two arithmetic)
    for t in (t1, t8):
        s = t.L / 2.0 ** t.level
        prefix = np.array([int(t.skey[b]) >> (63 - 3 * int(l)) if l else 0 for b, l in zip(t.begin, t.level)])
        for i in range(0, t.M, max(1, t.M // 50)):
            cell = [sum(((prefix[i] >> (3 * d + a)) & 1) << d for d in range(int(t.level[i]))) for a in range(3)]
            centre = (np.array(cell) + 0.5) * s[i]          # centre of the unit-cube cell
            assert np.allclose(t.mono[i, :3], centre, rtol=0, atol=4e-16)


def test_tree_depth_cap_with_coincident_bodies():
    """R9: more than C coincident bodies cannot be separated; the chain stops at level 21."""
    pos = np.zeros((40, 3))
    pos[:20] = [0.3, 0.3, 0.3]
    pos[20:] = np.random.default_rng(3).random((20, 3))
    t = orc.build(pos, np.ones(40), 4)
    assert t.depth == 21
    deep = np.flatnonzero(t.level == 21)
    assert len(deep) == 1 and t.count[deep[0]] == 20 and t.first_child[deep[0]] == -1
    # single-child chain above it
    assert t.count[t.parent[deep[0]]] == 20


def test_tree_small_n_edge_cases():
    t = orc.build(np.array([[1.0, 2.0, 3.0]]), np.array([2.0]), 8)
    assert t.M == 1 and t.depth == 0 and t.first_child[0] == -1 and t.count[0] == 1
    assert np.array_equal(t.mono[0], [1.0, 2.0, 3.0, 2.0])
    w = wl.make("c1", 8)
    t = orc.build(w.pos, w.mass, 8)
    assert t.M == 1                                     # n <= C: the root is a leaf
    t = orc.build(w.pos, w.mass, 7)
    assert t.M > 1 and t.first_child[0] == 1
