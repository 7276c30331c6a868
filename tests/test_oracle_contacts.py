"""Pins of the oracle's broad phase (O17) and aggregate identification (O18,
PAPER.md:154-164): closed forms on lattices and hand cases, an independent cell-list search written
here in numpy, scipy's connected_components and a union-find written here.  CPU only."""
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import workloads as wl


def lattice(k, a=1.0):
    g = np.arange(k, dtype=np.float64) * a
    return np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)


def test_bound_radius_hand_values():
    vel = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 0.0], [1.0, 2.0, 2.0]])
    R = np.array([1.0, 0.5, 0.25])
    assert np.array_equal(orc.bound_radius(vel, R, 0.5), np.array([3.5, 0.5, 1.75]))   # |v| = 5, 0, 3
    assert np.array_equal(orc.bound_radius(None, R, 0.5), R)
    assert np.array_equal(orc.bound_radius(vel, R, 0.0), R)


def test_two_bodies_touching_counts_and_velocity_inflation():
    pos = np.array([[0.0, 0, 0], [3.0, 0, 0]])
    R = np.array([1.0, 2.0])
    assert orc.broadphase(pos, R).tolist() == [[0, 1]]                 # distance == b0 + b1: touching counts
    assert orc.broadphase(pos, np.array([1.0, 1.9999999])).tolist() == []
    # at rest the spheres miss each other; moving at |v| = 4 for dt = 0.25 the swept volume reaches
    R2 = np.array([0.5, 1.5])
    assert orc.broadphase(pos, orc.bound_radius(None, R2, 0.25)).tolist() == []
    vel = np.array([[4.0, 0, 0], [0.0, 0, 0]])
    assert orc.broadphase(pos, orc.bound_radius(vel, R2, 0.25)).tolist() == [[0, 1]]
    # direction of the velocity does not matter (a bound, not a trajectory)
    vel = np.array([[0.0, -4.0, 0], [0.0, 0, 0]])
    assert orc.broadphase(pos, orc.bound_radius(vel, R2, 0.25)).tolist() == [[0, 1]]


@pytest.mark.parametrize("k", [2, 3, 5])
def test_cubic_lattice_closed_forms(k):
    pos = lattice(k)
    n = k ** 3
    faces, edges, corners = 3 * k * k * (k - 1), 6 * k * (k - 1) ** 2, 4 * (k - 1) ** 3
    assert len(orc.broadphase(pos, np.full(n, 0.5))) == faces              # spacing 1, radii 1/2: face neighbours touch
    assert len(orc.broadphase(pos, np.full(n, 0.49))) == 0
    assert len(orc.broadphase(pos, np.full(n, 0.75))) == faces + edges     # sqrt(2) <= 1.5 < sqrt(3)
    assert len(orc.broadphase(pos, np.full(n, 0.9))) == faces + edges + corners   # sqrt(3) <= 1.8 < 2
    p = orc.broadphase(pos, np.full(n, 0.5))
    assert (p[:, 0] < p[:, 1]).all()
    assert np.array_equal(p, p[np.lexsort((p[:, 1], p[:, 0]))])            # lexicographic order


def cell_list_pairs(pos, b):
    """Independent search: hash bodies into a uniform grid of cell size 2 max(b), test the 27 cells."""
    h = 2.0 * b.max()
    q = np.floor((pos - pos.min(0)) / h).astype(np.int64)
    cells = {}
    for i, c in enumerate(map(tuple, q)):
        cells.setdefault(c, []).append(i)
    out = set()
    for (cx, cy, cz), members in cells.items():
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    other = cells.get((cx + dx, cy + dy, cz + dz))
                    if not other:
                        continue
                    for i in members:
                        for j in other:
                            if i < j:
                                d = pos[j] - pos[i]
                                d2 = float(np.float64(d[2]) * d[2] + (d[1] * d[1] + d[0] * d[0]))
                                s = b[i] + b[j]
                                # decide away from the boundary; leave near-ties to the oracle's exact rule
                                if d2 <= s * s * (1 - 1e-12):
                                    out.add((i, j))
                                elif d2 <= s * s * (1 + 1e-12):
                                    out.add((i, j, "tie"))
    return out


@pytest.mark.parametrize("n,mc,speed", [(2000, 1.5, 0.0), (3000, 3.0, 0.02), (500, 0.3, 0.0)])
def test_against_cell_list(n, mc, speed):
    w = wl.spheres(n, mean_contacts=mc, speed=speed)
    b = orc.bound_radius(w.vel, w.extra["radius"], 0.1)
    got = set(map(tuple, orc.broadphase(w.pos, b).tolist()))
    ref = cell_list_pairs(w.pos, b)
    sure = {p for p in ref if len(p) == 2}
    ties = {p[:2] for p in ref if len(p) == 3}
    assert sure <= got and got <= (sure | ties)
    assert abs(2 * len(got) / n - mc) < 0.5 * mc + 0.2 or speed > 0     # the recipe's mean contact number


# ------------------------------------------------------------------------------------------ O18
def test_aggregates_hand_graphs():
    # path 0-1-2-3, triangle 5-6-7, isolated 4 and 8, pair 9-10 given twice and a self pair
    pairs = [[0, 1], [2, 1], [2, 3], [5, 6], [7, 6], [5, 7], [9, 10], [10, 9], [8, 8]]
    r = orc.aggregates(11, pairs, mass=np.arange(11, dtype=np.float64))
    assert r["label"].tolist() == [0, 0, 0, 0, 4, 5, 5, 5, 8, 9, 9]
    assert r["size"].tolist() == [4, 0, 0, 0, 1, 3, 0, 0, 1, 2, 0]
    assert r["mass"].tolist() == [6.0, 0, 0, 0, 4.0, 18.0, 0, 0, 8.0, 19.0, 0]
    assert (r["components"], r["aggregates"]) == (5, 3)      # aggregates have more than one body
    # no contacts at all: every body is its own component, no aggregate
    r = orc.aggregates(4, np.zeros((0, 2), dtype=np.int32))
    assert r["label"].tolist() == [0, 1, 2, 3] and (r["components"], r["aggregates"]) == (4, 0)
    # star and chain in reverse order: the label is the smallest id whatever the edge order
    r = orc.aggregates(6, [[5, 4], [4, 3], [3, 2], [2, 1], [1, 0]])
    assert r["label"].tolist() == [0] * 6 and r["size"][0] == 6 and r["aggregates"] == 1
    with pytest.raises(ValueError):
        orc.aggregates(3, [[0, 3]])


def union_find_labels(n, pairs):
    parent = list(range(n))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x
    for a, b in pairs:
        ra, rb = find(a), find(b)
        if ra != rb:
            parent[max(ra, rb)] = min(ra, rb)
    return np.array([find(v) for v in range(n)])


@pytest.mark.parametrize("n,e,seed", [(1000, 400, 1), (5000, 5000, 2), (2000, 20000, 3), (50, 0, 4)])
def test_aggregates_against_scipy_and_union_find(n, e, seed):
    rng = np.random.default_rng(seed)
    pairs = rng.integers(0, n, size=(e, 2)).astype(np.int32)
    mass = rng.random(n)
    r = orc.aggregates(n, pairs, mass)
    g = coo_matrix((np.ones(e), (pairs[:, 0], pairs[:, 1])), shape=(n, n))
    nc, lab = connected_components(g, directed=False)
    assert r["components"] == nc
    # same partition, and the canonical label is the smallest member
    first = np.full(nc, n)
    np.minimum.at(first, lab, np.arange(n))
    assert np.array_equal(r["label"], first[lab])
    assert np.array_equal(r["label"], union_find_labels(n, pairs.tolist()))
    sizes = np.bincount(r["label"], minlength=n)
    assert np.array_equal(r["size"], sizes)
    assert r["aggregates"] == int((sizes > 1).sum())
    assert np.allclose(r["mass"], np.bincount(r["label"], weights=mass, minlength=n), rtol=1e-13, atol=0)


def test_broadphase_feeds_aggregates_percolation():
    # below the percolation threshold the largest aggregate is small, above it one aggregate dominates
    n = 4000
    sizes = []
    for mc in (0.5, 6.0):
        w = wl.spheres(n, mean_contacts=mc)
        p = orc.broadphase(w.pos, w.extra["radius"])
        sizes.append(orc.aggregates(n, p)["size"].max())
    assert sizes[0] < 0.02 * n and sizes[1] > 0.8 * n
