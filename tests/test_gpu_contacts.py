"""GPU parity for rows NEXT-3 / NEXT-4 of SURVEY.md 8(f): the tree-based broad phase against the oracle's
all-pairs definition (O17) — the SET of pairs must be identical (integer work: exact) — and the union-find
aggregate identification against the oracle's depth-first search (O18): labels, sizes and counts exact,
aggregate masses to rounding (atomic sums)."""
import numpy as np
import pytest
import torch

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import binding as bh
from paper_1912_04197_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def sorted_pairs(p):
    p = np.asarray(p, dtype=np.int32).reshape(-1, 2)
    return p[np.lexsort((p[:, 1], p[:, 0]))]


def gpu_pairs(pos, mass, radius, vel, dt, C):
    n = pos.shape[0]
    ctx = bh.Context(n, C)
    ctx.build(dev(pos), dev(mass))
    r, v = dev(radius), (dev(vel) if vel is not None else None)
    count = bh.bh_broadphase(ctx.ctx, r, v, dt, None)             # counting call
    buf = torch.full((max(count, 1), 2), -1, dtype=torch.int32, device="cuda")
    assert bh.bh_broadphase(ctx.ctx, r, v, dt, buf) == count
    ctx.close()
    return buf[:count].cpu().numpy()


@pytest.mark.parametrize("n,mc,speed,C", [(3000, 1.5, 0.0, 16), (20000, 3.0, 0.02, 16), (20000, 0.4, 0.0, 4),
                                           (5000, 8.0, 0.05, 32), (777, 2.0, 0.0, 1), (33, 2.0, 0.0, 16), (1, 1.0, 0.0, 8)])
def test_broadphase_pairs_exact(n, mc, speed, C):
    w = wl.spheres(n, mean_contacts=mc, speed=speed)
    dt = 0.1
    ref = orc.broadphase(w.pos, orc.bound_radius(w.vel, w.extra["radius"], dt))
    got = gpu_pairs(w.pos, w.mass, w.extra["radius"], w.vel, dt, C)
    assert (got[:, 0] < got[:, 1]).all() if len(got) else True
    assert np.array_equal(sorted_pairs(got), ref)                  # same set, each pair once


def test_broadphase_rubble_pile_radii():
    # configs[1]: power-law radii 5..50 m (ratio 10) in a 1 km ball, shrunk so that bodies touch
    w = wl.make("c2", 16384)
    pos = w.pos * 0.25
    ref = orc.broadphase(pos, w.extra["radius"])
    got = gpu_pairs(pos, w.mass, w.extra["radius"], None, 0.0, 16)
    assert len(ref) > 1000 and np.array_equal(sorted_pairs(got), ref)


def test_broadphase_lattice_touching_and_one_giant():
    # touching counts (<=): spacing 1, radii 1/2 -> exactly the face neighbours
    k = 12
    g = np.arange(k, dtype=np.float64)
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    n = k ** 3
    got = gpu_pairs(pos, np.ones(n), np.full(n, 0.5), None, 0.0, 8)
    assert len(got) == 3 * k * k * (k - 1)
    assert np.array_equal(sorted_pairs(got), orc.broadphase(pos, np.full(n, 0.5)))
    # one body whose sphere swallows the cloud: the largest radius in a node must reach the pruning test
    radius = np.full(n, 0.1)
    radius[n // 2] = 100.0
    got = gpu_pairs(pos, np.ones(n), radius, None, 0.0, 8)
    assert len(got) == n - 1 and np.array_equal(sorted_pairs(got), orc.broadphase(pos, radius))
    # a fast body: its swept sphere reaches everything
    vel = np.zeros((n, 3))
    vel[7] = [0.0, 300.0, 400.0]
    got = gpu_pairs(pos, np.ones(n), np.full(n, 0.1), vel, 0.2, 8)
    assert np.array_equal(sorted_pairs(got), orc.broadphase(pos, orc.bound_radius(vel, np.full(n, 0.1), 0.2)))
    assert len(got) == n - 1


def test_broadphase_capacity_and_state_errors():
    w = wl.spheres(4000, mean_contacts=3.0)
    ctx = bh.Context(4000, 16)
    r = dev(w.extra["radius"])
    with pytest.raises(bh.BhError) as ei:
        bh.bh_broadphase(ctx.ctx, r, None, 0.0, None)
    assert ei.value.status == bh.BH_ERR_STATE
    ctx.build(dev(w.pos), dev(w.mass))
    total = bh.bh_broadphase(ctx.ctx, r, None, 0.0, None)
    small = torch.full((total // 2, 2), -1, dtype=torch.int32, device="cuda")
    with pytest.raises(bh.BhError) as ei:
        bh.bh_broadphase(ctx.ctx, r, None, 0.0, small)
    assert ei.value.status == bh.BH_ERR_CAPACITY and ei.value.count == total
    ref = set(map(tuple, orc.broadphase(w.pos, w.extra["radius"]).tolist()))
    assert set(map(tuple, small.cpu().numpy().tolist())) <= ref      # what was written is valid
    ctx.close()


def gpu_aggregates(n, pairs, mass):
    ctx = bh.Context(n, 16)
    label = torch.empty(n, dtype=torch.int32, device="cuda")
    size = torch.empty(n, dtype=torch.int32, device="cuda")
    am = torch.empty(n, dtype=torch.float64, device="cuda")
    p = dev(pairs, torch.int32) if len(pairs) else None
    comps, aggs = bh.bh_aggregates(ctx.ctx, n, p, dev(mass), label, size, am)
    comps2, aggs2 = bh.bh_aggregates(ctx.ctx, n, p, None, label, None, None)      # labels only
    assert (comps, aggs) == (comps2, aggs2)
    ctx.close()
    return label.cpu().numpy(), size.cpu().numpy(), am.cpu().numpy(), comps, aggs


@pytest.mark.parametrize("n,e,seed", [(1000, 400, 1), (50000, 40000, 2), (20000, 200000, 3), (50, 0, 4), (1, 0, 5)])
def test_aggregates_random_graphs(n, e, seed):
    rng = np.random.default_rng(seed)
    pairs = rng.integers(0, n, size=(e, 2)).astype(np.int32)
    mass = rng.random(n)
    ref = orc.aggregates(n, pairs, mass)
    label, size, am, comps, aggs = gpu_aggregates(n, pairs, mass)
    assert np.array_equal(label, ref["label"]) and np.array_equal(size, ref["size"])
    assert (comps, aggs) == (ref["components"], ref["aggregates"])
    assert np.allclose(am, ref["mass"], rtol=1e-12, atol=0.0)


def test_aggregates_long_chain_and_bad_pair():
    n = 100000                                       # a path: the worst case for pointer chasing
    idx = np.random.default_rng(9).permutation(n).astype(np.int32)
    pairs = np.stack([idx[:-1], idx[1:]], axis=1)
    label, size, _, comps, aggs = gpu_aggregates(n, pairs, np.ones(n))
    assert (label == 0).all() and size[0] == n and (comps, aggs) == (1, 1)
    ctx = bh.Context(10, 8)
    lab = torch.empty(10, dtype=torch.int32, device="cuda")
    with pytest.raises(bh.BhError) as ei:
        bh.bh_aggregates(ctx.ctx, 10, dev(np.array([[0, 10]]), torch.int32), None, lab)
    assert ei.value.status == bh.BH_ERR_INVALID_ARG
    assert bh.bh_aggregates(ctx.ctx, 10, dev(np.array([[0, 9]]), torch.int32), None, lab) == (9, 1)   # flag does not stick
    ctx.close()


@pytest.mark.parametrize("mc", [0.5, 1.5, 6.0])
def test_broadphase_then_aggregates(mc):
    """The two rows chained as the paper chains them (contact container -> graph -> aggregates)."""
    n = 30000
    w = wl.spheres(n, mean_contacts=mc)
    ctx = bh.Context(n, 16)
    ctx.build(dev(w.pos), dev(w.mass))
    r = dev(w.extra["radius"])
    count = bh.bh_broadphase(ctx.ctx, r, None, 0.0, None)
    buf = torch.empty((max(count, 1), 2), dtype=torch.int32, device="cuda")
    bh.bh_broadphase(ctx.ctx, r, None, 0.0, buf)
    label = torch.empty(n, dtype=torch.int32, device="cuda")
    size = torch.empty(n, dtype=torch.int32, device="cuda")
    comps, aggs = bh.bh_aggregates(ctx.ctx, n, buf[:count], None, label, size, None)
    ref = orc.aggregates(n, orc.broadphase(w.pos, w.extra["radius"]))
    assert np.array_equal(label.cpu().numpy(), ref["label"]) and np.array_equal(size.cpu().numpy(), ref["size"])
    assert (comps, aggs) == (ref["components"], ref["aggregates"])
    ctx.close()


def test_degenerate_clouds_next_rows():
    """More coincident bodies than a leaf or a walk group holds (depth cap, R9): the potential counts every
    coincident neighbour (m/eps each) but never the body itself; the broad phase reports all their pairs."""
    rng = np.random.default_rng(12)
    pos = np.concatenate([np.full((70, 3), 0.25), rng.random((50, 3))])
    mass = rng.random(120) + 0.5
    radius = np.full(120, 1e-3)
    ctx = bh.Context(120, 4)
    ctx.build(dev(pos), dev(mass))
    t = orc.build(pos, mass, 4)
    for eps in (1e-2, 0.0):
        ref = orc.potential(t, 0.5, eps, 1.0)
        phi = ctx.potential(0.5, eps, 1.0).cpu().numpy()
        assert np.abs((phi - ref) / ref).max() <= 1e-11
        refd = orc.direct_potential(pos, mass, eps, 1.0)
        phid = ctx.direct_potential(eps, 1.0).cpu().numpy()
        assert np.abs((phid - refd) / refd).max() <= 1e-11
    ref = orc.broadphase(pos, radius)
    assert len(ref) >= 70 * 69 // 2
    cnt = bh.bh_broadphase(ctx.ctx, dev(radius), None, 0.0, None)
    buf = torch.empty((cnt, 2), dtype=torch.int32, device="cuda")
    bh.bh_broadphase(ctx.ctx, dev(radius), None, 0.0, buf)
    assert np.array_equal(sorted_pairs(buf.cpu().numpy()), ref)
    label = torch.empty(120, dtype=torch.int32, device="cuda")
    comps, aggs = bh.bh_aggregates(ctx.ctx, 120, buf, None, label)
    r = orc.aggregates(120, ref)
    assert (comps, aggs) == (r["components"], r["aggregates"]) and np.array_equal(label.cpu().numpy(), r["label"])
    ctx.close()


@pytest.mark.parametrize("n,C,speed,dt", [(2500, 1, 0.0, 0.0), (4000, 2, 3.0, 0.1), (3000, 16, 0.0, 0.0)])
def test_broadphase_non_local_search(n, C, speed, dt):
    """Bounding volumes that span a large part of the cloud (big radii, or fast bodies over a long step): the search
    is not local, most of a deep tree is near every group, and the node stack is held inside its bound by the pop
    rule (no overflow, no error), still the exact pair set."""
    w = wl.spheres(n, mean_contacts=2.0, speed=speed)
    radius = w.extra["radius"] * (1.0 if speed else 6.0)
    ref = orc.broadphase(w.pos, orc.bound_radius(w.vel if speed else None, radius, dt))
    got = gpu_pairs(w.pos, w.mass, radius, w.vel if speed else None, dt, C)
    assert len(ref) > 20 * n
    assert np.array_equal(sorted_pairs(got), ref)
