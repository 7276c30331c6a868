"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bit-exact: cube, sorted keys, permutation, node count, depth, level / begin / count / first_child /
child_mask / parent, monopoles, sorted bodies, group boxes, per-group list lengths.
Floating point: per-body accelerations, max_i |a_gpu - a_ref| / |a_ref| <= 1e-11 (north_star).
"""
import numpy as np
import pytest
import torch

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import binding as bh
from paper_1912_04197_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-11


def dev(a, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def relerr(a, b):
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


def gpu_build(pos, mass, C):
    ctx = bh.Context(pos.shape[0], C)
    ctx.build(dev(pos), dev(mass))
    return ctx


def assert_tree_equal(ctx, t):
    g = ctx.tree()
    assert g["lo"] == list(t.lo) and g["L"] == t.L
    assert np.array_equal(g["skey"].cpu().numpy().view(np.uint64), t.skey)
    assert np.array_equal(g["perm"].cpu().numpy().view(np.uint32), t.perm)
    assert (g["M"], g["depth"]) == (t.M, t.depth)
    assert np.array_equal(g["level"].cpu().numpy(), t.level)
    assert np.array_equal(g["begin"].cpu().numpy().view(np.uint32), t.begin)
    assert np.array_equal(g["count"].cpu().numpy().view(np.uint32), t.count)
    assert np.array_equal(g["first_child"].cpu().numpy(), t.first_child)
    assert np.array_equal(g["child_mask"].cpu().numpy(), t.child_mask)
    assert np.array_equal(g["parent"].cpu().numpy(), t.parent)
    assert np.array_equal(g["sbody"].cpu().numpy(), t.sbody)
    assert g["ng"] == t.ngroups and np.array_equal(g["gstart"].cpu().numpy().view(np.uint32), t.gstart)
    assert np.array_equal(g["glo"].cpu().numpy(), t.glo) and np.array_equal(g["ghi"].cpu().numpy(), t.ghi)
    # monopoles bit for bit (fixed summation order on both sides)
    assert np.array_equal(g["mono"].cpu().numpy().view(np.uint64), t.mono.view(np.uint64))


CASES = [("c1", 1024, 8), ("c1", 1000, 8), ("c1", 777, 1), ("c2", 16384, 16), ("c3", 20000, 16),
         ("c4", 50000, 16), ("c4", 4097, 2), ("c5", 40000, 32), ("c3", 33, 16), ("c3", 5, 16)]


@pytest.mark.parametrize("name,n,C", CASES)
def test_build_bit_exact(name, n, C):
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = gpu_build(w.pos, w.mass, C)
    assert_tree_equal(ctx, t)
    ctx.close()


@pytest.mark.parametrize("name,n,C", CASES)
def test_accel_counts_exact_and_values_within_tolerance(name, n, C):
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = gpu_build(w.pos, w.mass, C)
    for theta in ([w.theta] if name != "c3" else [0.0, 0.3, 0.7, 1.0]):
        ref, nm, nd, kappa = orc.accel(t, theta, w.eps, w.G, want_kappa=True)
        a = ctx.accel(theta, w.eps, w.G).cpu().numpy()
        gm, gd = ctx.counts()
        assert np.array_equal(gm.cpu().numpy().view(np.uint32), nm)
        assert np.array_equal(gd.cpu().numpy().view(np.uint32), nd)
        e = relerr(a, ref)
        worst = int(np.argmax(e))
        assert e.max() <= TOL, f"theta={theta}: max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g})"
        st = bh.bh_get_stats(ctx.ctx)
        assert st["n_mono"] == int(nm.sum()) and st["n_direct"] == int(nd.sum())
    ctx.close()


@pytest.mark.parametrize("name,n,C", [("c4", 4097, 16), ("c2", 6000, 16), ("c4", 30000, 1), ("c5", 100000, 32),
                                      ("c3", 148 * 1024, 16), ("c3", 148 * 1024 + 1, 16)])
def test_one_kernel_build_of_mid_size_sets_is_bit_exact(name, n, C):
    # 4096 < n <= 1024 bodies per SM: cube, keys, eight digit passes, gather, tree and monopoles in one co-resident
    # kernel with grid barriers (bh_mid.cu); one body more and the streaming kernels take over.  Same arrays, bit for bit;
    # a second build in the same context (the barrier words and the look-back rows are reused) gives them again.
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = gpu_build(w.pos, w.mass, C)
    l0 = bh.bh_get_launches(ctx.ctx)
    ctx.build(dev(w.pos), dev(w.mass))
    launches = bh.bh_get_launches(ctx.ctx) - l0
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    assert launches == (1 if n <= sms * 1024 else 14)     # cube, keys, sort x7, tree x3, gather + boxes, monopoles
    assert_tree_equal(ctx, t)
    ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G, 0, min(t.ngroups, 64))
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    rows = t.perm[: t.gstart[min(t.ngroups, 64)]]
    assert relerr(a[rows], ref[rows]).max() <= TOL
    ctx.close()


@pytest.mark.parametrize("n,dup", [(200000, 0), (200000, 40), (200000, 300), (600000, 300), (6000, 100), (20000, 40), (20000, 300)])
def test_partial_key_sort_and_its_fallback(n, dup):
    # Above 4096 bodies (one-kernel build and streaming sort alike) the sort passes only take the five high digits and a repair pass orders the runs of equal
    # top bits; `dup` coincident bodies share all 63 key bits: 40 are within the repair's reach (run <= 64), 300 raise the
    # flag and the co-resident fallback kernel sorts from scratch with eight digits.  Same permutation either way, and
    # the flag is not an error: the next synchronising call reports success.
    w = wl.make("c4", n)
    pos = w.pos.copy()
    if dup:
        rows = np.random.default_rng(7).choice(n, size=dup, replace=False)
        pos[rows] = pos[rows[0]]
    t = orc.build(pos, w.mass, 16)
    ctx = gpu_build(pos, w.mass, 16)
    assert_tree_equal(ctx, t)
    ctx.build(dev(pos), dev(w.mass))            # again in the same context (flag cleared, rows reused)
    assert_tree_equal(ctx, t)
    bh.bh_synchronize(ctx.ctx)
    ctx.close()


def test_two_contexts_build_mid_size_sets_at_the_same_time():
    # two co-resident kernels with their own grid barriers on two streams
    ws = [wl.make("c3", 20000), wl.make("c4", 50000)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs, ts = [], []
    for w, s in zip(ws, streams):
        ctxs.append(bh.Context(w.n, w.leaf_cap, stream=s))
        ts.append(orc.build(w.pos, w.mass, w.leaf_cap))
    bufs = [(dev(w.pos), dev(w.mass)) for w in ws]
    torch.cuda.synchronize()
    for rep in range(5):
        for ctx, (p, m) in zip(ctxs, bufs):
            ctx.build(p, m)
    torch.cuda.synchronize()
    for ctx, t in zip(ctxs, ts):
        assert_tree_equal(ctx, t)
        ctx.close()


def _tested_nodes_from_lists(t, theta):
    """Nodes the opening criterion is applied to, from the oracle's lists alone: every tested node is accepted
    (it is in a monopole list) or opened (it is a strict ancestor of a list entry, or a leaf whose bodies are in a
    direct list); the root is tested, and so is every child of an opened internal node."""
    leaves = np.where(t.first_child < 0)[0]
    order = np.argsort(t.begin[leaves])
    leaves, lbegin = leaves[order], t.begin[leaves][order]
    total = 0
    for g in range(t.ngroups):
        mono, direct = orc.walk_lists(t, g, theta)
        opened_leaves = np.unique(leaves[np.searchsorted(lbegin, direct, side="right") - 1]) if len(direct) else []
        opened = set(int(x) for x in opened_leaves)
        for x in list(mono) + list(opened_leaves):
            x = int(t.parent[int(x)])
            while x >= 0 and x not in opened:
                opened.add(x)
                x = int(t.parent[x])
        total += len(mono) + len(opened)
    return total


@pytest.mark.parametrize("name,n,C,theta", [("c4", 5000, 16, 0.5), ("c1", 1024, 8, 0.5), ("c3", 3000, 4, 0.0),
                                            ("c5", 4000, 32, 0.9)])
def test_tested_node_count_follows_from_the_oracle_lists(name, n, C, theta):
    # stats[3] is counted by the producer at every pop (all siblings of a popped range are tested)
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = gpu_build(w.pos, w.mass, C)
    ctx.accel(theta, w.eps, w.G)
    assert bh.bh_get_stats(ctx.ctx)["nodes_tested"] == _tested_nodes_from_lists(t, theta)
    ctx.close()


@pytest.mark.parametrize("name,n,C", [("c1", 1024, 8), ("c2", 16384, 16), ("c4", 5000, 16), ("c1", 300, 8)])
def test_direct_sum(name, n, C):
    w = wl.make(name, n)
    ref = orc.direct(w.pos, w.mass, w.eps, w.G)
    ctx = gpu_build(w.pos, w.mass, C)
    a = ctx.direct(w.eps, w.G).cpu().numpy()
    assert relerr(a, ref).max() <= TOL
    tg = np.random.default_rng(1).choice(n, size=min(n, 200), replace=False).astype(np.int32)
    b = ctx.direct(w.eps, w.G, targets=dev(tg, torch.int32)).cpu().numpy()
    assert relerr(b, ref[tg]).max() <= TOL
    ctx.close()


def test_degenerate_inputs():
    # one body; coincident bodies with eps = 0 (R13); more than C coincident bodies (depth cap, R9)
    for pos, mass, C in [
        (np.array([[1.0, 2.0, 3.0]]), np.array([2.0]), 8),
        (np.array([[0.0, 0, 0], [0.0, 0, 0], [1.0, 0, 0]]), np.ones(3), 1),
        (np.concatenate([np.full((20, 3), 0.3), np.random.default_rng(3).random((20, 3))]), np.ones(40), 4),
        (np.full((70, 3), -2.5), np.full(70, 0.5), 16),
    ]:
        t = orc.build(pos, mass, C)
        ctx = gpu_build(pos, mass, C)
        assert_tree_equal(ctx, t)
        ref, nm, nd, _ = orc.accel(t, 0.5, 0.0, 1.0)
        a = ctx.accel(0.5, 0.0, 1.0).cpu().numpy()
        gm, gd = ctx.counts()
        assert np.array_equal(gm.cpu().numpy().view(np.uint32), nm) and np.array_equal(gd.cpu().numpy().view(np.uint32), nd)
        assert np.isfinite(a).all()
        nz = np.linalg.norm(ref, axis=1) > 0
        assert np.array_equal(a[~nz], ref[~nz])
        if nz.any():
            assert relerr(a[nz], ref[nz]).max() <= TOL
        ctx.close()


def test_lattice_and_si_magnitudes():
    g = (np.arange(16) + 0.5) / 16
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    mass = np.full(len(pos), 1.0 / len(pos))
    for C in (1, 8):
        t = orc.build(pos, mass, C)
        ctx = gpu_build(pos, mass, C)
        assert_tree_equal(ctx, t)
        assert t.M == ((8 ** 5 - 1) // 7 if C == 1 else (8 ** 4 - 1) // 7)
        ctx.close()


def test_rebuild_reuses_context_and_smaller_n():
    ctx = bh.Context(20000, 16)
    for name, n in [("c4", 20000), ("c1", 1024), ("c3", 12345), ("c4", 20000)]:
        w = wl.make(name, n)
        t = orc.build(w.pos, w.mass, 16)
        ctx.build(dev(w.pos), dev(w.mass))
        assert_tree_equal(ctx, t)
        a = ctx.accel(0.5, 1e-3, 1.0).cpu().numpy()
        assert relerr(a, orc.accel(t, 0.5, 1e-3, 1.0)[0]).max() <= TOL
    ctx.close()


def test_kdk_steps_match_oracle_per_evaluation():
    """Per evaluation on bit-identical inputs: after s GPU steps the GPU positions
    go to the oracle, whose accelerations must match the GPU's; kick and drift are single fused
    multiply-adds and are checked bit for bit from the GPU's own accelerations."""
    w = wl.make("c4", 8192)
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    ctx = bh.Context(w.n, w.leaf_cap)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    p_prev, v_prev = w.pos.copy(), w.vel.copy()
    a_prev = orc.accel(orc.build(p_prev, w.mass, w.leaf_cap), w.theta, w.eps, w.G)[0]
    for step in range(3):
        bh.bh_kdk_step(ctx.ctx, w.dt)
        bh.bh_synchronize(ctx.ctx)
        p, v = pos.cpu().numpy(), vel.cpu().numpy()
        ctx.n = w.n
        a_gpu = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()          # same tree, same positions
        a_ref = orc.accel(orc.build(p, w.mass, w.leaf_cap), w.theta, w.eps, w.G)[0]
        assert relerr(a_gpu, a_ref).max() <= TOL
        # positions: x1 = fma(v_half, dt, x0) with v_half = fma(a0, dt/2, v0); velocities one more kick
        if step == 0:
            vh = v_prev.copy(); orc.kick(vh, a_prev, w.dt * 0.5)
            assert np.abs(vh - (v_prev + a_prev * w.dt * 0.5)).max() < 1e-12
            x1 = p_prev.copy(); orc.drift(x1, vh, w.dt)
            # a_prev is the oracle's, the GPU used its own (<=1e-11 apart): positions agree closely
            assert np.abs(p - x1).max() <= 1e-12 * max(1.0, np.abs(x1).max())
        p_prev, v_prev, a_prev = p, v, a_ref
    ctx.close()


def test_kdk_update_arithmetic_bit_exact():
    """theta=0-free check of the update kernels alone: with the GPU's own accelerations, kick and
    drift must equal the oracle's canonical fma updates bit for bit."""
    w = wl.make("c1", 2048)
    pos, vel, mass = dev(w.pos), dev(w.vel if w.vel is not None else np.zeros_like(w.pos)), dev(w.mass)
    ctx = bh.Context(w.n, 8)
    ctx.build(pos, mass)
    a0 = ctx.accel(0.5, w.eps, w.G).cpu().numpy()
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, 0.5, w.eps, w.G)
    bh.bh_kdk_step(ctx.ctx, 0.01)
    bh.bh_synchronize(ctx.ctx)
    v = np.zeros_like(w.pos); x = w.pos.copy()
    orc.kick(v, a0, 0.005); orc.drift(x, v, 0.01)
    assert np.array_equal(pos.cpu().numpy(), x)
    ctx.n = w.n
    a1 = ctx.accel(0.5, w.eps, w.G).cpu().numpy()
    orc.kick(v, a1, 0.005)
    assert np.array_equal(vel.cpu().numpy(), v)
    ctx.close()


def test_eval_host_end_to_end():
    w = wl.make("c3", 30000)
    ref = orc.accel(orc.build(w.pos, w.mass, 16), 0.5, w.eps, w.G)[0]
    ctx = bh.Context(w.n, 16)
    ph = torch.as_tensor(w.pos).pin_memory()
    mh = torch.as_tensor(w.mass).pin_memory()
    out = torch.empty((w.n, 3), dtype=torch.float64).pin_memory()
    bh.bh_eval_host(ctx.ctx, ph, mh, 0.5, w.eps, w.G, out)
    assert relerr(out.numpy(), ref).max() <= TOL
    ctx.close()


def test_error_reporting():
    ctx = bh.Context(1024, 8)
    acc = torch.empty((1024, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(bh.BhError) as e:
        bh.bh_accel(ctx.ctx, 0.5, 0.0, 1.0, acc)
    assert e.value.status == bh.BH_ERR_STATE
    with pytest.raises(bh.BhError) as e:
        bh.bh_kdk_step(ctx.ctx, 0.1)
    assert e.value.status == bh.BH_ERR_STATE
    w = wl.make("c1", 1024)
    with pytest.raises(bh.BhError) as e:
        bh.bh_build(ctx.ctx, dev(np.zeros((2048, 3))), dev(np.ones(2048)))
    assert e.value.status == bh.BH_ERR_INVALID_ARG
    ctx.build(dev(w.pos), dev(w.mass))
    with pytest.raises(bh.BhError) as e:
        bh.bh_accel(ctx.ctx, -0.5, 0.0, 1.0, acc)
    assert e.value.status == bh.BH_ERR_INVALID_ARG
    bad = w.pos.copy()
    bad[77, 1] = np.nan
    ctx.build(dev(bad), dev(w.mass))
    with pytest.raises(bh.BhError) as e:
        bh.bh_synchronize(ctx.ctx)
    assert e.value.status == bh.BH_ERR_NONFINITE
    ctx.build(dev(w.pos), dev(w.mass))          # the error is not sticky across builds
    bh.bh_synchronize(ctx.ctx)
    ctx.close()


def test_full_size_headline_config():
    """configs[3] at its full size (N = 1M Plummer, C=16, theta=0.5), in the launch configuration
    bench.py times: tree bit-exact against the oracle; accelerations of ALL bodies and the list lengths of
    ALL groups against the oracle's walk; totals consistent."""
    w = wl.make("c4")
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    assert_tree_equal(ctx, t)
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    assert np.isfinite(a).all()
    ng = t.ngroups
    assert gm.shape[0] == ng
    # north_star's target as stated: the maximum over ALL bodies.  The oracle walks every one of the ~36 000 groups
    # (about 10 s on 16 cores): list lengths of every group exactly, every body's acceleration within TOL.
    ref, nm, nd, kappa = orc.accel(t, w.theta, w.eps, w.G, want_kappa=True)
    assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
    e = relerr(a, ref)
    worst = int(e.argmax())
    assert e.max() <= TOL, f"max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g})"
    print(f"c4 all bodies: max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g}), median {np.median(e):.3e}")
    st = bh.bh_get_stats(ctx.ctx)
    assert st["n_mono"] == int(gm.astype(np.int64).sum()) and st["n_direct"] == int(gd.astype(np.int64).sum())
    assert st["interactions"] == int(((gm.astype(np.int64) + gd) * np.diff(t.gstart.astype(np.int64))).sum())
    # sampled direct-sum check (bh_direct_targets) against the oracle's direct sum on the same targets
    tg = np.random.default_rng(4).choice(w.n, size=64, replace=False).astype(np.int32)
    b = ctx.direct(w.eps, w.G, targets=dev(tg, torch.int32)).cpu().numpy()
    refd = orc.direct(w.pos, w.mass, w.eps, w.G, targets=tg)
    assert relerr(b, refd).max() <= TOL
    # Newton's third law over the whole tree result, to the size of the BH error
    net = (w.mass[:, None] * a).sum(axis=0)
    assert np.linalg.norm(net) < 1e-3 * (w.mass * np.linalg.norm(a, axis=1)).sum()
    ctx.close()


def test_eval_host_pageable_and_pinned_agree():
    """bh_eval_host: a pinned output is written by the walk kernel itself, a pageable one is staged and copied;
    nothing else decides the path.  Pageable and pinned buffers, first and later calls, many and few interactions
    per body all give the same accelerations bit for bit (no state is carried between calls)."""
    w = wl.make("c4", 20000)
    ctx = bh.Context(w.n, 16)
    pos_h, mass_h = torch.as_tensor(w.pos), torch.as_tensor(w.mass)
    for theta in (0.2, 1.0):
        out_page = torch.empty((w.n, 3), dtype=torch.float64)
        out_pin = torch.empty((w.n, 3), dtype=torch.float64).pin_memory()
        out_pin2 = torch.zeros((w.n, 3), dtype=torch.float64).pin_memory()
        bh.bh_eval_host(ctx.ctx, pos_h, mass_h, theta, w.eps, w.G, out_page)
        bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), theta, w.eps, w.G, out_pin)
        bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), theta, w.eps, w.G, out_pin2)
        assert np.array_equal(out_page.numpy(), out_pin.numpy()) and np.array_equal(out_page.numpy(), out_pin2.numpy())
        ref = orc.accel(orc.build(w.pos, w.mass, 16), theta, w.eps, w.G)[0]
        assert relerr(out_pin.numpy(), ref).max() <= TOL
    ctx.close()


def test_full_size_largest_config():
    """configs[4] at its full size (N = 4 194 304 rotating ball, C = 32, theta = 0.6): tree bit-exact, all
    groups and all bodies against the oracle's walk, and the config's own check — the direct sum on random targets."""
    w = wl.make("c5")
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    assert_tree_equal(ctx, t)
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    ng = t.ngroups
    assert gm.shape[0] == ng
    # every group, every body (the oracle's walk of all ~147 000 groups: about 20 s on 16 cores)
    ref, nm, nd, kappa = orc.accel(t, w.theta, w.eps, w.G, want_kappa=True)
    assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
    e = relerr(a, ref)
    worst = int(e.argmax())
    assert e.max() <= TOL, f"max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g})"
    print(f"c5 all bodies: max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g}), median {np.median(e):.3e}")
    tg = np.random.default_rng(5).choice(w.n, size=128, replace=False).astype(np.int32)
    b = ctx.direct(w.eps, w.G, targets=dev(tg, torch.int32)).cpu().numpy()
    refd = orc.direct(w.pos, w.mass, w.eps, w.G, targets=tg)
    assert relerr(b, refd).max() <= TOL
    # tree against direct on those targets: the size of the Barnes-Hut error at theta = 0.6 (median 7.5e-3)
    assert np.median(relerr(a[tg], refd)) < 3e-2
    ctx.close()


def test_headline_config_after_ten_kdk_steps():
    """configs[3] as BASELINE.json states it: 10 leapfrog steps at N = 1M with a rebuild every step.  Compared
    per evaluation on bit-identical inputs: the GPU's positions after step 10 go to the
    oracle; its tree must equal the GPU's last build bit for bit and its accelerations on sampled groups
    must match the accelerations the GPU's last step used."""
    w = wl.make("c4")
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    ctx = bh.Context(w.n, w.leaf_cap)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    for _ in range(w.steps):
        bh.bh_kdk_step(ctx.ctx, w.dt)
    bh.bh_synchronize(ctx.ctx)
    p = pos.cpu().numpy()
    assert np.isfinite(p).all() and np.abs(p - w.pos).max() > 0
    t = orc.build(p, w.mass, w.leaf_cap)
    ctx.n = w.n
    assert_tree_equal(ctx, t)                      # the tree of the last step's rebuild
    a = torch.empty((w.n, 3), dtype=torch.float64, device="cuda")
    bh.bh_copy_state_acc(ctx.ctx, a)
    a = a.cpu().numpy()
    ng = t.ngroups
    for g0 in list(range(0, ng, ng // 8))[:8]:
        ref = orc.accel(t, w.theta, w.eps, w.G, g0, g0 + 2)[0]
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 2]]
        assert relerr(a[rows], ref[rows]).max() <= TOL
    # the cloud is in equilibrium: ten steps of dt = 1e-3 move bodies by about |v| * 0.01
    assert np.abs(p - w.pos).max() < 0.05
    ctx.close()


# ---------------------------------------------------------------------------------------------------------
# configs[2] and configs[4] at their stated sizes
def test_c3_full_size_theta_sweep():
    """configs[2]: N = 131072 uniform ball, C = 16, theta in {0, 0.3, 0.5, 0.7, 1.0}.  Tree bit for bit; for
    theta >= 0.3 the list lengths of ALL groups and the accelerations of ALL bodies against the oracle; for
    theta = 0 (the oracle's walk is N^2 in long double) the lists of all groups by the property that fixes them
    (theta = 0 is the direct sum: no node is accepted, every body is a source) and the accelerations
    of 64 groups spread over the cloud, against the oracle's walk and against its direct sum (Eq. (1))."""
    w = wl.make("c3")
    assert w.n == 131072 and w.leaf_cap == 16
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    assert_tree_equal(ctx, t)
    sizes = np.diff(t.gstart.astype(np.int64))
    inter_prev = None
    for theta in (0.3, 0.5, 0.7, 1.0):
        ref, nm, nd, kappa = orc.accel(t, theta, w.eps, w.G, want_kappa=True)
        a = ctx.accel(theta, w.eps, w.G).cpu().numpy()
        gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
        assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
        e = relerr(a, ref)
        worst = int(np.argmax(e))
        assert e.max() <= TOL, f"theta={theta}: max rel err {e.max():.3e} at body {worst} (kappa {kappa[worst]:.3g})"
        st = bh.bh_get_stats(ctx.ctx)
        inter = int(((nm.astype(np.int64) + nd) * sizes).sum())
        assert st["interactions"] == inter
        assert inter_prev is None or inter < inter_prev          # fewer interactions as theta grows
        inter_prev = inter
    # theta = 0
    a0 = ctx.accel(0.0, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    assert not gm.any() and (gd == w.n).all()
    st = bh.bh_get_stats(ctx.ctx)
    assert st["interactions"] == w.n * w.n and st["n_mono"] == 0
    ng = t.ngroups
    picks = np.unique(np.linspace(0, ng - 1, 64).astype(np.int64))
    rows_all = []
    for g0 in picks:
        ref, nm, nd, _ = orc.accel(t, 0.0, w.eps, w.G, int(g0), int(g0) + 1)
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 1]]
        assert nm[0] == 0 and nd[0] == w.n
        assert relerr(a0[rows], ref[rows]).max() <= TOL
        rows_all.append(rows)
    rows_all = np.concatenate(rows_all).astype(np.int32)
    refd = orc.direct(w.pos, w.mass, w.eps, w.G, targets=rows_all)
    assert relerr(a0[rows_all], refd).max() <= 1e-13             # "equivalent to direct": same terms, other order
    # the direct kernel on the same targets
    b = ctx.direct(w.eps, w.G, targets=dev(rows_all, torch.int32)).cpu().numpy()
    assert relerr(b, refd).max() <= TOL
    ctx.close()


def test_c5_after_fifty_kdk_steps():
    """configs[4] as BASELINE.json states it: 50 leapfrog steps at N = 4 194 304, tree rebuilt every step
    (PAPER.md:62).  Per evaluation on bit-identical inputs: the GPU's positions after step 50 go
    to the oracle; its tree must equal the GPU's last build bit for bit, and its accelerations and list lengths
    on sampled groups must match those of the GPU's last evaluation."""
    w = wl.make("c5")
    assert w.n == 4194304 and w.steps == 50
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    ctx = bh.Context(w.n, w.leaf_cap)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    for _ in range(w.steps):
        bh.bh_kdk_step(ctx.ctx, w.dt)
    bh.bh_synchronize(ctx.ctx)
    p = pos.cpu().numpy()
    assert np.isfinite(p).all() and np.abs(p - w.pos).max() > 0
    t = orc.build(p, w.mass, w.leaf_cap)
    ctx.n = w.n
    assert_tree_equal(ctx, t)
    a = torch.empty((w.n, 3), dtype=torch.float64, device="cuda")
    bh.bh_copy_state_acc(ctx.ctx, a)
    a = a.cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    ng = t.ngroups
    for g0 in list(range(0, ng, ng // 12))[:12] + [ng - 2]:
        ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G, g0, g0 + 2)
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 2]]
        assert np.array_equal(gm[g0:g0 + 2], nm) and np.array_equal(gd[g0:g0 + 2], nd)
        assert relerr(a[rows], ref[rows]).max() <= TOL
    ctx.close()


def test_scale_16m_bodies():
    """Beyond the largest BASELINE.json configuration: configs[4]'s cloud at N = 16 777 216 (7 GB of workspace; the
    arrays no longer fit the L2, 4096 sort tiles per pass, 590 000 groups).  Tree bit for bit, sampled groups
    against the oracle's walk, the walk's totals consistent with the per-group counts."""
    w = wl.make("c5", 16777216)
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    g = ctx.tree()
    assert g["lo"] == list(t.lo) and g["L"] == t.L and (g["M"], g["depth"]) == (t.M, t.depth)
    for key, ref, view in [("skey", t.skey, np.uint64), ("perm", t.perm, np.uint32), ("begin", t.begin, np.uint32),
                           ("count", t.count, np.uint32), ("gstart", t.gstart, np.uint32)]:
        assert np.array_equal(g[key].cpu().numpy().view(view), ref), key
    for key, ref in [("level", t.level), ("first_child", t.first_child), ("child_mask", t.child_mask), ("parent", t.parent)]:
        assert np.array_equal(g[key].cpu().numpy(), ref), key
    assert np.array_equal(g["mono"].cpu().numpy().view(np.uint64), t.mono.view(np.uint64))
    assert np.array_equal(g["glo"].cpu().numpy(), t.glo) and np.array_equal(g["ghi"].cpu().numpy(), t.ghi)
    del g
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    ng = t.ngroups
    for g0 in list(range(0, ng, ng // 6))[:6] + [ng - 2]:
        ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G, g0, g0 + 2)
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 2]]
        assert np.array_equal(gm[g0:g0 + 2], nm) and np.array_equal(gd[g0:g0 + 2], nd)
        assert relerr(a[rows], ref[rows]).max() <= TOL
    st = bh.bh_get_stats(ctx.ctx)
    assert st["interactions"] == int(((gm.astype(np.int64) + gd) * np.diff(t.gstart.astype(np.int64))).sum())
    ctx.close()


@pytest.mark.parametrize("name,n,C,theta,sampled", [("c4", 30000, 1, 0.1, False), ("c3", 131072, 4, 0.0, True),
                                                     ("c4", 100000, 1, 0.0, True)])
def test_stack_spill_path(name, n, C, theta, sampled):
    """Traversals whose LIFO stack of sibling ranges outgrows the 512 entries held in shared memory spill 128
    entries at a time to the workspace and refill from it (deep trees, small theta: everything is opened).  The
    spill counter of bh_get_stats proves the path ran; lists and accelerations must still equal the oracle's."""
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = gpu_build(w.pos, w.mass, C)
    assert_tree_equal(ctx, t)
    a = ctx.accel(theta, w.eps, w.G).cpu().numpy()
    st = bh.bh_get_stats(ctx.ctx)
    assert st["stack_spills"] > 0, "the walk's stack-spill path was not reached"
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    if theta == 0.0:
        assert not gm.any() and (gd == n).all() and st["interactions"] == n * n
    ng = t.ngroups
    groups = np.unique(np.linspace(0, ng - 1, 48).astype(np.int64)) if sampled else [None]
    for g0 in groups:
        if g0 is None:
            ref, nm, nd, _ = orc.accel(t, theta, w.eps, w.G)
            assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
            assert relerr(a, ref).max() <= TOL
        else:
            g0 = int(g0)
            ref, nm, nd, _ = orc.accel(t, theta, w.eps, w.G, g0, g0 + 1)
            rows = t.perm[t.gstart[g0]:t.gstart[g0 + 1]]
            assert gm[g0] == nm[0] and gd[g0] == nd[0]
            assert relerr(a[rows], ref[rows]).max() <= TOL
    ctx.close()


# ---------------------------------------------------------------------------------------------------------
# the grouping parameters of reading R6 are the oracle's: the CUDA path follows them at other values too
@pytest.mark.parametrize("name,n,C,W,Gc", [("c4", 20000, 16, 32, 64), ("c3", 9000, 16, 8, 512), ("c1", 3000, 8, 1, 512),
                                           ("c4", 5000, 4, 5, 20), ("c5", 12000, 32, 32, 2048), ("c2", 4000, 1, 1, 1)])
def test_group_parameters_follow_the_oracle(name, n, C, W, Gc):
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C, W=W, Gc=Gc)
    ctx = bh.Context(n, C, group_size=W, group_cell=Gc)
    ctx.build(dev(w.pos), dev(w.mass))
    assert_tree_equal(ctx, t)
    for theta in (0.5, 0.9):
        ref, nm, nd, _ = orc.accel(t, theta, w.eps, w.G)
        a = ctx.accel(theta, w.eps, w.G).cpu().numpy()
        gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
        assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
        assert relerr(a, ref).max() <= TOL
    ctx.close()


def test_per_body_walk_is_the_papers_and_group_walk_opens_a_superset():
    """W = 1, C = 1 on the GPU is the paper's own tree and walk.  The group reading R6
    (W = 32) accepts a node only if every member's own test accepts it, so per body it evaluates at least the
    interactions of the per-body walk, and is at least as close to the direct sum on average."""
    w = wl.make("c1", 2000)
    pos, mass = dev(w.pos), dev(w.mass)
    one = bh.Context(w.n, 1, group_size=1)
    one.build(pos, mass)
    t1 = orc.build(w.pos, w.mass, 1, W=1)
    assert_tree_equal(one, t1)
    a1 = one.accel(0.5, w.eps, w.G).cpu().numpy()
    ref1, nm1, nd1, _ = orc.accel(t1, 0.5, w.eps, w.G)
    g1m, g1d = (x.cpu().numpy().view(np.uint32) for x in one.counts())
    assert np.array_equal(g1m, nm1) and np.array_equal(g1d, nd1)
    assert relerr(a1, ref1).max() <= TOL
    grp = bh.Context(w.n, 1)
    grp.build(pos, mass)
    a32 = grp.accel(0.5, w.eps, w.G).cpu().numpy()
    i1 = bh.bh_get_stats(one.ctx)["interactions"]
    i32 = bh.bh_get_stats(grp.ctx)["interactions"]
    assert i32 >= i1
    d = orc.direct(w.pos, w.mass, w.eps, w.G)
    assert np.median(relerr(a32, d)) <= np.median(relerr(a1, d))
    one.close()
    grp.close()


# ---------------------------------------------------------------------------------------------------------
# the documented range of the input (include/bh.h)
@pytest.mark.parametrize("k", [-300, -150, 150, 299])
def test_extreme_scales(k):
    """Positions and masses scaled by 2^k (accelerations then scale by 2^-k; m x and m / r^3 stay far from the ends
    of the exponent range, as bh.h asks): the keys, the tree and the list lengths do not change (power-of-two
    scalings are exact), the monopoles scale exactly, and the accelerations match the oracle at the scaled
    inputs.  k = -300 and 299 are the edges of the documented extent range."""
    w = wl.make("c3", 6000)
    t0 = orc.build(w.pos, w.mass, 16)
    sc = float(np.ldexp(1.0, k))
    pos, mass, eps = w.pos * sc, w.mass * sc, w.eps * sc
    t = orc.build(pos, mass, 16)
    assert np.array_equal(t.skey, t0.skey) and np.array_equal(t.gstart, t0.gstart) and t.M == t0.M
    assert np.array_equal(t.mono, t0.mono * sc)
    ctx = gpu_build(pos, mass, 16)
    assert_tree_equal(ctx, t)
    for theta in (0.0, 0.5, 1.0):
        ref, nm, nd, _ = orc.accel(t, theta, eps, w.G)
        a = ctx.accel(theta, eps, w.G).cpu().numpy()
        gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
        assert np.array_equal(gm, nm) and np.array_equal(gd, nd)
        assert np.isfinite(a).all() and relerr(a, ref).max() <= TOL
    ctx.close()


def test_extent_outside_documented_range_is_reported():
    w = wl.make("c1", 500)
    ctx = bh.Context(w.n, 8)
    for k in (-320, 320):
        ctx.build(dev(w.pos * float(np.ldexp(1.0, k))), dev(w.mass))
        with pytest.raises(bh.BhError) as e:
            bh.bh_synchronize(ctx.ctx)
        assert e.value.status == bh.BH_ERR_INVALID_ARG and "extent" in str(e.value)
    ctx.build(dev(w.pos), dev(w.mass))
    bh.bh_synchronize(ctx.ctx)
    ctx.close()


def test_tiny_softening_is_treated_as_none():
    """0 < eps^2 < smallest normal double: the self term and coincident pairs have a subnormal softened distance;
    they must contribute nothing (bh.h), exactly as with eps = 0 — not infinity times zero."""
    rng = np.random.default_rng(11)
    pos = np.concatenate([rng.random((300, 3)), np.full((5, 3), 0.5)])
    mass = np.full(len(pos), 1.0 / len(pos))
    ctx = gpu_build(pos, mass, 4)
    a0 = ctx.accel(0.5, 0.0, 1.0).cpu().numpy()
    a1 = ctx.accel(0.5, 1e-160, 1.0).cpu().numpy()
    d0 = ctx.direct(0.0, 1.0).cpu().numpy()
    d1 = ctx.direct(1e-160, 1.0).cpu().numpy()
    assert np.isfinite(a1).all() and np.array_equal(a0, a1) and np.array_equal(d0, d1)
    ref = orc.accel(orc.build(pos, mass, 4), 0.5, 1e-160, 1.0)[0]
    assert relerr(a1, ref).max() <= TOL
    ctx.close()


def test_device_errors_are_sticky_until_reported():
    """A non-finite coordinate seen by one build is reported by the next synchronising call even if another,
    clean, build ran in between; once reported it is cleared (bh.h)."""
    w = wl.make("c1", 1024)
    bad = w.pos.copy()
    bad[5, 0] = np.inf
    ctx = bh.Context(w.n, 8)
    ctx.build(dev(bad), dev(w.mass))
    ctx.build(dev(w.pos), dev(w.mass))
    with pytest.raises(bh.BhError) as e:
        bh.bh_synchronize(ctx.ctx)
    assert e.value.status == bh.BH_ERR_NONFINITE
    bh.bh_synchronize(ctx.ctx)
    ctx.build(dev(w.pos), dev(w.mass))
    assert_tree_equal(ctx, orc.build(w.pos, w.mass, 8))
    ctx.close()
