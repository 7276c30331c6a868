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
    bench.py times: tree bit-exact against the oracle; accelerations on sampled groups that the
    oracle can compute one by one; list lengths exact on those groups; totals consistent."""
    w = wl.make("c4")
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    assert_tree_equal(ctx, t)
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    assert np.isfinite(a).all()
    ng = t.ngroups
    assert gm.shape[0] == ng
    for g0 in list(range(0, ng, ng // 24))[:24] + [ng - 2]:
        ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G, g0, g0 + 2)
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 2]]
        assert np.array_equal(gm[g0:g0 + 2], nm) and np.array_equal(gd[g0:g0 + 2], nd)
        assert relerr(a[rows], ref[rows]).max() <= TOL
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


def test_eval_host_pageable_output_is_staged():
    """bh_eval_host with ordinary (pageable) host memory takes the staged path; with pinned memory, from the
    second call on and when a body has enough interactions (>= 3400), the walk stores straight into the output.
    All paths must give the same accelerations bit for bit."""
    w = wl.make("c4", 20000)
    theta = 0.2                                      # ~ 6000 interactions per body: the direct-store path is taken
    ctx = bh.Context(w.n, 16)
    pos_h, mass_h = torch.as_tensor(w.pos), torch.as_tensor(w.mass)
    out_page = torch.empty((w.n, 3), dtype=torch.float64)
    out_pin = torch.empty((w.n, 3), dtype=torch.float64).pin_memory()
    out_pin2 = torch.zeros((w.n, 3), dtype=torch.float64).pin_memory()
    bh.bh_eval_host(ctx.ctx, pos_h, mass_h, theta, w.eps, w.G, out_page)
    assert bh.bh_get_stats(ctx.ctx)["interactions"] / w.n >= 3400
    bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), theta, w.eps, w.G, out_pin)
    bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), theta, w.eps, w.G, out_pin2)
    assert np.array_equal(out_page.numpy(), out_pin.numpy()) and np.array_equal(out_page.numpy(), out_pin2.numpy())
    ref = orc.accel(orc.build(w.pos, w.mass, 16), theta, w.eps, w.G)[0]
    assert relerr(out_pin.numpy(), ref).max() <= TOL
    # few interactions per body (theta = 1): staged again, same contract
    bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), 1.0, w.eps, w.G, out_pin)
    bh.bh_eval_host(ctx.ctx, pos_h.pin_memory(), mass_h.pin_memory(), 1.0, w.eps, w.G, out_pin2)
    assert np.array_equal(out_pin.numpy(), out_pin2.numpy())
    assert relerr(out_pin.numpy(), orc.accel(orc.build(w.pos, w.mass, 16), 1.0, w.eps, w.G)[0]).max() <= TOL
    ctx.close()


def test_full_size_largest_config():
    """configs[4] at its full size (N = 4 194 304 rotating ball, C = 32, theta = 0.6): tree bit-exact, sampled
    groups against the oracle's walk, and the config's own check — the direct sum on random targets."""
    w = wl.make("c5")
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    ctx = gpu_build(w.pos, w.mass, w.leaf_cap)
    assert_tree_equal(ctx, t)
    a = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    gm, gd = (x.cpu().numpy().view(np.uint32) for x in ctx.counts())
    ng = t.ngroups
    for g0 in list(range(0, ng, ng // 12))[:12] + [ng - 2]:
        ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G, g0, g0 + 2)
        rows = t.perm[t.gstart[g0]:t.gstart[g0 + 2]]
        assert np.array_equal(gm[g0:g0 + 2], nm) and np.array_equal(gd[g0:g0 + 2], nd)
        assert relerr(a[rows], ref[rows]).max() <= TOL
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
