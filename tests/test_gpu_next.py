"""GPU parity for the rows "next" of SURVEY.md 8(f) (NEXT-1, NEXT-2): tree / direct potential, conserved
quantities, Eq. (7) position error, semi-implicit Euler and two-rate stepping, against the CPU oracle
(O12-O16 of oracle/bh_oracle.c) on the same seeded inputs.

Bit-exact: Eq. (7) maximum (canonical arithmetic), the updates of the steppers given the same
accelerations, the two-rate step against n_sub separate updates.  Floating point: potential within
1e-11 relative per body (the bound north_star sets for accelerations); conserved quantities within
1e-15 of the sum of |terms| (they cancel, so a relative bound on the result would be meaningless).
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


@pytest.mark.parametrize("name,n,C", [("c1", 1024, 8), ("c2", 16384, 16), ("c4", 30000, 16), ("c3", 777, 1),
                                       ("c5", 20000, 32), ("c3", 5, 16)])
def test_tree_potential(name, n, C):
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = bh.Context(n, C)
    ctx.build(dev(w.pos), dev(w.mass))
    for theta in (w.theta, 0.0) if n <= 20000 else (w.theta,):
        ref = orc.potential(t, theta, w.eps, w.G)
        phi = ctx.potential(theta, w.eps, w.G).cpu().numpy()
        assert np.abs(phi - ref).max() <= TOL * np.abs(ref).min(), (theta, np.abs((phi - ref) / ref).max())
        # the lists are those of the acceleration walk
        _, nm, nd, _ = orc.accel(t, theta, w.eps, w.G, 0, 1)
        gm, gd = ctx.counts()
        assert gm[0].item() == nm[0] and gd[0].item() == nd[0]
    ctx.close()


@pytest.mark.parametrize("name,n,C", [("c1", 1024, 8), ("c2", 16384, 16), ("c4", 3001, 16)])
def test_direct_potential(name, n, C):
    w = wl.make(name, n)
    ref = orc.direct_potential(w.pos, w.mass, w.eps, w.G)
    ctx = bh.Context(n, C)
    ctx.build(dev(w.pos), dev(w.mass))
    phi = ctx.direct_potential(w.eps, w.G).cpu().numpy()
    assert np.abs((phi - ref) / ref).max() <= TOL
    ctx.close()


def test_potential_coincident_bodies_eps0():
    # R13/R24: a pair at zero softened distance adds nothing; a lone body has potential 0
    pos = np.array([[0.0, 0, 0], [0.0, 0, 0], [2.0, 0, 0]])
    mass = np.array([1.0, 3.0, 5.0])
    ctx = bh.Context(3, 1)
    ctx.build(dev(pos), dev(mass))
    for phi in (ctx.potential(0.5, 0.0, 1.0).cpu().numpy(), ctx.direct_potential(0.0, 1.0).cpu().numpy()):
        assert np.allclose(phi, np.array([-2.5, -2.5, -2.0]), rtol=1e-14, atol=0.0)
    ctx.close()
    ctx = bh.Context(1, 4)
    ctx.build(dev(np.array([[1.0, 2.0, 3.0]])), dev(np.array([7.0])))
    assert ctx.potential(0.5, 0.0, 1.0).item() == 0.0 and ctx.direct_potential(0.0, 1.0).item() == 0.0
    ctx.close()


def _sum_abs_terms(pos, vel, mass, phi):
    m = mass[:, None]
    lx = np.abs(pos[:, [1, 2, 0]] * vel[:, [2, 0, 1]]) + np.abs(pos[:, [2, 0, 1]] * vel[:, [1, 2, 0]])
    return dict(ekin=(0.5 * mass * (vel ** 2).sum(1)).sum(), epot=np.abs(0.5 * mass * phi).sum(),
                P=np.abs(m * vel).sum(0), L=(m * lx).sum(0))


@pytest.mark.parametrize("name,n", [("c4", 100000), ("c5", 65537), ("c1", 1024), ("c4", 1)])
def test_diagnostics(name, n):
    w = wl.make(name, n)
    rng = np.random.default_rng(7)
    if w.vel is None:
        w.vel = rng.standard_normal((n, 3))
    phi = -rng.random(n) - 0.1
    ctx = bh.Context(n, 16)
    ref = orc.diagnostics(w.pos, w.vel, w.mass, phi)
    scale = _sum_abs_terms(w.pos, w.vel, w.mass, phi)
    d1 = bh.bh_diagnostics(ctx.ctx, dev(w.pos), dev(w.vel), dev(w.mass), dev(phi))
    d2 = bh.bh_diagnostics(ctx.ctx, dev(w.pos), dev(w.vel), dev(w.mass), dev(phi))
    assert d1 == d2                                    # fixed reduction order: reproducible bit for bit
    for k in ("ekin", "epot"):
        assert abs(d1[k] - ref[k]) <= 1e-15 * scale[k] + 1e-300
    for k in ("P", "L"):
        assert (np.abs(np.array(d1[k]) - ref[k]) <= 1e-15 * scale[k] + 1e-300).all()
    d0 = bh.bh_diagnostics(ctx.ctx, dev(w.pos), dev(w.vel), dev(w.mass), None)
    assert d0["epot"] == 0.0 and d0["ekin"] == d1["ekin"]
    ctx.close()


def test_diagnostics_exact_cancellation():
    # momentum of +-v pairs cancels to ~2^-100 of the sum of |terms| (double-double accumulation), where a
    # plain fp64 sum of terms spanning 16 decades would keep nothing
    rng = np.random.default_rng(11)
    n = 50000
    v = rng.standard_normal((n, 3)) * 10.0 ** rng.integers(-8, 8, (n, 1))
    x = rng.standard_normal((n, 3))
    pos, vel, mass = np.concatenate([x, x]), np.concatenate([v, -v]), np.full(2 * n, 0.37)
    ctx = bh.Context(2 * n, 16)
    d = bh.bh_diagnostics(ctx.ctx, dev(pos), dev(vel), dev(mass), None)
    sc = _sum_abs_terms(pos, vel, mass, np.zeros(2 * n))
    assert (np.abs(d["P"]) <= 1e-28 * sc["P"]).all() and (np.abs(d["L"]) <= 1e-28 * sc["L"]).all()
    ctx.close()


@pytest.mark.parametrize("n", [1, 33, 100000])
def test_position_error_bit_exact(n):
    rng = np.random.default_rng(n)
    ref = rng.standard_normal((n, 3))
    pos = ref + 1e-6 * rng.standard_normal((n, 3))
    if n > 10:
        ref[3] = 0.0            # R25: skipped
        pos[5] = ref[5]         # zero error
    ctx = bh.Context(n, 16)
    e = bh.bh_position_error(ctx.ctx, dev(pos), dev(ref))
    assert e == orc.position_error(pos, ref)
    assert bh.bh_position_error(ctx.ctx, dev(ref), dev(ref)) == 0.0
    ctx.close()


def test_gravity_dt():
    for G, rho in [(6.674e-11, 3000.0), (1.0, 0.24), (6.674e-11, 2000.0)]:
        assert bh.bh_gravity_dt(G, rho) == orc.gravity_dt(G, rho)


@pytest.mark.parametrize("name,n,C", [("c4", 20000, 16), ("c5", 10000, 32)])
def test_euler_and_multirate_steps(name, n, C):
    """Per evaluation on bit-identical inputs: the oracle advances from the GPU's own
    positions of the previous step; accelerations within 1e-11, and the update itself bit-exact when fed
    the GPU's accelerations."""
    w = wl.make(name, n)
    dt = 1e-3
    ctx = bh.Context(n, C)
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    for kind, n_sub in (("euler", 1), ("multirate", 5), ("euler", 1)):
        p0, v0 = pos.cpu().numpy().copy(), vel.cpu().numpy().copy()
        if kind == "euler":
            bh.bh_euler_step(ctx.ctx, dt)
        else:
            bh.bh_multirate_step(ctx.ctx, dt, n_sub)
        bh.bh_synchronize(ctx.ctx)
        # the accelerations the step used: a(x_k)
        a_dev = torch.empty((n, 3), dtype=torch.float64, device="cuda")
        bh.bh_copy_state_acc(ctx.ctx, a_dev)
        a_gpu = a_dev.cpu().numpy()
        t = orc.build(p0, w.mass, C)
        a_ref = orc.accel(t, w.theta, w.eps, w.G)[0]
        e = np.linalg.norm(a_gpu - a_ref, axis=1) / np.linalg.norm(a_ref, axis=1)
        assert e.max() <= TOL
        # oracle update from the GPU's accelerations: bit for bit
        pr, vr = p0.copy(), v0.copy()
        for _ in range(n_sub):
            orc.kick(vr, a_gpu, dt)
            orc.drift(pr, vr, dt)
        assert np.array_equal(vel.cpu().numpy(), vr) and np.array_equal(pos.cpu().numpy(), pr)
        # and the whole oracle step (its own accelerations) agrees to the tolerance of the accelerations
        s = orc.Stepper(p0, v0, w.mass, w.theta, w.eps, w.G, C)
        s.euler(dt) if kind == "euler" else s.multirate(dt, n_sub)
        assert np.abs(vel.cpu().numpy() - s.vel).max() <= TOL * np.abs(a_ref).max() * dt * n_sub * 10
    ctx.close()


def test_stepper_state_errors():
    ctx = bh.Context(100, 8)
    with pytest.raises(bh.BhError) as ei:
        bh.bh_euler_step(ctx.ctx, 1e-3)
    assert ei.value.status == bh.BH_ERR_STATE
    w = wl.make("c1", 100)
    pos, vel, mass = dev(w.pos), dev(np.zeros((100, 3))), dev(w.mass)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, 0.5, 1e-3, 1.0)
    with pytest.raises(bh.BhError) as ei:
        bh.bh_multirate_step(ctx.ctx, 1e-3, 0)
    assert ei.value.status == bh.BH_ERR_INVALID_ARG
    # Euler then KDK: the KDK step re-evaluates a(x) (the Euler step leaves a(x_k) behind).  Checked per evaluation on
    # the GPU's own positions (never trajectory against trajectory): one kick + drift from the oracle's
    # a(p0) must give the GPU's new positions to what 1e-11 on the accelerations allows, and the stale a(x_k) must not.
    dt = 1e-3
    p_before = pos.cpu().numpy().copy()
    bh.bh_euler_step(ctx.ctx, dt)
    bh.bh_synchronize(ctx.ctx)
    p0, v0 = pos.cpu().numpy().copy(), vel.cpu().numpy().copy()
    bh.bh_kdk_step(ctx.ctx, dt)
    bh.bh_synchronize(ctx.ctx)
    p1 = pos.cpu().numpy()

    def drifted(a):
        vh = v0.copy(); orc.kick(vh, a, dt * 0.5)
        x = p0.copy(); orc.drift(x, vh, dt)
        return x
    a0 = orc.accel(orc.build(p0, w.mass, 8), 0.5, 1e-3, 1.0)[0]
    a_stale = orc.accel(orc.build(p_before, w.mass, 8), 0.5, 1e-3, 1.0)[0]
    tol_x = TOL * np.abs(a0).max() * dt * dt * 0.5 + 2 * np.finfo(float).eps * np.abs(p1).max()
    assert np.abs(p1 - drifted(a0)).max() <= tol_x
    assert np.abs(p1 - drifted(a_stale)).max() > 10 * tol_x
    ctx.close()


def test_steppers_with_direct_gravity():
    """bh_set_gravity_method(1): the steppers evaluate Eq. (1) directly, no tree."""
    w = wl.make("c1", 600)
    rng = np.random.default_rng(5)
    v0 = 0.1 * rng.standard_normal((600, 3))
    ctx = bh.Context(600, 8)
    pos, vel, mass = dev(w.pos), dev(v0), dev(w.mass)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    bh.bh_set_gravity_method(ctx.ctx, 1)
    # per evaluation, on the GPU's own positions: after every step the accelerations the context holds
    # are Eq. (1) at the new positions within TOL, and the update is the canonical kick / drift / kick of the GPU's own
    # accelerations, bit for bit (the first step's a(x0) is not kept: the oracle's stands in, to what TOL allows)
    dt = 1e-3
    a = torch.empty((600, 3), dtype=torch.float64, device="cuda")
    a_prev = None
    for step in range(3):
        p_prev, v_prev = pos.cpu().numpy().copy(), vel.cpu().numpy().copy()
        bh.bh_kdk_step(ctx.ctx, dt)
        bh.bh_copy_state_acc(ctx.ctx, a)
        bh.bh_synchronize(ctx.ctx)
        p, v, a_gpu = pos.cpu().numpy(), vel.cpu().numpy(), a.cpu().numpy().copy()
        ref = orc.direct(p, w.mass, w.eps, w.G)
        assert (np.linalg.norm(a_gpu - ref, axis=1) / np.linalg.norm(ref, axis=1)).max() <= TOL
        first = a_prev is None
        if first:
            a_prev = orc.direct(p_prev, w.mass, w.eps, w.G)
        vh = v_prev.copy(); orc.kick(vh, a_prev, dt * 0.5)
        x = p_prev.copy(); orc.drift(x, vh, dt)
        v1 = vh.copy(); orc.kick(v1, a_gpu, dt * 0.5)
        if first:
            amax = np.abs(a_prev).max()
            assert np.abs(p - x).max() <= TOL * amax * dt * dt * 0.5 + 2 * np.finfo(float).eps * np.abs(x).max()
            assert np.abs(v - v1).max() <= TOL * amax * dt + 2 * np.finfo(float).eps * np.abs(v1).max()
        else:
            assert np.array_equal(p, x) and np.array_equal(v, v1)
        a_prev = a_gpu
    # no tree after a direct evaluation
    with pytest.raises(bh.BhError) as ei:
        ctx.n = 600
        ctx.accel(0.5, 1e-3, 1.0)
    assert ei.value.status == bh.BH_ERR_STATE
    # Euler with direct gravity (the context then holds a(x_k) at the positions the step started from), then back to the tree
    p0, v0 = pos.cpu().numpy().copy(), vel.cpu().numpy().copy()
    bh.bh_euler_step(ctx.ctx, dt)
    bh.bh_copy_state_acc(ctx.ctx, a)
    bh.bh_synchronize(ctx.ctx)
    a_gpu = a.cpu().numpy()
    ref = orc.direct(p0, w.mass, w.eps, w.G)
    assert (np.linalg.norm(a_gpu - ref, axis=1) / np.linalg.norm(ref, axis=1)).max() <= TOL
    v1 = v0.copy(); orc.kick(v1, a_gpu, dt)
    x1 = p0.copy(); orc.drift(x1, v1, dt)
    assert np.array_equal(vel.cpu().numpy(), v1) and np.array_equal(pos.cpu().numpy(), x1)
    bh.bh_set_gravity_method(ctx.ctx, 0)
    bh.bh_euler_step(ctx.ctx, 1e-3)
    bh.bh_synchronize(ctx.ctx)
    assert bh.bh_get_node_count(ctx.ctx)[0] > 1
    ctx.close()


@pytest.mark.parametrize("n,method", [(3000, 0), (500, 1), (40000, 0), (6000, 0), (200000, 0)])
def test_cuda_graph_steppers_bit_identical(n, method):
    """bh_set_graph: captured / replayed steps equal plain steps bit for bit, across steppers and dt changes."""
    w = wl.make("c4", n)
    outs = []
    for graph in (False, True):
        ctx = bh.Context(n, 16)
        pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
        bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
        bh.bh_set_gravity_method(ctx.ctx, method)
        bh.bh_set_graph(ctx.ctx, graph)
        l0 = bh.bh_get_launches(ctx.ctx)
        for _ in range(6):
            bh.bh_kdk_step(ctx.ctx, 1e-3)
        for _ in range(4):
            bh.bh_euler_step(ctx.ctx, 5e-4)
        for _ in range(3):
            bh.bh_multirate_step(ctx.ctx, 1e-4, 4)
        for _ in range(3):
            bh.bh_kdk_step(ctx.ctx, 2e-3)       # new dt: plain, capture, replay
        bh.bh_synchronize(ctx.ctx)
        outs.append((pos.cpu().numpy(), vel.cpu().numpy(), bh.bh_get_launches(ctx.ctx) - l0))
        if method == 0:
            assert bh.bh_get_node_count(ctx.ctx)[0] > 1
        ctx.close()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert outs[0][2] == outs[1][2]             # the launch count is the same claim on both paths


def test_graph_replay_keeps_the_host_view_of_the_context():
    """A replayed stepper graph rebuilds the tree of the BOUND state on the device; the host-side view (n, built,
    walked) must say so even if the caller built another, smaller, set of bodies in between: a following bh_accel
    writes all bound_n rows and the getters describe the bound state's tree."""
    w, w2 = wl.make("c4", 1000), wl.make("c1", 500)
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    ctx = bh.Context(w.n, 16)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    bh.bh_set_graph(ctx.ctx, True)
    for _ in range(4):                                   # plain (a(x0) too), plain, capture, replay
        bh.bh_kdk_step(ctx.ctx, 1e-3)
    ctx.build(dev(w2.pos), dev(w2.mass))                 # another body set, n = 500
    assert bh.bh_get_groups(ctx.ctx) == len(orc.build(w2.pos, w2.mass, 16).gstart) - 1
    bh.bh_kdk_step(ctx.ctx, 1e-3)                        # replay: the device now holds the 1000-body tree again
    bh.bh_synchronize(ctx.ctx)
    p = pos.cpu().numpy()
    t = orc.build(p, w.mass, 16)
    assert bh.bh_get_node_count(ctx.ctx) == (t.M, t.depth)
    ctx.n = w.n
    guard = torch.full((w.n + 64, 3), 7.0, dtype=torch.float64, device="cuda")
    bh.bh_accel(ctx.ctx, w.theta, w.eps, w.G, guard[:w.n])
    a = guard.cpu().numpy()
    assert (a[w.n:] == 7.0).all()
    ref = orc.accel(t, w.theta, w.eps, w.G)[0]
    assert (np.linalg.norm(a[:w.n] - ref, axis=1) / np.linalg.norm(ref, axis=1)).max() <= 1e-11
    # direct method: after a (replayed) step the context holds no tree, whatever was built before
    bh.bh_set_gravity_method(ctx.ctx, 1)
    for _ in range(4):
        bh.bh_kdk_step(ctx.ctx, 1e-3)
    ctx.build(dev(w2.pos), dev(w2.mass))
    bh.bh_kdk_step(ctx.ctx, 1e-3)
    with pytest.raises(bh.BhError) as e:
        bh.bh_accel(ctx.ctx, w.theta, w.eps, w.G, guard[:w.n])
    assert e.value.status == bh.BH_ERR_STATE
    ctx.close()


@pytest.mark.parametrize("name,n,C", [("c1", 1024, 8), ("c2", 16384, 16), ("c4", 30000, 16), ("c3", 777, 1), ("c3", 5, 16)])
def test_accel_and_potential_from_one_walk(name, n, C):
    """bh_accel_potential: both outputs of the fused walk against the oracle's two evaluations (same lists)."""
    w = wl.make(name, n)
    t = orc.build(w.pos, w.mass, C)
    ctx = bh.Context(n, C)
    ctx.build(dev(w.pos), dev(w.mass))
    acc = torch.empty((n, 3), dtype=torch.float64, device="cuda")
    phi = torch.empty(n, dtype=torch.float64, device="cuda")
    bh.bh_accel_potential(ctx.ctx, w.theta, w.eps, w.G, acc, phi)
    a_ref, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G)
    p_ref = orc.potential(t, w.theta, w.eps, w.G)
    a = acc.cpu().numpy()
    nz = np.linalg.norm(a_ref, axis=1) > 0
    assert (np.linalg.norm(a - a_ref, axis=1)[nz] / np.linalg.norm(a_ref, axis=1)[nz]).max() <= TOL
    assert np.abs(phi.cpu().numpy() - p_ref).max() <= TOL * np.abs(p_ref).min()
    gm, gd = ctx.counts()
    assert np.array_equal(gm.cpu().numpy().view(np.uint32), nm) and np.array_equal(gd.cpu().numpy().view(np.uint32), nd)
    # and it equals the two separate calls to rounding
    a2 = ctx.accel(w.theta, w.eps, w.G).cpu().numpy()
    assert np.abs(a - a2).max() <= 1e-12 * np.abs(a2).max()
    ctx.close()
