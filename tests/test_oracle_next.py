"""Pins for the oracle's "next" rows: potential (O12/O13), conserved quantities
(O14), Eq. (7) position error (O15), Eq. (8) time-step bound (O16), semi-implicit Euler and the
two-rate step (Stepper).  Expected values are closed forms, exact rational arithmetic, the paper's
own statements, or invariants — never the oracle itself.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import workloads as wl


# ------------------------------------------------------------------ O12 / O13 potential
def test_two_body_potential_closed_form():
    # phi_1 = -G m_2 / sqrt(d^2 + eps^2): d = 3, eps = 4 -> -G m_2 / 5 (exactly representable)
    pos = np.array([[0.0, 0.0, 0.0], [3.0, 0.0, 0.0]])
    mass = np.array([2.0, 10.0])
    phi = orc.direct_potential(pos, mass, 4.0, 0.5)
    assert phi[0] == -0.5 * 10.0 / 5.0 and phi[1] == -0.5 * 2.0 / 5.0
    # eps = 0: -G m / d
    phi = orc.direct_potential(pos, mass, 0.0, 1.0)
    assert phi[0] == -10.0 / 3.0 and phi[1] == -2.0 / 3.0
    # the tree path (both bodies in one leaf) gives the same
    t = orc.build(pos, mass, 8)
    assert np.array_equal(orc.potential(t, 0.5, 0.0, 1.0), phi)


def test_potential_against_exact_rational_brute_force():
    """N = 24 bodies on a dyadic lattice: d^2 + eps^2 is an exact rational; sqrt in 60 digits."""
    from decimal import Decimal, getcontext
    getcontext().prec = 60
    rng = np.random.default_rng(5)
    pos = rng.integers(-64, 64, size=(24, 3)).astype(np.float64) / 16.0
    mass = rng.integers(1, 9, size=24).astype(np.float64) / 8.0
    eps, G = 0.25, 3.0
    phi = orc.direct_potential(pos, mass, eps, G)
    for i in range(24):
        s = Decimal(0)
        for k in range(24):
            if k == i:
                continue
            r2 = sum((Fraction(pos[k, a]) - Fraction(pos[i, a])) ** 2 for a in range(3)) + Fraction(eps) ** 2
            s += Decimal(mass[k]) / (Decimal(r2.numerator) / Decimal(r2.denominator)).sqrt()
        want = float(-Decimal(G) * s)
        assert abs(phi[i] - want) <= 2 ** -52 * abs(want)


def test_coincident_bodies_and_self_exclusion():
    # two bodies at the same point: eps = 0 -> the pair adds nothing (r2 == 0); eps > 0 -> -G m / eps.
    # a body never sees itself, whatever eps.
    pos = np.array([[1.0, 2.0, 3.0], [1.0, 2.0, 3.0], [1.0, 2.0, 7.0]])
    mass = np.array([1.0, 2.0, 4.0])
    phi0 = orc.direct_potential(pos, mass, 0.0, 1.0)
    assert np.array_equal(phi0, [-4.0 / 4.0, -4.0 / 4.0, -3.0 / 4.0])
    phi1 = orc.direct_potential(pos, mass, 3.0, 1.0)          # sqrt(16 + 9) = 5
    want = np.array([-(2.0 / 3.0 + 4.0 / 5.0), -(1.0 / 3.0 + 4.0 / 5.0), -3.0 / 5.0])
    assert np.abs(phi1 - want).max() <= 2.0 ** -52                # two terms summed: last-bit freedom
    t = orc.build(pos, mass, 8)
    assert np.array_equal(orc.potential(t, 0.5, 3.0, 1.0), phi1)


def test_acceleration_is_minus_gradient_of_potential():
    """Central finite difference of the direct potential of a probe against the oracle's direct
    acceleration on it: pins sign, softening and exponent of both (a dropped eps^2, a wrong power or
    sign fails at the 1e-3 level; the difference formula is good to ~1e-8)."""
    w = wl.make("c1", 200)
    eps, G = 0.05, 1.7
    acc = orc.direct(w.pos, w.mass, eps, G)
    h = 1e-5
    for i in (0, 17, 150):
        g = np.zeros(3)
        for a in range(3):
            pp, pm = w.pos.copy(), w.pos.copy()
            pp[i, a] += h
            pm[i, a] -= h
            g[a] = (orc.direct_potential(pp, w.mass, eps, G)[i] - orc.direct_potential(pm, w.mass, eps, G)[i]) / (2 * h)
        assert np.linalg.norm(acc[i] + g) <= 1e-7 * np.linalg.norm(acc[i])


def test_tree_potential_theta_zero_equals_direct_and_error_grows():
    w = wl.make("c3", 3000)
    t = orc.build(w.pos, w.mass, 16)
    ref = orc.direct_potential(w.pos, w.mass, w.eps, w.G)
    p0 = orc.potential(t, 0.0, w.eps, w.G)
    assert np.abs(p0 - ref).max() <= 1e-15 * np.abs(ref).max()
    errs = [np.median(np.abs(orc.potential(t, th, w.eps, w.G) - ref) / np.abs(ref)) for th in (0.3, 0.6, 1.0)]
    assert 0 < errs[0] < errs[1] < errs[2] < 1e-2


def test_potential_of_uniform_sphere():
    """Smooth-field sanity: inside a uniform ball of mass M, radius R: phi(r) = -G M (3 R^2 - r^2) / (2 R^3)."""
    w = wl.make("c3", 20000)
    phi = orc.potential(orc.build(w.pos, w.mass, 16), 0.5, w.eps, w.G)
    r = np.linalg.norm(w.pos, axis=1)
    want = -(3.0 - r ** 2) / 2.0
    sel = r < 0.8
    assert np.abs(phi[sel] / want[sel] - 1.0).mean() < 0.01


# ------------------------------------------------------------------ O14 conserved quantities
def test_diagnostics_hand_computed():
    pos = np.array([[1.0, 0.0, 0.0], [0.0, 2.0, 0.0], [0.0, 0.0, -1.0]])
    vel = np.array([[0.0, 3.0, 0.0], [1.0, 0.0, 2.0], [0.5, 0.5, 0.0]])
    mass = np.array([2.0, 1.0, 4.0])
    phi = np.array([-1.0, -2.0, -0.5])
    d = orc.diagnostics(pos, vel, mass, phi)
    assert d["ekin"] == 0.5 * (2 * 9 + 1 * 5 + 4 * 0.5)
    assert d["epot"] == 0.5 * (2 * -1.0 + 1 * -2.0 + 4 * -0.5)
    assert np.array_equal(d["P"], [0 + 1 + 2, 6 + 0 + 2, 0 + 2 + 0])
    # L = sum m x cross v: body0 (1,0,0)x(0,3,0) = (0,0,3) *2; body1 (0,2,0)x(1,0,2) = (4,0,-2); body2 (0,0,-1)x(.5,.5,0) = (.5,-.5,0) *4
    assert np.array_equal(d["L"], [0 + 4 + 2, 0 + 0 - 2, 6 - 2 + 0])
    assert orc.diagnostics(pos, vel, mass)["epot"] == 0.0


def test_potential_energy_counts_every_pair_once():
    """1/2 sum m_i phi_i == - G sum_{i<k} m_i m_k / r_ik on an exactly representable system."""
    pos = np.array([[0.0, 0.0, 0.0], [3.0, 0.0, 0.0], [0.0, 4.0, 0.0]])     # distances 3, 4, 5
    mass = np.array([6.0, 12.0, 20.0])
    phi = orc.direct_potential(pos, mass, 0.0, 1.0)
    d = orc.diagnostics(pos, np.zeros((3, 3)), mass, phi)
    assert d["epot"] == -(6 * 12 / 3.0 + 6 * 20 / 4.0 + 12 * 20 / 5.0)


# ------------------------------------------------------------------ O15 Eq. (7)
def test_position_error_hand_cases():
    ref = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 2.0], [0.0, 0.0, 0.0]])
    pos = np.array([[3.0, 4.0, 5.0], [0.0, 0.0, 2.0], [9.0, 9.0, 9.0]])
    # body 0: |d| = 5, |ref| = 5 -> 100 %; body 1: 0; body 2: reference at the origin, skipped (R25)
    assert orc.position_error(pos, ref) == 100.0
    pos[0] = [3.0, 4.0, 0.0]
    assert orc.position_error(pos, ref) == 0.0
    pos[1] = [0.0, 0.0, 2.5]
    assert orc.position_error(pos, ref) == 25.0
    assert orc.position_error(ref[:2], pos[:2]) == 20.0          # relative to the reference, not symmetric


# ------------------------------------------------------------------ O16 Eq. (8)
def test_gravity_time_step_bound():
    G = 6.674e-11
    # "For typical values of asteroid material density ranging between 1 and 4 g/cm3 ...
    # maximum time steps are in the order of thousands of seconds."
    for rho in (1000.0, 2000.0, 3000.0, 4000.0):
        dt = orc.gravity_dt(G, rho)
        assert 900.0 < dt < 2000.0
        assert abs(dt * 2.0 * math.sqrt(G * rho) - 1.0) < 1e-15
    assert orc.gravity_dt(1.0, 0.25) == 1.0                      # 1 / (2 sqrt(1/4))
    assert orc.gravity_dt(4.0, 4.0) == 0.125
    # T_g/2 with T_g = 1/sqrt(G rho): quadrupling the density halves the bound
    assert orc.gravity_dt(G, 4000.0) * 2.0 == pytest.approx(orc.gravity_dt(G, 1000.0), rel=1e-15)


# ------------------------------------------------------------------ semi-implicit Euler, two-rate step
def _two_body(ecc=0.0):
    m = np.array([1.0, 1e-3])
    M = m.sum()
    r = 1.0
    v = math.sqrt(M / r * (1.0 + ecc))
    pos = np.array([[-m[1] / M * r, 0.0, 0.0], [m[0] / M * r, 0.0, 0.0]])
    vel = np.array([[0.0, -m[1] / M * v, 0.0], [0.0, m[0] / M * v, 0.0]])
    return pos, vel, m


def _energy(s):
    phi = orc.direct_potential(s.pos, s.mass, s.eps, s.G)
    d = orc.diagnostics(s.pos, s.vel, s.mass, phi)
    return d["ekin"] + d["epot"], d["L"], d["P"]


def test_euler_update_is_the_stated_fma_sequence():
    w = wl.make("c1", 64)
    vel = np.linspace(-1, 1, 64 * 3).reshape(64, 3)
    s = orc.Stepper(w.pos, vel, w.mass, 0.5, 1e-3, 1.0, 8, use_direct=True)
    a = orc.direct(w.pos, w.mass, 1e-3, 1.0)
    dt = 0.0123
    s.euler(dt)
    for i in range(64):
        for c in range(3):
            v1 = float(Fraction(a[i, c]) * Fraction(dt) + Fraction(vel[i, c]))
            assert s.vel[i, c] == v1
            assert s.pos[i, c] == float(Fraction(v1) * Fraction(dt) + Fraction(w.pos[i, c]))


def test_euler_conserves_angular_momentum_and_is_first_order():
    """Symplectic Euler: x_{k+1} x v_{k+1} = x_k x v_k for a central force (to rounding); the energy
    error is bounded and first order in dt (halving dt halves it) — a leapfrog would give a quarter."""
    amp = []
    for dt in (2e-3, 1e-3):
        pos, vel, m = _two_body(0.3)
        s = orc.Stepper(pos, vel, m, 0.0, 0.0, 1.0, 8, use_direct=True)
        e0, L0, P0 = _energy(s)
        worst = 0.0
        for _ in range(int(round(8.0 / dt))):
            s.euler(dt)
            e, L, P = _energy(s)
            worst = max(worst, abs(e - e0))
            assert abs(L[2] - L0[2]) <= 1e-13 * abs(L0[2])
            assert np.abs(P - P0).max() <= 1e-17
        amp.append(worst)
    assert amp[0] / amp[1] == pytest.approx(2.0, rel=0.1)
    assert amp[1] < 1e-3 * abs(e0)


def test_multirate_closed_form_and_reduction_to_euler():
    w = wl.make("c1", 32)
    vel = np.cos(np.arange(96.0)).reshape(32, 3)
    a = orc.direct(w.pos, w.mass, 1e-3, 1.0)
    # n_sub = 1 is one semi-implicit Euler step, bit for bit
    s1 = orc.Stepper(w.pos, vel, w.mass, 0.5, 1e-3, 1.0, 8, use_direct=True)
    s2 = orc.Stepper(w.pos, vel, w.mass, 0.5, 1e-3, 1.0, 8, use_direct=True)
    s1.euler(0.01)
    s2.multirate(0.01, 1)
    assert np.array_equal(s1.pos, s2.pos) and np.array_equal(s1.vel, s2.vel)
    # frozen acceleration over n sub-steps: v_n = v_0 + n a dt, x_n = x_0 + n v_0 dt + a dt^2 n (n+1) / 2
    n, dt = 7, 0.003
    s = orc.Stepper(w.pos, vel, w.mass, 0.5, 1e-3, 1.0, 8, use_direct=True)
    s.multirate(dt, n)
    v_want = vel + n * a * dt
    x_want = w.pos + n * vel * dt + a * dt * dt * n * (n + 1) / 2
    assert np.abs(s.vel - v_want).max() <= 1e-14 * np.abs(v_want).max()
    assert np.abs(s.pos - x_want).max() <= 1e-14 * np.abs(x_want).max()
    assert np.array_equal(s.acc, a)                              # one evaluation, at x_k


def test_multirate_tree_equals_direct_at_theta_zero():
    w = wl.make("c1", 500)
    vel = np.zeros_like(w.pos)
    st = orc.Stepper(w.pos, vel, w.mass, 0.0, 1e-3, 1.0, 8)
    sd = orc.Stepper(w.pos, vel, w.mass, 0.0, 1e-3, 1.0, 8, use_direct=True)
    for _ in range(3):
        st.multirate(1e-3, 4)
        sd.multirate(1e-3, 4)
    assert np.abs(st.pos - sd.pos).max() <= 1e-14
