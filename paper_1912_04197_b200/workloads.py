"""Seeded synthetic body clouds for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no cube, keys, tree, forces): it only draws
inputs.  It is the one module that both the CPU oracle's tests and the CUDA path's tests/bench
import, so that both sides see bit-identical arrays (SURVEY.md §8(d) "Synthetic inputs").

Random numbers come from a counter-based generator written out here (SplitMix64's output mix
applied to ``key + (i+1)*GOLDEN``), so a stream is a pure function of (seed, stream id, index):
vectorised in numpy, independent of numpy's own generators and versions.

Shapes follow the paper's scenarios: uniform random positions, gravity only (§3.2);
aggregation clouds of fragments with random velocity directions and a residual solid-body spin
(§4.3).  The paper uses no public dataset on this path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
BASE_SEED = 1912041970


def _mix(z: np.ndarray) -> np.ndarray:
    """SplitMix64 output function on a uint64 array (wrap-around arithmetic)."""
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def _stream_key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = _mix(np.array([np.uint64(seed)], dtype=np.uint64) * _GOLDEN + np.uint64(stream + 1))
        k = _mix(k + _GOLDEN * np.uint64(stream + 1))
    return k[0]


def uniform(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count doubles in [0,1): element i is a pure function of (seed, stream, start+i)."""
    key = _stream_key(seed, stream)
    idx = np.arange(start + 1, start + count + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        bits = _mix(key + idx * _GOLDEN)
    return (bits >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _ball(seed: int, stream: int, n: int, radius: float) -> np.ndarray:
    """First n candidates of the stream that fall inside the unit ball (rejection from [-1,1]^3)."""
    out = np.empty((n, 3), dtype=np.float64)
    have, start = 0, 0
    while have < n:
        m = max(1024, 2 * (n - have) + 64)
        u = uniform(seed, stream, 3 * start, 3 * m).reshape(m, 3) * 2.0 - 1.0
        ok = (u * u).sum(axis=1) < 1.0
        acc = u[ok][: n - have]
        out[have:have + len(acc)] = acc
        have += len(acc)
        start += m
    return out * radius


def _isotropic(seed: int, stream: int, n: int) -> np.ndarray:
    u = uniform(seed, stream, 0, 2 * n).reshape(n, 2)
    z = 1.0 - 2.0 * u[:, 0]
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    phi = 2.0 * math.pi * u[:, 1]
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def _gauss(seed: int, stream: int, n: int) -> np.ndarray:
    """n standard normals by Box-Muller (cosine branch only)."""
    u = uniform(seed, stream, 0, 2 * n).reshape(n, 2)
    return np.sqrt(-2.0 * np.log(1.0 - u[:, 0])) * np.cos(2.0 * math.pi * u[:, 1])


@dataclass
class Workload:
    name: str
    pos: np.ndarray              # [n,3] float64
    mass: np.ndarray             # [n] float64
    vel: np.ndarray | None       # [n,3] float64 or None
    G: float
    eps: float
    theta: float
    leaf_cap: int
    dt: float = 0.0
    steps: int = 0
    thetas: tuple = ()
    seed: int = 0
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])


def c1(n: int = 1024, seed: int = BASE_SEED + 1) -> Workload:
    """configs[0]: uniform unit ball, equal masses 1/N, G=1, eps=1e-3, theta=.5, C=8."""
    pos = _ball(seed, 0, n, 1.0)
    mass = np.full(n, 1.0 / n)
    return Workload("c1", pos, mass, None, 1.0, 1e-3, 0.5, 8, seed=seed,
                    note="uniform unit ball, m=1/N")


def c2(n: int = 16384, seed: int = BASE_SEED + 2) -> Workload:
    """configs[1]: rubble pile, ball R=1 km, radii dN/dr ~ r^-3 on [5,50] m, rho=2000, SI units."""
    pos = _ball(seed, 0, n, 1000.0)
    u = uniform(seed, 1, 0, n)
    rmin, rmax = 5.0, 50.0
    a, b = rmin ** -2, rmax ** -2
    r = (a - u * (a - b)) ** -0.5
    mass = 2000.0 * (4.0 / 3.0) * math.pi * r ** 3
    return Workload("c2", pos, mass, None, 6.674e-11, 0.0, 0.5, 16, seed=seed,
                    note="ball R=1000 m, radii power law r^-3 on [5,50] m, rho=2000 kg/m^3",
                    extra={"radius": r})


def c3(n: int = 131072, seed: int = BASE_SEED + 3) -> Workload:
    """configs[2]: uniform unit ball, equal masses, eps=1e-4, theta sweep, C=16."""
    pos = _ball(seed, 0, n, 1.0)
    mass = np.full(n, 1.0 / n)
    return Workload("c3", pos, mass, None, 1.0, 1e-4, 0.5, 16, seed=seed,
                    thetas=(0.0, 0.3, 0.5, 0.7, 1.0), note="uniform unit ball, m=1/N")


def c4(n: int = 1048576, seed: int = BASE_SEED + 4, rmax: float = 64.0) -> Workload:
    """configs[3]: Plummer sphere a=1 truncated at r<=rmax (re-draw), equilibrium velocities."""
    # radii: r = (u^(-2/3) - 1)^(-1/2), candidates in stream order, first n with r <= rmax
    r = np.empty(n)
    have, start = 0, 0
    while have < n:
        m = max(1024, (n - have) + (n - have) // 64 + 64)
        u = uniform(seed, 0, start, m)
        u = np.where(u > 0.0, u, 0.5)
        rr = (u ** (-2.0 / 3.0) - 1.0) ** -0.5
        rr = rr[rr <= rmax][: n - have]
        r[have:have + len(rr)] = rr
        have += len(rr)
        start += m
    pos = _isotropic(seed, 1, n) * r[:, None]
    # speeds: von Neumann rejection on g(q) = q^2 (1-q^2)^(7/2), q in [0,1], g_max < 0.1
    q = np.zeros(n)
    todo = np.arange(n)
    rnd = 0
    while len(todo):
        u = uniform(seed, 16 + rnd, 0, 2 * n).reshape(n, 2)[todo]
        x, y = u[:, 0], 0.1 * u[:, 1]
        ok = y < x * x * (1.0 - x * x) ** 3.5
        q[todo[ok]] = x[ok]
        todo = todo[~ok]
        rnd += 1
    speed = q * math.sqrt(2.0) * (1.0 + r * r) ** -0.25
    vel = _isotropic(seed, 2, n) * speed[:, None]
    mass = np.full(n, 1.0 / n)
    return Workload("c4", pos, mass, vel, 1.0, 1e-4, 0.5, 16, dt=1e-3, steps=10, seed=seed,
                    note=f"Plummer a=1 truncated r<={rmax:g}, m=1/N, equilibrium velocities")


def c5(n: int = 4194304, seed: int = BASE_SEED + 5) -> Workload:
    """configs[4]: uniform ball R=10, M=1, solid-body spin 0.3*sqrt(GM/R^3) about z + N(0,0.05^2)."""
    R = 10.0
    pos = _ball(seed, 0, n, R)
    mass = np.full(n, 1.0 / n)
    omega = 0.3 * math.sqrt(1.0 / R ** 3)
    vel = np.stack([-omega * pos[:, 1], omega * pos[:, 0], np.zeros(n)], axis=1)
    for a in range(3):
        vel[:, a] += 0.05 * _gauss(seed, 8 + a, n)
    return Workload("c5", pos, mass, vel, 1.0, 1e-3, 0.6, 32, dt=1e-3, steps=50, seed=seed,
                    note="uniform ball R=10, m=1/N, spin 0.3 critical + sigma=0.05")


def spheres(n: int, seed: int = BASE_SEED + 6, mean_contacts: float = 1.5, speed: float = 0.0) -> Workload:
    """Cloud of finite-size bodies for the broad phase / aggregate rows:
    centres uniform in the unit ball, bounding radii uniform in [0.5, 1.5] r0 with r0 chosen so that a
    body's sphere overlaps `mean_contacts` others on average (N (2 r0)^3 = mean_contacts) — around the
    percolation threshold, so aggregates of every size appear, as at the end of the paper's transient
    phase.  Optional random velocities of typical magnitude `speed`."""
    pos = _ball(seed, 0, n, 1.0)
    r0 = 0.5 * (mean_contacts / n) ** (1.0 / 3.0)
    radius = r0 * (0.5 + uniform(seed, 1, 0, n))
    vel = _isotropic(seed, 2, n) * (speed * uniform(seed, 3, 0, n))[:, None] if speed > 0 else None
    mass = (4.0 / 3.0) * math.pi * radius ** 3
    return Workload("spheres", pos, mass, vel, 1.0, 0.0, 0.5, 16, seed=seed,
                    note=f"unit ball, radii U[0.5,1.5] r0, r0={r0:.3e}", extra={"radius": radius})


CONFIGS = {"c1": c1, "c2": c2, "c3": c3, "c4": c4, "c5": c5}


def make(name: str, n: int | None = None) -> Workload:
    """Workload `name` at its BASELINE.json size, or scaled to n bodies (same distribution)."""
    f = CONFIGS[name]
    return f() if n is None else f(n=n)
