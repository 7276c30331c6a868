"""The paper's two gravity experiments on one B200, through the C ABI only:

    python -m paper_1912_04197_b200.experiments fig4      # PAPER.md:201-211, Figure 4
    python -m paper_1912_04197_b200.experiments fig5      # PAPER.md:213-232, Figure 5

fig4  Time of one integration step against the number of bodies: direct N^2 against the Barnes-Hut tree
      at theta = 0.1, 0.25, 0.5, 0.75.  As in the paper: bodies at rest, uniform in a cube, gravity only,
      a very short time step so the dynamics stay steady, the time of one step averaged over several
      steps, the paper's preferred semi-implicit Euler stepper.  The paper stops at
      N = 1e4 (a 940M laptop GPU); here N runs to 1e6.  Reported: ms per step, and the crossover N below
      which the direct sum is the faster method (paper: about 700).
fig5  Maximum relative position error, Eq. (7), of Barnes-Hut runs against a direct-sum run
      of the same N = 1000 cold uniform cloud through one contraction and re-expansion, with the energy
      drift of the direct run ("conservation of energy ... checked").  The paper does not
      give the cloud's size, masses or softening; DESIGN.md records the choices made here (G = M = 1, cube
      of side 2, eps = 0.05, leapfrog for the reference accuracy and semi-implicit Euler as the paper's
      own), so the figures are comparable in shape, not in absolute value.

Prints markdown tables.  Product path only: nothing here touches oracle/.
"""
from __future__ import annotations

import math
import sys

import numpy as np
import torch

from . import binding as bh
from . import workloads as wl

THETAS = (0.1, 0.25, 0.5, 0.75)


def cube_cloud(n: int, seed: int, half: float = 1.0) -> np.ndarray:
    """n positions uniform in the cube [-half, half]^3, from the counter-based stream."""
    return (wl.uniform(seed, 0, 0, 3 * n).reshape(n, 3) * 2.0 - 1.0) * half


def _time_steps(ctx, steps: int, dt: float) -> float:
    for _ in range(3):               # warm-up (with bh_set_graph: plain, capture, replay)
        bh.bh_euler_step(ctx.ctx, dt)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(steps):
        bh.bh_euler_step(ctx.ctx, dt)
    b.record()
    torch.cuda.synchronize()
    bh.bh_synchronize(ctx.ctx)
    return a.elapsed_time(b) / steps


def fig4(ns=None, leaf_cap: int = 16, graph: bool = False):
    ns = ns or [10, 30, 100, 300, 700, 1000, 2000, 3000, 5000, 10000, 30000, 100000, 300000, 1000000]
    dev = torch.device("cuda:0")
    print("| N | direct N^2 ms/step | " + " | ".join(f"BH theta={t:g} ms/step" for t in THETAS) + " | fastest |")
    print("|---|---|" + "---|" * (len(THETAS) + 1))
    rows = []
    for n in ns:
        p0 = cube_cloud(n, wl.BASE_SEED + 40)
        mass = torch.full((n,), 1.0 / n, dtype=torch.float64, device=dev)
        ctx = bh.Context(n, leaf_cap, device=dev)
        times = []
        for method, theta in [(1, 0.0)] + [(0, t) for t in THETAS]:
            pos = torch.as_tensor(p0).to(dev)
            vel = torch.zeros_like(pos)
            bh.bh_bind_state(ctx.ctx, pos, vel, mass, theta, 1e-3, 1.0)
            bh.bh_set_gravity_method(ctx.ctx, method)
            bh.bh_set_graph(ctx.ctx, graph)
            steps = 50 if n <= 100000 else (10 if method == 0 else 2)
            times.append(_time_steps(ctx, steps, 1e-6))
        ctx.close()
        best = int(np.argmin(times))
        label = "direct" if best == 0 else f"BH {THETAS[best - 1]:g}"
        print(f"| {n} | {times[0]:.4g} | " + " | ".join(f"{t:.4g}" for t in times[1:]) + f" | {label} |", flush=True)
        rows.append((n, times))
    # crossover against theta = 0.5: log-log interpolation between the bracketing sizes
    k = THETAS.index(0.5) + 1
    cross = None
    for (n0, t0), (n1, t1) in zip(rows, rows[1:]):
        r0, r1 = math.log(t0[0] / t0[k]), math.log(t1[0] / t1[k])
        if r0 < 0 <= r1:
            f = -r0 / (r1 - r0)
            cross = math.exp(math.log(n0) + f * (math.log(n1) - math.log(n0)))
    print(f"\ncrossover (direct = BH at theta 0.5): N ~ {cross:.0f}" if cross else "\nno crossover in range")
    return rows


def fig5(n: int = 1000, eps: float = 0.05, leaf_cap: int = 16, steps: int = 3000, every: int = 250):
    dev = torch.device("cuda:0")
    p0 = cube_cloud(n, wl.BASE_SEED + 41)
    p0 -= p0.mean(axis=0)          # barycentre at the origin: Eq. (7) is relative to |r| from there
    mass = torch.full((n,), 1.0 / n, dtype=torch.float64, device=dev)
    rho = 1.0 / 8.0                 # mean density of M = 1 in a cube of side 2
    t_ff = math.sqrt(3.0 * math.pi / (32.0 * rho))
    dt = 2.0 * t_ff / steps         # one contraction and re-expansion
    print(f"N = {n}, G = M = 1, cube side 2, eps = {eps}, free-fall time {t_ff:.4f}, dt = {dt:.3e} "
          f"({dt / bh.bh_gravity_dt(1.0, rho):.2e} of the Eq. (8) bound), {steps} steps\n")
    for stepper in ("kdk", "euler"):
        step = bh.bh_kdk_step if stepper == "kdk" else bh.bh_euler_step
        runs = []                   # direct first, then the tree runs
        for method, theta in [(1, 0.0)] + [(0, t) for t in THETAS]:
            ctx = bh.Context(n, leaf_cap, device=dev)
            pos = torch.as_tensor(p0).to(dev)
            vel = torch.zeros_like(pos)
            bh.bh_bind_state(ctx.ctx, pos, vel, mass, theta, eps, 1.0)
            bh.bh_set_gravity_method(ctx.ctx, method)
            runs.append((ctx, pos, vel))
        ctx0, pos0, vel0 = runs[0]
        phi = torch.empty(n, dtype=torch.float64, device=dev)

        def energy():
            ctx0.build(pos0, mass)
            bh.bh_direct_potential(ctx0.ctx, eps, 1.0, phi)
            d = bh.bh_diagnostics(ctx0.ctx, pos0, vel0, mass, phi)
            return d["ekin"] + d["epot"], d

        e0, _ = energy()
        print(f"stepper: {'leapfrog KDK' if stepper == 'kdk' else 'semi-implicit Euler (PAPER.md:148)'}")
        print("| t / t_ff | " + " | ".join(f"max e_i % theta={t:g}" for t in THETAS) +
              " | direct run: (E-E0)/|E0| | |P| | |L| |")
        print("|---|" + "---|" * (len(THETAS) + 3))
        worst = [0.0] * len(THETAS)
        for k in range(1, steps + 1):
            for ctx, _, _ in runs:
                step(ctx.ctx, dt)
            if k % every == 0 or k == steps:
                errs = [bh.bh_position_error(ctx.ctx, pos, pos0) for ctx, pos, _ in runs[1:]]
                worst = [max(a, b) for a, b in zip(worst, errs)]
                e, d = energy()
                print(f"| {k * dt / t_ff:.3f} | " + " | ".join(f"{x:.3e}" for x in errs) +
                      f" | {(e - e0) / abs(e0):.2e} | {np.linalg.norm(d['P']):.1e} | {np.linalg.norm(d['L']):.1e} |",
                      flush=True)
        print("| worst | " + " | ".join(f"{x:.3e}" for x in worst) + " | | | |\n")
        for ctx, _, _ in runs:
            ctx.close()


if __name__ == "__main__":
    which = sys.argv[1] if len(sys.argv) > 1 else "fig4"
    if which in ("fig4", "fig4-graph"):     # fig4-graph: the steps replayed through a CUDA graph (bh_set_graph)
        fig4([int(x) for x in sys.argv[2:]] or None, graph=which == "fig4-graph")
    elif which == "fig5":
        fig5()
    else:
        raise SystemExit("usage: python -m paper_1912_04197_b200.experiments fig4|fig5")
