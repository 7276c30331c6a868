"""Per-config report on one B200: `python -m paper_1912_04197_b200.report [c1 c2 ...]`.

For each BASELINE.json config: build and walk times (CUDA events inside the library), body
accelerations per second, interactions per second, the direct N^2 kernel beside it (all bodies up to
N = 131072, 4096 sampled targets above, PAPER.md:201-211 compares the two methods), the Barnes-Hut
error against the direct sum per theta (Eq. (7) PAPER.md:223 applied to accelerations
"the error increases monotonically with theta"), and for the KDK configs the time per step.
Prints one markdown table row per (config, theta).  Product path only: nothing here touches oracle/.
"""
from __future__ import annotations

import sys

import numpy as np
import torch

from . import binding as bh
from . import workloads as wl

BUILD_PHASES = ("cube", "keys", "sort", "gather", "tree", "monopoles")


def _median(xs):
    return float(np.median(np.asarray(xs)))


def run_config(name: str, reps: int = 5):
    w = wl.make(name)
    dev = torch.device("cuda:0")
    ctx = bh.Context(w.n, w.leaf_cap, device=dev)
    pos, mass = torch.as_tensor(w.pos).to(dev), torch.as_tensor(w.mass).to(dev)
    acc = torch.empty((w.n, 3), dtype=torch.float64, device=dev)
    bh.bh_set_timing(ctx.ctx, True)
    # direct sum: the reference for the BH error and the comparison method
    ctx.build(pos, mass)
    full = w.n <= 131072
    if full:
        ref = ctx.direct(w.eps, w.G)
        rows = None
    else:
        rows = torch.as_tensor(np.random.default_rng(w.seed).choice(w.n, size=4096, replace=False).astype(np.int32)).to(dev)
        ref = ctx.direct(w.eps, w.G, targets=rows)
    t_direct = []
    for _ in range(2):
        (ctx.direct(w.eps, w.G) if full else ctx.direct(w.eps, w.G, targets=rows))
        t_direct.append(bh.bh_get_phase_ms(ctx.ctx)["direct"])
    t_direct_full = min(t_direct) * (1.0 if full else w.n / 4096.0)
    pairs_per_s = (w.n if full else 4096) * float(w.n) / (min(t_direct) * 1e-3)
    M, depth = bh.bh_get_node_count(ctx.ctx)
    ng = bh.bh_get_groups(ctx.ctx)
    out = []
    for theta in (w.thetas if w.thetas else (w.theta,)):
        tb, tw = [], []
        for _ in range(reps):
            ctx.build(pos, mass)
            bh.bh_accel(ctx.ctx, theta, w.eps, w.G, acc)
            ph = bh.bh_get_phase_ms(ctx.ctx)
            tb.append(sum(ph[k] for k in BUILD_PHASES))
            tw.append(ph["walk"])
        st = bh.bh_get_stats(ctx.ctx)
        a = acc if rows is None else acc[rows.long()]
        err = (torch.linalg.norm(a - ref, dim=1) / torch.linalg.norm(ref, dim=1)).cpu().numpy()
        t_b, t_w = _median(tb), _median(tw)
        out.append(dict(config=name, n=w.n, theta=theta, nodes=M, depth=depth, groups=ng, t_build_ms=t_b, t_walk_ms=t_w,
                        evals_per_s=w.n / ((t_b + t_w) * 1e-3), inter_per_body=st["interactions"] / w.n,
                        inter_per_s=st["interactions"] / (t_w * 1e-3), t_direct_ms=t_direct_full,
                        direct_extrapolated=not full, direct_pairs_per_s=pairs_per_s,
                        speedup=t_direct_full / (t_b + t_w), err_median=float(np.median(err)), err_max=float(err.max())))
    step_ms = None
    if w.steps:
        vel = torch.as_tensor(w.vel).to(dev)
        p2 = pos.clone()
        bh.bh_bind_state(ctx.ctx, p2, vel, mass, w.theta, w.eps, w.G)
        bh.bh_kdk_step(ctx.ctx, w.dt)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(w.steps):
            bh.bh_kdk_step(ctx.ctx, w.dt)
        b.record()
        torch.cuda.synchronize()
        bh.bh_synchronize(ctx.ctx)
        step_ms = a.elapsed_time(b) / w.steps
    ctx.close()
    return out, step_ms


def main(argv):
    names = argv or ["c1", "c2", "c3", "c4", "c5"]
    print("| config | N | theta | nodes | depth | groups | t_build ms | t_walk ms | evals/s | inter/body | inter/s | "
          "t_direct ms | speedup | BH vs direct median | max | KDK ms/step |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    for name in names:
        rows, step_ms = run_config(name)
        for r in rows:
            d = f"{r['t_direct_ms']:.4g}" + (" (x N/4096)" if r["direct_extrapolated"] else "")
            print(f"| {r['config']} | {r['n']} | {r['theta']:g} | {r['nodes']} | {r['depth']} | {r['groups']} | "
                  f"{r['t_build_ms']:.3f} | {r['t_walk_ms']:.3f} | {r['evals_per_s']:.4g} | {r['inter_per_body']:.0f} | "
                  f"{r['inter_per_s']:.4g} | {d} | {r['speedup']:.4g} | {r['err_median']:.3g} | {r['err_max']:.3g} | "
                  f"{'' if step_ms is None else f'{step_ms:.3f}'} |", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
