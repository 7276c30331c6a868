#!/usr/bin/env python
"""bench.py — throughput of the Barnes-Hut hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config c4]

One "step" is one leapfrog KDK step through the C ABI (bh_kdk_step): kick+drift kernel, octree
rebuild (cube, keys, radix sort, gather, tree, group boxes, monopoles), group walk, kick kernel —
steps a1-a7 and a9 of SURVEY.md §8(a).  The direct N^2 kernel (a8) is the paper's comparison method
(PAPER.md:201-211): it is timed once beside the steps and gives `speedup_vs_direct`.

value   = body-accelerations per second = n_gpus * N * K / (sum of the K per-step durations), each
          step timed with CUDA events on the library's stream, L2 flushed between steps, max over
          ranks.  Inputs are resident in HBM.
e2e     = the same metric through bh_eval_host: pinned host pos/mass in, acc out, copies timed.
roofline= the walk kernel (dominant): 20 flops per body-source interaction over its
          CUDA-event duration, against the fp64 FMA peak 148 SM x 64 lanes x 2 x 1.965 GHz.
cpu_baseline = the oracle as it stands on the host cores, on a bounded sample of the same workload.

Multi-GPU: the path does not shard (north_star: one GPU, no collectives) -> replicas only; every
rank runs the same workload, value is the aggregate, scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "BH accel evals/s (build+walk) N=1M theta=0.5 fp64; speedup vs direct N^2"
UNIT = "body-accelerations/s"
FLOPS_PER_INTERACTION = 20.0
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12      # derived: SMs x fp64 FMA lanes x 2 x max SM clock
# dram__bytes_read.sum + dram__bytes_write.sum of one walk_kernel launch, from the committed ncu --set full
# capture (profiles/r01_walk_ncu_full.md: 65.32 MB + 15.84 MB); a profiler figure, not measured by this run
WALK_TRAFFIC_NCU = {"c4": 81.15e6}


def workload_desc(w):
    return (f"{w.name}: N={w.n} {w.note}, G={w.G:g}, eps={w.eps:g}, theta={w.theta:g}, leaf cap {w.leaf_cap}, "
            f"W=32, Gc=512, KDK dt={w.dt:g}")


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
                 "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80)}
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        med = statistics.median(self.samples) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ oracle arm
def oracle_sample(w, budget_s: float, seed: int = 0):
    """Time the oracle on a bounded sample: full build once, walk of a random set of groups sized to
    the budget.  Returns (evals/s, description, cores)."""
    import numpy as np
    from oracle import bh_oracle as orc
    cores = orc.num_threads()
    t0 = time.perf_counter()
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    t_build = time.perf_counter() - t0
    ng = t.ngroups
    # calibrate on a few groups spread over the cloud
    cal = max(8, min(64, ng))
    g0 = (ng // 2 // cal) * cal
    t0 = time.perf_counter()
    orc.accel(t, w.theta, w.eps, w.G, g0, min(ng, g0 + cal))
    per_group = (time.perf_counter() - t0) / cal
    want = int(max(cal, min(ng, budget_s / max(per_group, 1e-9))))
    rng = np.random.default_rng(seed)
    # contiguous chunks of 32 groups at random offsets (the oracle API walks ranges)
    chunks = max(1, want // 32)
    starts = rng.choice(max(1, ng - 32), size=chunks, replace=False) if ng > 64 else np.array([0])
    bodies, t_walk = 0, 0.0
    for s in starts:
        e = min(ng, int(s) + 32)
        t0 = time.perf_counter()
        orc.accel(t, w.theta, w.eps, w.G, int(s), e)
        t_walk += time.perf_counter() - t0
        bodies += int(t.gstart[e] - t.gstart[int(s)])
    frac = bodies / w.n
    value = bodies / (t_build * frac + t_walk)
    desc = (f"oracle build of all N={w.n} bodies ({t_build:.2f} s, prorated) + walk of {bodies} bodies in "
            f"{len(starts)} chunks of 32 groups ({t_walk:.2f} s)")
    return value, desc, cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1912_04197_b200 import workloads as wl
    w = wl.make(args.config)
    total_budget = 150.0
    per_step = max(0.5, total_budget / (args.steps + args.warmup))
    vals = []
    t_all0 = time.perf_counter()
    for s in range(args.warmup + args.steps):
        v, desc, cores = oracle_sample(w, per_step, seed=s)
        if s >= args.warmup:
            vals.append(v)
    value = len(vals) / sum(1.0 / v for v in vals)     # harmonic mean = total bodies / total time
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * (time.perf_counter() - t_all0) / (args.steps + args.warmup),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_desc(w), "sampled": True},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ multi-rank
def aggregate(total_ms: float, bodies_per_rank: int, steps: int, world: int, device=None):
    """Replicas only: every rank runs the same workload; the job's time is the MAX over
    ranks of the summed per-step device time, its throughput the bodies of ALL ranks over that time.
    Works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([total_ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tmax = float(t.item())
    return tmax, world * bodies_per_rank * steps / (tmax * 1e-3)


# ------------------------------------------------------------------------------------------ rows "next"
def next_rows(ctx, w, pos, vel, mass, dev, hbm_peak):
    """SURVEY.md 8(f) rows NEXT-1..4 timed beside the headline (CUDA events on the library's stream, median of
    3, inputs resident): tree potential, conserved quantities, Eq. (7), semi-implicit Euler step on the
    headline workload; broad phase + aggregate identification on a cloud of N finite-size bodies."""
    import torch
    from paper_1912_04197_b200 import binding as bh
    from paper_1912_04197_b200 import workloads as wl
    stream = torch.cuda.current_stream()

    def timed(fn, reps=3):
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            r = fn()
            b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return statistics.median(ts), r

    out = {}
    n = w.n
    ctx.build(pos, mass)
    phi = torch.empty(n, dtype=torch.float64, device=dev)
    bh.bh_potential(ctx.ctx, w.theta, w.eps, w.G, phi)
    ms, _ = timed(lambda: bh.bh_potential(ctx.ctx, w.theta, w.eps, w.G, phi))
    inter = bh.bh_get_stats(ctx.ctx)["interactions"]
    out["potential_walk"] = {"ms": ms, "interactions_per_s": inter / (ms * 1e-3),
                             "fp64_instr_per_interaction": 12}
    acc2 = torch.empty((n, 3), dtype=torch.float64, device=dev)
    bh.bh_accel_potential(ctx.ctx, w.theta, w.eps, w.G, acc2, phi)
    ms, _ = timed(lambda: bh.bh_accel_potential(ctx.ctx, w.theta, w.eps, w.G, acc2, phi))
    out["accel_and_potential_walk"] = {"ms": ms, "interactions_per_s": inter / (ms * 1e-3),
                                       "fp64_instr_per_interaction": 19}
    ms, d = timed(lambda: bh.bh_diagnostics(ctx.ctx, pos, vel, mass, phi))
    out["diagnostics"] = {"ms": ms, "GB_per_s": 64.0 * n / (ms * 1e-3) / 1e9, "frac_of_hbm_peak": 64.0 * n / (ms * 1e-3) / 1e9 / hbm_peak,
                          "bytes_per_body": 64, "virial_2K_over_W": -2.0 * d["ekin"] / d["epot"]}
    ref = pos.clone()
    ms, _ = timed(lambda: bh.bh_position_error(ctx.ctx, pos, ref))
    out["position_error"] = {"ms": ms, "GB_per_s": 48.0 * n / (ms * 1e-3) / 1e9, "bytes_per_body": 48}
    p2, v2 = pos.clone(), vel.clone()
    bh.bh_bind_state(ctx.ctx, p2, v2, mass, w.theta, w.eps, w.G)
    bh.bh_euler_step(ctx.ctx, w.dt or 1e-3)
    ms, _ = timed(lambda: bh.bh_euler_step(ctx.ctx, w.dt or 1e-3))
    out["euler_step"] = {"ms": ms, "body_accelerations_per_s": n / (ms * 1e-3)}
    ms, _ = timed(lambda: bh.bh_multirate_step(ctx.ctx, (w.dt or 1e-3) / 8, 8))
    out["multirate_step_8_substeps"] = {"ms": ms}

    # broad phase + aggregates: N finite-size bodies around the percolation threshold (workloads.spheres)
    sp = wl.spheres(n, mean_contacts=3.0, speed=0.01)
    sctx = bh.Context(n, 16, device=dev)
    spos, smass = torch.as_tensor(sp.pos).to(dev), torch.as_tensor(sp.mass).to(dev)
    srad, svel = torch.as_tensor(sp.extra["radius"]).to(dev), torch.as_tensor(sp.vel).to(dev)
    sctx.build(spos, smass)
    count = bh.bh_broadphase(sctx.ctx, srad, svel, 0.1, None)
    pairs = torch.empty((max(count, 1), 2), dtype=torch.int32, device=dev)
    ms, _ = timed(lambda: bh.bh_broadphase(sctx.ctx, srad, svel, 0.1, pairs))
    out["broadphase"] = {"workload": f"spheres N={n} mean_contacts=3 speed=0.01 dt=0.1", "ms": ms, "pairs": count,
                         "bodies_per_s": n / (ms * 1e-3), "pairs_per_s": count / (ms * 1e-3)}
    label = torch.empty(n, dtype=torch.int32, device=dev)
    size = torch.empty(n, dtype=torch.int32, device=dev)
    ms, (comps, aggs) = timed(lambda: bh.bh_aggregates(sctx.ctx, n, pairs[:count], None, label, size, None))
    out["aggregates"] = {"ms": ms, "edges": count, "edges_per_s": count / (ms * 1e-3), "components": comps,
                         "aggregates": aggs, "largest": int(size.max().item())}
    sctx.close()
    return out


# ------------------------------------------------------------------------------------------ own arm
def run_own(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1912_04197_b200 import binding as bh
    from paper_1912_04197_b200 import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")

    w = wl.make(args.config)
    ctx = bh.Context(w.n, w.leaf_cap, device=dev)
    pos0, mass = torch.as_tensor(w.pos).to(dev), torch.as_tensor(w.mass).to(dev)
    vel0 = torch.as_tensor(w.vel if w.vel is not None else np.zeros_like(w.pos)).to(dev)
    pos, vel = pos0.clone(), vel0.clone()
    dt = w.dt if w.dt > 0 else 1e-3
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    for _ in range(max(3, args.warmup)):
        bh.bh_kdk_step(ctx.ctx, dt)
    bh.bh_synchronize(ctx.ctx)
    bh.bh_set_timing(ctx.ctx, True)
    l0 = bh.bh_get_launches(ctx.ctx)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phase_sum = {k: 0.0 for k in bh.PHASE_NAMES}
    walk_ms, inter = [], []
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                   # evict L2 between timed iterations
        ev[k][0].record(stream)
        bh.bh_kdk_step(ctx.ctx, dt)
        ev[k][1].record(stream)
        if args.phases or k < 8 or k == args.steps - 1:   # per-phase events need a sync; sample them
            ph = bh.bh_get_phase_ms(ctx.ctx)
            st = bh.bh_get_stats(ctx.ctx)
            for name in phase_sum:
                phase_sum[name] += ph[name]
            walk_ms.append(ph["walk"])
            inter.append(st["interactions"])
    barrier()
    wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = bh.bh_get_launches(ctx.ctx) - l0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms, value = aggregate(sum(step_ms), w.n, args.steps, world, dev)
    nph = len(walk_ms)
    phases = {k: v / nph for k, v in phase_sum.items() if k != "direct"}
    M, depth = bh.bh_get_node_count(ctx.ctx)
    ng = bh.bh_get_groups(ctx.ctx)
    st = bh.bh_get_stats(ctx.ctx)

    # ---- roofline of the walk kernel (dominant) ----
    walk_avg_ms = sum(walk_ms) / nph
    inter_avg = sum(inter) / nph
    achieved = FLOPS_PER_INTERACTION * inter_avg / (walk_avg_ms * 1e-3) / 1e12
    peak_meas = bh.bh_measure_fp64_peak(ctx.ctx)
    issue = bh.bh_measure_issue_model(ctx.ctx)
    roofline = {"bound": "alu", "kernel": "walk_kernel", "achieved": achieved, "peak": FP64_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_TFLOPS,
                "peak_source": "derived 148 SM x 64 fp64 FMA lanes x 2 x 1.965 GHz (DESIGN.md); "
                               "MEASURED_PEAKS.json has no fp64 entry",
                "peak_measured_dfma": peak_meas, "frac_of_measured_dfma": achieved / peak_meas,
                "flops_per_interaction": FLOPS_PER_INTERACTION, "interactions_per_launch": inter_avg,
                "interactions_per_s": inter_avg / (walk_avg_ms * 1e-3), "kernel_ms": walk_avg_ms,
                "issue_model_interactions_per_s": issue,
                "frac_of_eval_loop_alone": inter_avg / (walk_avg_ms * 1e-3) / issue["eval_loop_alone"],
                "traffic": args.walk_traffic if args.walk_traffic is not None else WALK_TRAFFIC_NCU.get(w.name),
                "traffic_source": "profiles/r01_walk_ncu_full.md (ncu --set full, bytes per launch)"}
    # build kernels against HBM: algorithmic bytes per body over the build time
    build_ms = sum(phases[k] for k in ("cube", "keys", "sort", "gather", "tree", "monopoles"))
    build_bytes = 390.0 * w.n
    hbm_peak = 6546.9
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass
    build_roof = {"bound": "hbm", "achieved": build_bytes / (build_ms * 1e-3) / 1e9, "peak": hbm_peak,
                  "unit": "GB/s", "frac": build_bytes / (build_ms * 1e-3) / 1e9 / hbm_peak,
                  "algorithmic_bytes_per_body": 390, "build_ms": build_ms}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_desc(w), "parallelism": "replicas only" if world > 1 else "1 gpu",
                      "l2": "flushed between steps (256 MiB write); per-step CUDA events summed",
                      "nodes": M, "depth": depth, "groups": ng},
           "clocks": clocks, "gpu_launches": int(launches), "wall_s": wall,
           "phases_ms": phases, "roofline": roofline, "build_roofline": build_roof,
           "interactions_per_body": st["interactions"] / w.n}

    if rank == 0:
        # ---- direct N^2 beside it (the paper's comparison) ----
        ctx.build(pos, mass)
        nt = w.n if args.full_direct else min(w.n, 16384)
        tg = torch.arange(0, w.n, max(1, w.n // nt), dtype=torch.int32, device=dev)[:nt].contiguous()
        accd = torch.empty((tg.numel(), 3), dtype=torch.float64, device=dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        bh.bh_direct_targets(ctx.ctx, tg, w.eps, w.G, accd)
        a.record(stream)
        bh.bh_direct_targets(ctx.ctx, tg, w.eps, w.G, accd)
        b.record(stream)
        torch.cuda.synchronize()
        dms = a.elapsed_time(b)
        direct_full_ms = dms * w.n / tg.numel()
        pairs = float(tg.numel()) * w.n
        out["direct"] = {"targets": int(tg.numel()), "ms": dms, "full_n2_ms": direct_full_ms,
                         "extrapolated": tg.numel() != w.n, "interactions_per_s": pairs / (dms * 1e-3),
                         "tflops": FLOPS_PER_INTERACTION * pairs / (dms * 1e-3) / 1e12,
                         "frac_of_fp64_peak": FLOPS_PER_INTERACTION * pairs / (dms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS}
        out["speedup_vs_direct"] = direct_full_ms / (total_ms / args.steps)

        # ---- end to end through the C ABI with host buffers ----
        ph, mh = torch.as_tensor(w.pos).pin_memory(), torch.as_tensor(w.mass).pin_memory()
        ah = torch.empty((w.n, 3), dtype=torch.float64).pin_memory()
        for _ in range(2):
            bh.bh_eval_host(ctx.ctx, ph, mh, w.theta, w.eps, w.G, ah)
        ke = max(3, min(args.steps, 20))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(ke):
            bh.bh_eval_host(ctx.ctx, ph, mh, w.theta, w.eps, w.G, ah)   # synchronising call
        te = (time.perf_counter() - t0) / ke
        out["e2e"] = {"value": w.n / te, "unit": UNIT, "h2d_bytes_per_step": 32 * w.n, "d2h_bytes_per_step": 24 * w.n,
                      "ms_per_step": te * 1e3, "call": "bh_eval_host (pinned host pos+mass in, acc out; mass upload beside the first build kernels, "
                              "accelerations stored by the walk kernel straight into the pinned output)"}

        # ---- rows "next" of SURVEY.md 8(f), timed beside the headline ----
        if not args.no_next:
            out["next_rows"] = next_rows(ctx, w, pos0, vel0, mass, dev, hbm_peak)

        # ---- the oracle on the host cores, bounded sample ----
        if not args.no_cpu:
            v, desc, cores = oracle_sample(w, args.cpu_budget)
            out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        print(json.dumps(out), flush=True)
    ctx.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--config", default="c4", help="workload (default c4 = BASELINE configs[3], the metric's)")
    ap.add_argument("--phases", action="store_true", help="read per-phase events after every step")
    ap.add_argument("--full-direct", action="store_true", help="time the direct kernel on all N targets")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle leg")
    ap.add_argument("--no-next", action="store_true", help="skip the timings of the SURVEY 8(f) 'next' rows")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--walk-traffic", type=float, default=None,
                    help="dram bytes per walk launch from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
