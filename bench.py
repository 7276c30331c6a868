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
          CUDA-event duration, against the fp64 FMA rate MEASURED in the same run (libbh_microbench.so;
          MEASURED_PEAKS.json has no fp64 entry); the nominal 148 SM x 64 lanes x 2 x 1.965 GHz beside it.
          traffic and l2_hit_rate are profiler figures read from profiles/r03_roofline.csv (ncu --set full).
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
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # nominal: SMs x fp64 FMA lanes x 2 x max SM clock
PROFILE_CSV = os.path.join(ROOT, "profiles", "r03_roofline.csv")


def workload_desc(w):
    return (f"{w.name}: N={w.n} {w.note}, G={w.G:g}, eps={w.eps:g}, theta={w.theta:g}, leaf cap {w.leaf_cap}, "
            f"W=32, Gc=512, KDK dt={w.dt:g}")


def config_dict(w, world: int):
    """The `config` object of BOTH arms (the driver compares them): the workload and how the timed region treats the
    caches.  What a run found out about the workload (tree size, sample) goes into other keys."""
    return {"workload": workload_desc(w), "parallelism": "replicas only" if world > 1 else "1 gpu",
            "l2": "own arm: L2 flushed between steps (256 MiB write), per-step CUDA events summed; "
                  "reference arm: the oracle on host cores, bounded sample of the workload"}


def source_sha1(files: str) -> str:
    """sha1 over the contents of the CUDA sources a kernel is compiled from (';'-separated names under csrc/), the
    fingerprint a row of the profile CSV carries: a row whose sources have changed since its capture is stale."""
    import hashlib
    h = hashlib.sha1()
    for name in files.split(";"):
        with open(os.path.join(ROOT, "paper_1912_04197_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def profile_row(kernel: str, config: str):
    """Profiler figures of one kernel launch (dram bytes, L2 hit rate, ...) from the committed summary of the
    ncu --set full captures, profiles/r03_roofline.csv (its .md names the commands and the commit).  The row gets
    "stale": True when the kernel's sources no longer hash to what they did at the capture."""
    import csv
    try:
        with open(PROFILE_CSV) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel and row["config"] == config:
                    try:
                        row["stale"] = source_sha1(row["source_files"]) != row["source_sha1"]
                    except (OSError, KeyError):
                        row["stale"] = True
                    return row
    except OSError:
        pass
    return None


class Microbench:
    """libbh_microbench.so: measurement-only kernels (fp64 FMA rate, the walk's evaluation loop alone)."""

    def __init__(self):
        import ctypes as C
        from paper_1912_04197_b200 import build as pbuild
        self.C = C
        self.lib = C.CDLL(pbuild.MICRO_LIB)
        for name in ("bhmb_fp64_peak", "bhmb_issue_model", "bhmb_fp64_mma"):
            getattr(self.lib, name).restype = C.c_int
            getattr(self.lib, name).argtypes = [C.c_void_p, C.POINTER(C.c_double)]

    def fp64_peak(self, stream) -> float:
        v = self.C.c_double()
        if self.lib.bhmb_fp64_peak(stream.cuda_stream, self.C.byref(v)) != 0:
            raise RuntimeError("bhmb_fp64_peak failed")
        return v.value

    def fp64_mma(self, stream):
        """The fp64 tensor-core MMA against the vector fp64 pipe: rates alone and whether they overlap."""
        v = (self.C.c_double * 3)()
        if self.lib.bhmb_fp64_mma(stream.cuda_stream, v) != 0:
            raise RuntimeError("bhmb_fp64_mma failed")
        return {"dfma_tflops": v[0], "dmma_m8n8k4_tflops": v[1], "interleaved_time_over_sum_of_times_alone": v[2]}

    def issue_model(self, stream):
        v = (self.C.c_double * 3)()
        if self.lib.bhmb_issue_model(stream.cuda_stream, v) != 0:
            raise RuntimeError("bhmb_issue_model failed")
        return {"eval_loop_alone": v[0], "beside_low_duty_integer_warps": v[1], "beside_full_rate_integer_warps": v[2]}


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
    rng = np.random.default_rng(1912041970 + seed)    # fixed: the same chunks in every run with the same budget
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
            f"{len(starts)} chunks of 32 groups at seeded offsets (seed 1912041970+{seed}; the count follows a "
            f"{budget_s:g} s budget calibrated on {cal} groups) ({t_walk:.2f} s)")
    return value, desc, cores


def oracle_context(w, budget_s: float = 10.0):
    """The two oracle timings SURVEY.md 8(d) lists for scale beside the headline (PAPER.md:194-197 gives the paper's
    own CPU/GPU context): (i) the oracle on ONE thread at configs[2] (N = 131072, theta = 0.5), bounded sample;
    (ii) the oracle's direct sum, Eq. (1), on 4096 targets of this workload, the full N^2 time extrapolated
    x N/4096 and labelled so."""
    import ctypes as C
    import numpy as np
    from oracle import bh_oracle as orc
    from paper_1912_04197_b200 import workloads as wl
    out = {}
    cores = orc.num_threads()
    gomp = None
    try:
        gomp = C.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(1)
        w3 = wl.make("c3")
        t0 = time.perf_counter()
        t3 = orc.build(w3.pos, w3.mass, w3.leaf_cap)
        tb = time.perf_counter() - t0
        ng = t3.ngroups
        step = 4
        t0 = time.perf_counter()
        bodies = 0
        for g0 in range(0, ng, step):                   # every step-th group until the budget is spent
            orc.accel(t3, 0.5, w3.eps, w3.G, g0, g0 + 1)
            bodies += int(t3.gstart[g0 + 1] - t3.gstart[g0])
            if time.perf_counter() - t0 > budget_s:
                break
        tw = time.perf_counter() - t0
        out["single_thread_c3"] = {"value": bodies / (tb * bodies / w3.n + tw), "unit": UNIT, "cores": 1,
                                   "sample": f"c3 N={w3.n} theta=0.5: full build ({tb:.2f} s, prorated) + walk of {bodies} "
                                             f"bodies (every {step}-th group, {tw:.2f} s)"}
    except OSError:
        out["single_thread_c3"] = None
    finally:
        if gomp is not None:
            gomp.omp_set_num_threads(cores)
    nt = min(4096, w.n)
    tg = np.arange(0, w.n, max(1, w.n // nt), dtype=np.int32)[:nt]
    t0 = time.perf_counter()
    orc.direct(w.pos, w.mass, w.eps, w.G, targets=tg)
    td = time.perf_counter() - t0
    out["direct_sum"] = {"targets": int(nt), "seconds": td, "interactions_per_s": nt * float(w.n) / td, "cores": cores,
                         "full_n2_seconds_extrapolated": td * w.n / nt, "extrapolated": nt != w.n,
                         "body_accelerations_per_s": nt / td}
    return out


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
            "data": "synthetic", "config": config_dict(w, args.gpus),
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
    l0 = bh.bh_get_launches(ctx.ctx)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phase_sum = {k: 0.0 for k in bh.PHASE_NAMES}
    walk_ms, inter = [], []
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        # per-phase events (two per phase inside the step, and a sync to read them) on a sample of the steps only: they
        # cost the step ~35 us of gaps between its kernels (5.245 against 5.281 ms at c4 with them on every step)
        sample = args.phases or k < 8 or k == args.steps - 1
        bh.bh_set_timing(ctx.ctx, sample)
        flush.zero_()                                   # evict L2 between timed iterations
        ev[k][0].record(stream)
        bh.bh_kdk_step(ctx.ctx, dt)
        ev[k][1].record(stream)
        if sample:
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
    mb = Microbench()
    # ONE denominator: the best DFMA rate this run measured (two kernels of libbh_microbench.so time the same eight
    # register-resident chains per thread; they differ in loop shape only)
    mma = mb.fp64_mma(stream)
    peak_meas = max(mb.fp64_peak(stream), mma["dfma_tflops"])
    issue = mb.issue_model(stream)
    prof = profile_row("walk_kernel", w.name)
    roofline = {"bound": "alu", "kernel": "walk_kernel", "achieved": achieved, "peak": peak_meas,
                "unit": "TFLOP/s", "frac": achieved / peak_meas,
                "peak_source": "best fp64 FMA rate measured in this run (register-resident DFMA chains on every SM, "
                               "libbh_microbench.so: max of bhmb_fp64_peak and bhmb_fp64_mma's DFMA leg); "
                               "MEASURED_PEAKS.json has no fp64 entry",
                "peak_nominal": FP64_NOMINAL_TFLOPS, "frac_of_nominal": achieved / FP64_NOMINAL_TFLOPS,
                "flops_per_interaction": FLOPS_PER_INTERACTION, "interactions_per_launch": inter_avg,
                "interactions_per_s": inter_avg / (walk_avg_ms * 1e-3), "kernel_ms": walk_avg_ms,
                "issue_model_interactions_per_s": issue, "fp64_tensor_core": mma,
                "frac_of_eval_loop_alone": inter_avg / (walk_avg_ms * 1e-3) / issue["eval_loop_alone"],
                "traffic": float(prof["dram_bytes_per_launch"]) if prof else None,
                "l2_hit_rate": float(prof["l2_hit_pct"]) / 100.0 if prof else None,
                "fp64_pipe_active": float(prof["fp64_pipe_pct"]) / 100.0 if prof else None,
                "profile_source": (f"profiles/r03_roofline.csv (ncu --set full at commit {prof['commit']}; profiler "
                                   "figures, not measured by this run)") if prof else None,
                "profile_stale": bool(prof["stale"]) if prof else None}
    # build kernels against HBM: algorithmic bytes per body over the time of the SAME phases.
    # Inside a KDK step above the one-kernel builds' sizes the drift kernel takes the bounding cube (step a1): that pass
    # is timed under "kick_drift", phases["cube"] is 0, and a1's 24 B/body leave the numerator with it.
    build_ms = sum(phases[k] for k in ("cube", "keys", "sort", "gather", "tree", "monopoles"))
    cube_in_drift = phases["cube"] == 0.0 and phases["keys"] > 0.0
    survey_bytes = 390 - (24 if cube_in_drift else 0)      # eight sort passes, boxes re-read the bodies
    executed_bytes = survey_bytes - 32 - 48                # boxes taken from registers (-32), six sort passes of eight (-48)
    hbm_peak, hbm_source = 6650.0, "B200_PROFILING.md fallback (MEASURED_PEAKS.json absent): of fallback"
    try:
        hbm_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
        hbm_source = "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        pass
    gbs = lambda b: b * w.n / (build_ms * 1e-3) / 1e9
    build_roof = {"bound": "hbm", "achieved": gbs(survey_bytes), "peak": hbm_peak, "peak_source": hbm_source,
                  "unit": "GB/s", "frac": gbs(survey_bytes) / hbm_peak,
                  "algorithmic_bytes_per_body": survey_bytes,
                  "count": "SURVEY.md 8(d) count for the phases in build_ms (390 B/body with step a1, 366 without)",
                  "cube_in_drift": cube_in_drift,
                  "executed_bytes_per_body": executed_bytes, "achieved_executed": gbs(executed_bytes),
                  "frac_executed": gbs(executed_bytes) / hbm_peak,
                  "executed_count": "as executed: group boxes from registers (-32 B), 5 digit passes + repair instead "
                                    "of 8 passes (-48 B)",
                  "build_ms": build_ms}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": max(3, args.warmup), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": config_dict(w, world), "tree": {"nodes": M, "depth": depth, "groups": ng},
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
        dprof = profile_row("direct_kernel", w.name)
        dtf = FLOPS_PER_INTERACTION * pairs / (dms * 1e-3) / 1e12
        out["direct"] = {"targets": int(tg.numel()), "ms": dms, "full_n2_ms": direct_full_ms,
                         "extrapolated": tg.numel() != w.n, "interactions_per_s": pairs / (dms * 1e-3),
                         "roofline": {"bound": "alu", "kernel": "direct_kernel", "achieved": dtf, "peak": peak_meas,
                                      "unit": "TFLOP/s", "frac": dtf / peak_meas, "frac_of_nominal": dtf / FP64_NOMINAL_TFLOPS,
                                      "traffic": float(dprof["dram_bytes_per_launch"]) if dprof else None,
                                      "l2_hit_rate": float(dprof["l2_hit_pct"]) / 100.0 if dprof else None,
                                      "fp64_pipe_active": float(dprof["fp64_pipe_pct"]) / 100.0 if dprof else None,
                                      "profile_stale": bool(dprof["stale"]) if dprof else None}}
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
                      "ms_per_step": te * 1e3, "call": "bh_eval_host (pinned host pos+mass in, acc out; mass upload beside the "
                              "first build kernels; the walk stores into the pinned output, no D2H copy; no state between calls)"}

        # ---- rows "next" of SURVEY.md 8(f), timed beside the headline ----
        if not args.no_next:
            out["next_rows"] = next_rows(ctx, w, pos0, vel0, mass, dev, hbm_peak)

        # ---- the oracle on the host cores, bounded sample ----
        if not args.no_cpu:
            v, desc, cores = oracle_sample(w, args.cpu_budget)
            out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
            if not args.no_cpu_context:
                out["cpu_baseline"]["context"] = oracle_context(w)
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
    ap.add_argument("--no-cpu-context", action="store_true",
                    help="skip the two extra oracle timings (single thread at c3, direct sum on 4096 targets)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_own(args)


if __name__ == "__main__":
    main()
