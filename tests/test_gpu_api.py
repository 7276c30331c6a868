"""GPU tests of the parts of the C ABI the parity tests do not reach: streams, phase timing, launch counts,
the microbenchmarks behind the roofline figures, two contexts side by side."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import binding as bh
from paper_1912_04197_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a, dtype=torch.float64):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype).cuda()


def relerr(a, b):
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


def test_other_stream_and_two_contexts():
    """A context on a non-default stream (bh_create with a stream, then bh_set_stream) and a second context
    interleaved with it give the results of the oracle."""
    w1, w2 = wl.make("c4", 20000), wl.make("c1", 3000)
    r1 = orc.accel(orc.build(w1.pos, w1.mass, 16), w1.theta, w1.eps, w1.G)[0]
    r2 = orc.accel(orc.build(w2.pos, w2.mass, 8), w2.theta, w2.eps, w2.G)[0]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    p1, m1, p2, m2 = dev(w1.pos), dev(w1.mass), dev(w2.pos), dev(w2.mass)
    torch.cuda.synchronize()
    c1 = bh.Context(w1.n, 16, stream=s1)
    c2 = bh.Context(w2.n, 8)
    with torch.cuda.stream(s1):
        c1.build(p1, m1)
        a1 = c1.accel(w1.theta, w1.eps, w1.G)
    c2.build(p2, m2)
    a2 = c2.accel(w2.theta, w2.eps, w2.G)
    bh.bh_synchronize(c1.ctx)
    bh.bh_synchronize(c2.ctx)
    assert relerr(a1.cpu().numpy(), r1).max() <= 1e-11 and relerr(a2.cpu().numpy(), r2).max() <= 1e-11
    bh.bh_set_stream(c1.ctx, s2)                      # move the first context to another stream
    with torch.cuda.stream(s2):
        c1.build(p1, m1)
        a1b = c1.accel(w1.theta, w1.eps, w1.G)
    bh.bh_synchronize(c1.ctx)
    assert np.array_equal(a1b.cpu().numpy(), a1.cpu().numpy())
    c1.close()
    c2.close()


def test_phase_timing_and_launch_count():
    w = wl.make("c4", 200000)     # above one tree tile per SM: the streaming kernels
    ctx = bh.Context(w.n, 16)
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    bh.bh_set_timing(ctx.ctx, True)
    l0 = bh.bh_get_launches(ctx.ctx)
    ctx.build(pos, mass)
    ctx.accel(w.theta, w.eps, w.G)
    assert bh.bh_get_launches(ctx.ctx) - l0 == 2 + 7 + 3 + 1 + 1 + 1     # cube, keys, sort (5 digit passes, repair, fallback), tree x3, gather + boxes, monopoles, walk
    ph = bh.bh_get_phase_ms(ctx.ctx)
    for k in ("cube", "keys", "sort", "gather", "tree", "monopoles", "walk"):
        assert 0.0 < ph[k] < 50.0, (k, ph[k])
    assert ph["direct"] == 0.0
    ctx.direct(w.eps, w.G)
    assert bh.bh_get_phase_ms(ctx.ctx)["direct"] > 0.0
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    l0 = bh.bh_get_launches(ctx.ctx)
    bh.bh_kdk_step(ctx.ctx, 1e-3)                    # first step: a(x0) once more
    bh.bh_kdk_step(ctx.ctx, 1e-3)
    assert bh.bh_get_launches(ctx.ctx) - l0 == 2 * 16 + 15      # a(x0): build 14 + walk; a step: kick+drift (with the cube), 13, walk, kick
    ph = bh.bh_get_phase_ms(ctx.ctx)
    assert ph["kick_drift"] > 0.0 and ph["walk"] > 0.0
    # a build reports the phases it ran: this step's cube was taken by the drift (part of kick_drift), the direct sum
    # of before is not part of the step
    assert ph["cube"] == 0.0 and ph["direct"] == 0.0
    # ... and a one-kernel build on the context that just ran streaming builds reports its one kernel under "tree"
    ctx.build(pos[:2000].contiguous(), mass[:2000].contiguous())
    ph = bh.bh_get_phase_ms(ctx.ctx)
    assert ph["tree"] > 0.0 and all(ph[k] == 0.0 for k in ("cube", "keys", "sort", "gather", "monopoles"))
    # one sort tile (n <= 4096): the whole build is one launch of one block
    small = bh.Context(2000, 16)
    w2 = wl.make("c1", 2000)
    l0 = bh.bh_get_launches(small.ctx)
    small.build(dev(w2.pos), dev(w2.mass))
    assert bh.bh_get_launches(small.ctx) - l0 == 1
    small.close()
    # up to one tree tile (1024 bodies) per SM: one co-resident kernel with grid barriers
    mid = bh.Context(50000, 16)
    w3 = wl.make("c4", 50000)
    l0 = bh.bh_get_launches(mid.ctx)
    mid.build(dev(w3.pos), dev(w3.mass))
    assert bh.bh_get_launches(mid.ctx) - l0 == 1
    mid.close()
    ctx.close()


def test_sort_survives_a_refused_cooperative_launch():
    """The streaming sort ends with a co-resident (cooperative) kernel that a driver may refuse to launch (MPS, a busy
    partition).  The build must then start its sort again with the eight plain digit passes and keep to them on that
    device, with the same permutation.  BH_TEST_REFUSE_COOPERATIVE_SORT makes the launcher behave as if refused; the
    switch is read once per process, hence the subprocess.  The parity test it runs builds twice per context: the first
    build takes the recovery path, the second the plain passes from the start; 300 coincident bodies need the full
    eight digits."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, BH_TEST_REFUSE_COOPERATIVE_SORT="1")
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-p", "no:cacheprovider",
                        os.path.join(root, "tests", "test_gpu_parity.py"), "-k",
                        "test_partial_key_sort_and_its_fallback and (200000 or 600000)"],
                       env=env, cwd=root, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "4 passed" in r.stdout, r.stdout[-3000:] + r.stderr[-1000:]


def test_state_acc_pointer_and_sorted_bodies():
    w = wl.make("c5", 12000)
    ctx = bh.Context(w.n, 32)
    pos, vel, mass = dev(w.pos), dev(w.vel), dev(w.mass)
    bh.bh_bind_state(ctx.ctx, pos, vel, mass, w.theta, w.eps, w.G)
    ptr = C.c_void_p()
    assert bh.lib().bh_get_state_acc(ctx.ctx, C.byref(ptr)) == bh.BH_ERR_STATE      # no step yet
    bh.bh_kdk_step(ctx.ctx, 1e-3)
    assert bh.lib().bh_get_state_acc(ctx.ctx, C.byref(ptr)) == bh.BH_OK and ptr.value
    a = torch.empty((w.n, 3), dtype=torch.float64, device="cuda")
    bh.bh_copy_state_acc(ctx.ctx, a)
    bh.bh_synchronize(ctx.ctx)
    p = pos.cpu().numpy()
    ref = orc.accel(orc.build(p, w.mass, 32), w.theta, w.eps, w.G)[0]
    assert relerr(a.cpu().numpy(), ref).max() <= 1e-11
    # sorted bodies are the bodies in permutation order, bit for bit
    ctx.n = w.n
    g = ctx.tree()
    perm = g["perm"].cpu().numpy().view(np.uint32)
    sb = g["sbody"].cpu().numpy()
    assert np.array_equal(sb[:, :3], p[perm]) and np.array_equal(sb[:, 3], w.mass[perm])
    ctx.close()


def test_roofline_microbenchmarks_are_sane():
    """The measurement-only library behind bench.py's roofline denominator (not part of libbh)."""
    import bench
    mb = bench.Microbench()
    stream = torch.cuda.current_stream()
    peak = mb.fp64_peak(stream)
    assert 20.0 < peak < 45.0                         # B200: 148 SM x 64 lanes x 2 x <= 1.965 GHz = 37.2 TFLOP/s
    m = mb.issue_model(stream)
    bound = 148 * 4 * 1.965e9                         # one interaction per cycle per sub-partition
    assert 0.6 * bound < m["beside_low_duty_integer_warps"] < m["eval_loop_alone"] <= 1.02 * bound
    assert m["beside_full_rate_integer_warps"] < m["eval_loop_alone"]
    t = mb.fp64_mma(stream)
    # on sm_100 the fp64 MMA runs at the vector fp64 rate and does not overlap with it
    assert 0.8 * peak < t["dmma_m8n8k4_tflops"] < 1.2 * peak and t["interleaved_time_over_sum_of_times_alone"] > 0.85
