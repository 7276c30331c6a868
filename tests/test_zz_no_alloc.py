"""bh_diagnostics_static: the conserved quantities for callers that cannot allocate.

Who that is: code that is handed device pointers and nothing else.  An analysis hook inside an application
whose memory pool has taken the whole card cannot cudaMalloc the workspace bh_create wants; neither can a
monitor that runs inside a time-step loop, where cudaMalloc / cudaFree would stall every stream of the GPU.
For them libbh keeps the reduction's scratch (592 rows of partial sums and a ticket, 76 032 bytes) in a fixed
array inside the library, and the entry point takes only inputs, an 8-double device output and a stream.

What is checked here: the static-scratch call returns the SAME BITS as bh_diagnostics (same kernel, same
grid, so the same order of additions; the tolerance of tests/test_gpu_next.py would allow 1e-15 of the sum of
|terms|, this test asks for equality), on two calls in a row that share the array: the second call has other
inputs and another size, so anything the first left behind (partial rows, the ticket) would show.  It also
checks that the device's free memory does not move across the calls, and the argument checks.

This file sorts last on purpose (pytest -x stops at the first failure; nothing should hide behind this
one) and must pass alone in a fresh process — where its first libbh call is the static one, before any
context exists — as well as after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_1912_04197_b200 import binding as bh
from paper_1912_04197_b200 import workloads as wl


def _inputs(name, n, seed):
    w = wl.make(name, n)
    rng = np.random.default_rng(seed)
    vel = w.vel if w.vel is not None else rng.standard_normal((n, 3))
    phi = -rng.random(n) - 0.1
    return [torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda() for a in (w.pos, vel, w.mass, phi)]


def _with_context(pos, vel, mass, phi):
    """The existing path: bh_diagnostics on a context with a caller-allocated workspace."""
    ctx = bh.Context(pos.shape[0], 16)
    d = bh.bh_diagnostics(ctx.ctx, pos, vel, mass, phi)
    ctx.close()
    return np.array([d["ekin"], d["epot"], *d["P"], *d["L"]])


@pytest.mark.gpu
def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    # first: 200 000 bodies = more than 592 x 256, so all 592 partial rows are written and every thread
    # strides; second: 70 001 bodies, 274 blocks with a ragged last one, no potential — rows 274..591 of
    # the array then still hold the first call's sums and must not be read
    a = _inputs("c4", 200_000, 3)
    b = _inputs("c5", 70_001, 5)
    out = torch.full((2, 8), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    bh.bh_diagnostics_static(*a, out[0])                            # in a fresh process: the set-up call
    bh.bh_diagnostics_static(b[0], b[1], b[2], None, out[1])        # straight after it, same stream, no wait between
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref_a = _with_context(*a)
    ref_b = _with_context(b[0], b[1], b[2], None)
    assert np.isfinite(got).all()
    assert got[0].tobytes() == ref_a.tobytes(), (got[0], ref_a)
    assert got[1].tobytes() == ref_b.tobytes(), (got[1], ref_b)
    assert got[1][1] == 0.0                                         # epot without phi, as in bh_diagnostics

    # the same two calls again (the array now holds the second call's leftovers), swapped, with the free
    # memory of the device read around them: the library must not have taken or returned a byte
    out2 = torch.full((2, 8), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    bh.bh_diagnostics_static(b[0], b[1], b[2], None, out2[1])
    bh.bh_diagnostics_static(*a, out2[0])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert out2.cpu().numpy().tobytes() == got.tobytes()


@pytest.mark.gpu
def test_static_scratch_small_sets_and_side_stream():
    # one block, one body; and a stream of the caller's own
    for n in (1, 5, 257):
        x = _inputs("c1", n, n)
        out = torch.empty(8, dtype=torch.float64, device="cuda")
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        bh.bh_diagnostics_static(*x, out, stream=s)
        s.synchronize()
        assert out.cpu().numpy().tobytes() == _with_context(*x).tobytes()


def test_static_scratch_rejects_bad_sizes_before_touching_the_gpu():
    # host-side checks come first, so these run without a GPU: fake non-null pointers are never dereferenced
    L = bh.lib()
    p = C.c_void_p(4096)
    assert L.bh_diagnostics_static(p, p, p, None, bh.DIAG_STATIC_MAX_N + 1, p, None) == bh.BH_ERR_CAPACITY
    msg = L.bh_last_error(None).decode()
    assert "BH_DIAG_STATIC_MAX_N" in msg and str(bh.DIAG_STATIC_MAX_N) in msg and str(bh.DIAG_STATIC_MAX_N + 1) in msg
    assert L.bh_diagnostics_static(p, p, p, None, 0, p, None) == bh.BH_ERR_INVALID_ARG
    assert "n < 1" in L.bh_last_error(None).decode()
    for k in (0, 1, 2, 5):
        args = [p, p, p, None, 10, p, None]
        args[k] = None
        assert L.bh_diagnostics_static(*args) == bh.BH_ERR_INVALID_ARG
    assert "null" in L.bh_last_error(None).decode()


def test_static_scratch_size_is_the_stated_one():
    # bh.h states the array's size; the static_assert in bh_diag.cu ties the macro to the kernel's constants,
    # this ties the binding's copy to the header
    import os
    import re
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "bh.h")).read()
    assert int(re.search(r"#define BH_DIAG_STATIC_SCRATCH_BYTES (\d+)", src).group(1)) == bh.DIAG_STATIC_SCRATCH_BYTES \
        == 592 * 8 * 2 * 8 + 256
    assert re.search(r"#define BH_DIAG_STATIC_MAX_N \(\(int64_t\)1 << 30\)", src) and bh.DIAG_STATIC_MAX_N == 1 << 30
