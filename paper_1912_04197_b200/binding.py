"""Thin ctypes binding of libbh (include/bh.h): same call names, argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; torch is used for device memory
and streams.  There is no fallback: if libbh.so is missing, or a call returns a negative status,
this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbh.so")
NUM_PHASES = 9
PHASE_NAMES = ("cube", "keys", "sort", "gather", "tree", "monopoles", "walk", "direct", "kick_drift")

BH_OK, BH_ERR_INVALID_ARG, BH_ERR_CAPACITY, BH_ERR_NONFINITE, BH_ERR_STATE, BH_ERR_CUDA = 0, -1, -2, -3, -4, -5

_lib = None


class BhError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"libbh status {status}: {message}")
        self.status = status


def lib() -> C.CDLL:
    """Load libbh.so (built in-tree by paper_1912_04197_b200.build). Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1912_04197_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i64, dbl, i32 = C.c_void_p, C.c_int64, C.c_double, C.c_int
        L.bh_workspace_bytes.restype = C.c_size_t
        L.bh_workspace_bytes.argtypes = [i64, i32, i32]
        L.bh_last_error.restype = C.c_char_p
        L.bh_last_error.argtypes = [vp]
        L.bh_version.restype = C.c_char_p
        L.bh_gravity_dt.restype = dbl
        L.bh_gravity_dt.argtypes = [dbl, dbl]
        sigs = {
            "bh_create": [C.POINTER(vp), i64, i32, i32, vp, C.c_size_t, vp],
            "bh_destroy": [vp], "bh_set_stream": [vp, vp],
            "bh_build": [vp, vp, vp, i64],
            "bh_accel": [vp, dbl, dbl, dbl, vp],
            "bh_direct": [vp, dbl, dbl, vp],
            "bh_direct_targets": [vp, vp, i64, dbl, dbl, vp],
            "bh_bind_state": [vp, vp, vp, vp, i64, dbl, dbl, dbl],
            "bh_kdk_step": [vp, dbl],
            "bh_get_state_acc": [vp, C.POINTER(vp)],
            "bh_copy_state_acc": [vp, vp],
            "bh_set_gravity_method": [vp, i32],
            "bh_set_graph": [vp, i32],
            "bh_euler_step": [vp, dbl],
            "bh_multirate_step": [vp, dbl, i32],
            "bh_potential": [vp, dbl, dbl, dbl, vp],
            "bh_direct_potential": [vp, dbl, dbl, vp],
            "bh_accel_potential": [vp, dbl, dbl, dbl, vp, vp],
            "bh_diagnostics": [vp, vp, vp, vp, vp, i64, C.POINTER(dbl)],
            "bh_diagnostics_static": [vp, vp, vp, vp, i64, vp, vp],
            "bh_position_error": [vp, vp, vp, i64, C.POINTER(dbl)],
            "bh_broadphase": [vp, vp, vp, dbl, vp, i64, C.POINTER(i64)],
            "bh_aggregates": [vp, i64, vp, i64, vp, vp, vp, vp, C.POINTER(i64)],
            "bh_eval_host": [vp, vp, vp, i64, dbl, dbl, dbl, vp],
            "bh_synchronize": [vp],
            "bh_get_cube": [vp, C.POINTER(dbl), C.POINTER(dbl)],
            "bh_get_keys": [vp, vp, vp],
            "bh_get_node_count": [vp, C.POINTER(i64), C.POINTER(C.c_int32)],
            "bh_get_nodes": [vp, vp, vp, vp, vp, vp, vp, vp],
            "bh_get_groups": [vp, C.POINTER(i64), vp],
            "bh_get_bodies": [vp, vp, vp, vp],
            "bh_get_counts": [vp, vp, vp],
            "bh_get_stats": [vp, C.POINTER(C.c_uint64)],
            "bh_get_launches": [vp, C.POINTER(C.c_uint64)],
            "bh_set_timing": [vp, i32],
            "bh_get_phase_ms": [vp, C.POINTER(C.c_float)],
            "bh_set_group_cell": [vp, i32],
        }
        for name, args in sigs.items():
            f = getattr(L, name)
            f.restype = C.c_int
            f.argtypes = args
        _lib = L
    return _lib


EXPORTS = ("bh_workspace_bytes", "bh_create", "bh_destroy", "bh_set_stream", "bh_build", "bh_accel",
           "bh_direct", "bh_direct_targets", "bh_bind_state", "bh_kdk_step", "bh_get_state_acc",
           "bh_eval_host", "bh_synchronize", "bh_get_cube", "bh_get_keys", "bh_get_node_count",
           "bh_get_nodes", "bh_get_groups", "bh_get_bodies", "bh_get_counts", "bh_get_stats", "bh_get_launches",
           "bh_set_timing",
           "bh_get_phase_ms", "bh_set_group_cell", "bh_last_error", "bh_version",
           "bh_euler_step", "bh_multirate_step", "bh_potential", "bh_direct_potential", "bh_diagnostics",
           "bh_position_error", "bh_gravity_dt", "bh_copy_state_acc", "bh_set_gravity_method",
           "bh_broadphase", "bh_aggregates", "bh_set_graph", "bh_accel_potential", "bh_diagnostics_static")


def _check(ctx, status: int):
    if status != BH_OK:
        raise BhError(status, lib().bh_last_error(ctx).decode())


def _dev(t: torch.Tensor | None, dtype, what: str):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{what}: expected a contiguous CUDA tensor of {dtype}")
    return t.data_ptr()


def _host(t: torch.Tensor, what: str):
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{what}: expected a contiguous CPU float64 tensor")
    return t.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream


# ---- the C calls, one to one ----
def bh_workspace_bytes(max_n: int, leaf_cap: int, group_size: int = 0) -> int:
    return int(lib().bh_workspace_bytes(max_n, leaf_cap, group_size))


def bh_create(max_n: int, leaf_cap: int, group_size: int, workspace: torch.Tensor, stream=None):
    ctx = C.c_void_p()
    st = lib().bh_create(C.byref(ctx), max_n, leaf_cap, group_size, workspace.data_ptr(),
                         workspace.numel() * workspace.element_size(), _stream_ptr(stream))
    _check(None, st)
    return ctx


def bh_destroy(ctx):
    _check(ctx, lib().bh_destroy(ctx))


def bh_set_stream(ctx, stream):
    _check(ctx, lib().bh_set_stream(ctx, _stream_ptr(stream)))


def bh_set_group_cell(ctx, group_cell: int):
    _check(ctx, lib().bh_set_group_cell(ctx, group_cell))


def bh_build(ctx, pos: torch.Tensor, mass: torch.Tensor):
    n = pos.shape[0]
    if pos.dim() != 2 or pos.shape[1] != 3 or mass.shape != (n,):
        raise TypeError("bh_build: pos must be [n,3] and mass [n]")
    _check(ctx, lib().bh_build(ctx, _dev(pos, torch.float64, "pos"), _dev(mass, torch.float64, "mass"), n))


def bh_accel(ctx, theta: float, eps: float, G: float, acc: torch.Tensor):
    _check(ctx, lib().bh_accel(ctx, theta, eps, G, _dev(acc, torch.float64, "acc")))


def bh_direct(ctx, eps: float, G: float, acc: torch.Tensor):
    _check(ctx, lib().bh_direct(ctx, eps, G, _dev(acc, torch.float64, "acc")))


def bh_direct_targets(ctx, targets: torch.Tensor, eps: float, G: float, acc: torch.Tensor):
    _check(ctx, lib().bh_direct_targets(ctx, _dev(targets, torch.int32, "targets"), targets.numel(), eps, G,
                                        _dev(acc, torch.float64, "acc")))


def bh_bind_state(ctx, pos, vel, mass, theta: float, eps: float, G: float):
    _check(ctx, lib().bh_bind_state(ctx, _dev(pos, torch.float64, "pos"), _dev(vel, torch.float64, "vel"),
                                    _dev(mass, torch.float64, "mass"), pos.shape[0], theta, eps, G))


def bh_kdk_step(ctx, dt: float):
    _check(ctx, lib().bh_kdk_step(ctx, dt))


def bh_copy_state_acc(ctx, acc: torch.Tensor):
    _check(ctx, lib().bh_copy_state_acc(ctx, _dev(acc, torch.float64, "acc")))


def bh_set_gravity_method(ctx, method: int):
    _check(ctx, lib().bh_set_gravity_method(ctx, method))


def bh_set_graph(ctx, enable: bool):
    _check(ctx, lib().bh_set_graph(ctx, int(enable)))


def bh_euler_step(ctx, dt: float):
    _check(ctx, lib().bh_euler_step(ctx, dt))


def bh_multirate_step(ctx, dt_c: float, n_sub: int):
    _check(ctx, lib().bh_multirate_step(ctx, dt_c, n_sub))


def bh_potential(ctx, theta: float, eps: float, G: float, phi: torch.Tensor):
    _check(ctx, lib().bh_potential(ctx, theta, eps, G, _dev(phi, torch.float64, "phi")))


def bh_accel_potential(ctx, theta: float, eps: float, G: float, acc: torch.Tensor, phi: torch.Tensor):
    _check(ctx, lib().bh_accel_potential(ctx, theta, eps, G, _dev(acc, torch.float64, "acc"), _dev(phi, torch.float64, "phi")))


def bh_direct_potential(ctx, eps: float, G: float, phi: torch.Tensor):
    _check(ctx, lib().bh_direct_potential(ctx, eps, G, _dev(phi, torch.float64, "phi")))


def bh_diagnostics(ctx, pos, vel, mass, phi=None):
    out = (C.c_double * 8)()
    _check(ctx, lib().bh_diagnostics(ctx, _dev(pos, torch.float64, "pos"), _dev(vel, torch.float64, "vel"),
                                     _dev(mass, torch.float64, "mass"), _dev(phi, torch.float64, "phi"),
                                     pos.shape[0], out))
    return {"ekin": out[0], "epot": out[1], "P": [out[2], out[3], out[4]], "L": [out[5], out[6], out[7]]}


DIAG_STATIC_MAX_N = 1 << 30           # BH_DIAG_STATIC_MAX_N
DIAG_STATIC_SCRATCH_BYTES = 76032     # BH_DIAG_STATIC_SCRATCH_BYTES


def bh_diagnostics_static(pos, vel, mass, phi, out, stream=None, n=None):
    """bh_diagnostics for callers that cannot allocate device memory (include/bh.h): no context and no
    workspace; the reduction's scratch is a fixed array inside libbh.  `out` is a CUDA float64 tensor of 8
    elements that the caller owns; it is filled in stream order (ekin, epot, P[3], L[3]) and the call does
    not wait: synchronise before reading it on the host.  All calls on one GPU share the scratch, so keep them
    in one stream order.  This wrapper allocates nothing either."""
    if out.numel() < 8:
        raise TypeError("out: expected 8 float64 elements on the GPU")
    st = lib().bh_diagnostics_static(_dev(pos, torch.float64, "pos"), _dev(vel, torch.float64, "vel"),
                                     _dev(mass, torch.float64, "mass"), _dev(phi, torch.float64, "phi"),
                                     pos.shape[0] if n is None else n, _dev(out, torch.float64, "out"),
                                     _stream_ptr(stream))
    _check(None, st)
    return out


def bh_position_error(ctx, pos, ref) -> float:
    v = C.c_double()
    _check(ctx, lib().bh_position_error(ctx, _dev(pos, torch.float64, "pos"), _dev(ref, torch.float64, "ref"),
                                        pos.shape[0], C.byref(v)))
    return v.value


def bh_broadphase(ctx, radius, vel, dt: float, pairs: torch.Tensor | None) -> int:
    """Returns the number of pairs found; raises BhError(BH_ERR_CAPACITY) if `pairs` is too small
    (the exception's .count holds the number found)."""
    cnt = C.c_int64()
    cap = 0 if pairs is None else pairs.shape[0]
    st = lib().bh_broadphase(ctx, _dev(radius, torch.float64, "radius"), _dev(vel, torch.float64, "vel"), dt,
                             _dev(pairs, torch.int32, "pairs"), cap, C.byref(cnt))
    if st != BH_OK:
        err = BhError(st, lib().bh_last_error(ctx).decode())
        err.count = cnt.value
        raise err
    return cnt.value


def bh_aggregates(ctx, n: int, pairs: torch.Tensor | None, mass, label, size=None, agg_mass=None):
    counts = (C.c_int64 * 2)()
    npairs = 0 if pairs is None else pairs.shape[0]
    _check(ctx, lib().bh_aggregates(ctx, n, _dev(pairs, torch.int32, "pairs") if npairs else None, npairs,
                                    _dev(mass, torch.float64, "mass"), _dev(label, torch.int32, "label"),
                                    _dev(size, torch.int32, "size"), _dev(agg_mass, torch.float64, "agg_mass"), counts))
    return counts[0], counts[1]


def bh_gravity_dt(G: float, rho: float) -> float:
    return float(lib().bh_gravity_dt(G, rho))


def bh_eval_host(ctx, pos_host, mass_host, theta, eps, G, acc_host):
    _check(ctx, lib().bh_eval_host(ctx, _host(pos_host, "pos"), _host(mass_host, "mass"), pos_host.shape[0],
                                   theta, eps, G, _host(acc_host, "acc")))


def bh_synchronize(ctx):
    _check(ctx, lib().bh_synchronize(ctx))


def bh_get_cube(ctx):
    lo = (C.c_double * 3)()
    side = C.c_double()
    _check(ctx, lib().bh_get_cube(ctx, lo, C.byref(side)))
    return [lo[0], lo[1], lo[2]], side.value


def bh_get_keys(ctx, sorted_key: torch.Tensor | None, perm: torch.Tensor | None):
    _check(ctx, lib().bh_get_keys(ctx, _dev(sorted_key, torch.int64, "sorted_key"), _dev(perm, torch.int32, "perm")))


def bh_get_node_count(ctx):
    m = C.c_int64()
    d = C.c_int32()
    _check(ctx, lib().bh_get_node_count(ctx, C.byref(m), C.byref(d)))
    return m.value, d.value


def bh_get_nodes(ctx, level=None, begin=None, count=None, first_child=None, child_mask=None, parent=None, mono=None):
    _check(ctx, lib().bh_get_nodes(ctx, _dev(level, torch.uint8, "level"), _dev(begin, torch.int32, "begin"),
                                   _dev(count, torch.int32, "count"), _dev(first_child, torch.int32, "first_child"),
                                   _dev(child_mask, torch.uint8, "child_mask"), _dev(parent, torch.int32, "parent"),
                                   _dev(mono, torch.float64, "mono")))


def bh_get_groups(ctx, gstart: torch.Tensor | None = None) -> int:
    ng = C.c_int64()
    _check(ctx, lib().bh_get_groups(ctx, C.byref(ng), _dev(gstart, torch.int32, "gstart")))
    return ng.value


def bh_get_bodies(ctx, sbody=None, glo=None, ghi=None):
    _check(ctx, lib().bh_get_bodies(ctx, _dev(sbody, torch.float64, "sbody"), _dev(glo, torch.float64, "glo"),
                                    _dev(ghi, torch.float64, "ghi")))


def bh_get_counts(ctx, n_mono=None, n_direct=None):
    _check(ctx, lib().bh_get_counts(ctx, _dev(n_mono, torch.int32, "n_mono"), _dev(n_direct, torch.int32, "n_direct")))


def bh_get_stats(ctx):
    s = (C.c_uint64 * 5)()
    _check(ctx, lib().bh_get_stats(ctx, s))
    return {"n_mono": s[0], "n_direct": s[1], "interactions": s[2], "nodes_tested": s[3], "stack_spills": s[4]}


def bh_get_launches(ctx) -> int:
    v = C.c_uint64()
    _check(ctx, lib().bh_get_launches(ctx, C.byref(v)))
    return v.value


def bh_set_timing(ctx, enable: bool):
    _check(ctx, lib().bh_set_timing(ctx, int(enable)))


def bh_get_phase_ms(ctx):
    ms = (C.c_float * NUM_PHASES)()
    _check(ctx, lib().bh_get_phase_ms(ctx, ms))
    return {PHASE_NAMES[i]: ms[i] for i in range(NUM_PHASES)}


# ---- convenience owner of a context and its torch-allocated workspace (no arithmetic) ----
class Context:
    def __init__(self, max_n: int, leaf_cap: int, group_size: int = 0, device="cuda:0", stream=None,
                 group_cell: int | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("libbh needs a CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        self.max_n, self.leaf_cap, self.W = max_n, leaf_cap, group_size or 32
        nbytes = bh_workspace_bytes(max_n, leaf_cap, group_size)
        if nbytes == 0:
            raise BhError(BH_ERR_INVALID_ARG, "max_n, leaf_cap or group_size out of range")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            off = (-self.workspace.data_ptr()) % 256
            self._ws = self.workspace[off:off + nbytes]
            self.ctx = bh_create(max_n, leaf_cap, group_size, self._ws, stream)
            if group_cell is not None:
                bh_set_group_cell(self.ctx, group_cell)
        self.n = 0

    def close(self):
        if self.ctx is not None:
            bh_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def build(self, pos, mass):
        bh_build(self.ctx, pos, mass)
        self.n = pos.shape[0]

    def accel(self, theta, eps, G, out=None):
        out = torch.empty((self.n, 3), dtype=torch.float64, device=self.device) if out is None else out
        bh_accel(self.ctx, theta, eps, G, out)
        return out

    def direct(self, eps, G, targets=None, out=None):
        if targets is None:
            out = torch.empty((self.n, 3), dtype=torch.float64, device=self.device) if out is None else out
            bh_direct(self.ctx, eps, G, out)
        else:
            out = torch.empty((targets.numel(), 3), dtype=torch.float64, device=self.device) if out is None else out
            bh_direct_targets(self.ctx, targets, eps, G, out)
        return out

    def potential(self, theta, eps, G, out=None):
        out = torch.empty(self.n, dtype=torch.float64, device=self.device) if out is None else out
        bh_potential(self.ctx, theta, eps, G, out)
        return out

    def direct_potential(self, eps, G, out=None):
        out = torch.empty(self.n, dtype=torch.float64, device=self.device) if out is None else out
        bh_direct_potential(self.ctx, eps, G, out)
        return out

    def tree(self):
        """Copies of the last build's arrays (torch tensors on the device), for inspection."""
        M, depth = bh_get_node_count(self.ctx)
        d, n = self.device, self.n
        ng = bh_get_groups(self.ctx)
        out = dict(M=M, depth=depth, ng=ng, gstart=torch.empty(ng + 1, dtype=torch.int32, device=d),
                   skey=torch.empty(n, dtype=torch.int64, device=d), perm=torch.empty(n, dtype=torch.int32, device=d),
                   level=torch.empty(M, dtype=torch.uint8, device=d), begin=torch.empty(M, dtype=torch.int32, device=d),
                   count=torch.empty(M, dtype=torch.int32, device=d),
                   first_child=torch.empty(M, dtype=torch.int32, device=d),
                   child_mask=torch.empty(M, dtype=torch.uint8, device=d),
                   parent=torch.empty(M, dtype=torch.int32, device=d),
                   mono=torch.empty((M, 4), dtype=torch.float64, device=d),
                   sbody=torch.empty((n, 4), dtype=torch.float64, device=d),
                   glo=torch.empty((ng, 3), dtype=torch.float64, device=d),
                   ghi=torch.empty((ng, 3), dtype=torch.float64, device=d))
        bh_get_keys(self.ctx, out["skey"], out["perm"])
        bh_get_nodes(self.ctx, out["level"], out["begin"], out["count"], out["first_child"], out["child_mask"],
                     out["parent"], out["mono"])
        bh_get_groups(self.ctx, out["gstart"])
        bh_get_bodies(self.ctx, out["sbody"], out["glo"], out["ghi"])
        out["lo"], out["L"] = bh_get_cube(self.ctx)
        return out

    def counts(self):
        ng = bh_get_groups(self.ctx)
        a = torch.empty(ng, dtype=torch.int32, device=self.device)
        b = torch.empty(ng, dtype=torch.int32, device=self.device)
        bh_get_counts(self.ctx, a, b)
        return a, b
