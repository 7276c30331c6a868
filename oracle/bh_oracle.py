"""ctypes wrapper around oracle/libbh_oracle.so — TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this.
It marshals numpy arrays to the C oracle (oracle/bh_oracle.c, steps O1..O11) and composes the steps
in the order of PAPER.md:110-118 (bounding box -> tree -> mass properties -> sort -> forces; here the
sort comes first because the tree is built from sorted keys, reading R16).  No arithmetic of the
method lives in this file.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_morton_key.restype = C.c_uint64
        _lib.orc_morton_key.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32]
        _lib.orc_tree.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def morton_key(qx: int, qy: int, qz: int) -> int:
    return int(lib().orc_morton_key(qx, qy, qz))


def cube(pos: np.ndarray):
    """O1 -> (lo[3], L, e). Raises ValueError on non-finite input."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    lo = np.zeros(3)
    L = C.c_double()
    e = C.c_int32()
    rc = lib().orc_cube(_p(pos), C.c_int64(pos.shape[0]), _p(lo), C.byref(L), C.byref(e))
    if rc != 0:
        raise ValueError("non-finite position")
    return lo, L.value, e.value


def quantise(pos, lo, e) -> np.ndarray:
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    q = np.zeros((pos.shape[0], 3), dtype=np.uint32)
    lib().orc_quantise(_p(pos), C.c_int64(pos.shape[0]), _p(np.ascontiguousarray(lo)), C.c_int32(e), _p(q))
    return q


def morton(pos, lo, e) -> np.ndarray:
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    key = np.zeros(pos.shape[0], dtype=np.uint64)
    lib().orc_morton(_p(pos), C.c_int64(pos.shape[0]), _p(np.ascontiguousarray(lo)), C.c_int32(e), _p(key))
    return key


def sort(key):
    key = np.ascontiguousarray(key, dtype=np.uint64)
    n = key.shape[0]
    perm = np.zeros(n, dtype=np.uint32)
    skey = np.zeros(n, dtype=np.uint64)
    lib().orc_sort(_p(key), C.c_int64(n), _p(perm), _p(skey))
    return perm, skey


@dataclass
class Tree:
    n: int
    C: int
    W: int
    lo: np.ndarray
    L: float
    e: int
    key: np.ndarray          # [n] u64, original order
    perm: np.ndarray         # [n] u32
    skey: np.ndarray         # [n] u64 sorted
    sbody: np.ndarray        # [n,4] sorted (x,y,z,m)
    M: int
    depth: int
    level: np.ndarray        # [M] u8
    begin: np.ndarray        # [M] u32
    count: np.ndarray        # [M] u32
    first_child: np.ndarray  # [M] i32
    child_mask: np.ndarray   # [M] u8
    parent: np.ndarray       # [M] i32
    mono: np.ndarray         # [M,4] (cx,cy,cz,m)
    Gc: int                  # group-cell capacity
    gstart: np.ndarray       # [Ng+1] u32: group g = sorted bodies [gstart[g], gstart[g+1])
    glo: np.ndarray          # [Ng,3]
    ghi: np.ndarray          # [Ng,3]

    @property
    def ngroups(self) -> int:
        return self.gstart.shape[0] - 1


def tree_from_keys(skey: np.ndarray, leaf_cap: int):
    """O5 alone -> (M, depth, level, begin, count, first_child, child_mask, parent)."""
    skey = np.ascontiguousarray(skey, dtype=np.uint64)
    n = skey.shape[0]
    cap = n + 21 * (n // (leaf_cap + 1)) + 1
    level = np.zeros(cap, dtype=np.uint8)
    begin = np.zeros(cap, dtype=np.uint32)
    count = np.zeros(cap, dtype=np.uint32)
    first_child = np.zeros(cap, dtype=np.int32)
    child_mask = np.zeros(cap, dtype=np.uint8)
    parent = np.zeros(cap, dtype=np.int32)
    depth = C.c_int32()
    M = lib().orc_tree(_p(skey), C.c_int64(n), C.c_int32(leaf_cap), C.c_int64(cap), _p(level),
                       _p(begin), _p(count), _p(first_child), _p(child_mask), _p(parent), C.byref(depth))
    if M < 0:
        raise RuntimeError("oracle node capacity bound violated")
    M = int(M)
    return (M, depth.value, level[:M].copy(), begin[:M].copy(), count[:M].copy(),
            first_child[:M].copy(), child_mask[:M].copy(), parent[:M].copy())


def monopoles(sbody, begin, count, first_child, child_mask) -> np.ndarray:
    M = begin.shape[0]
    mono = np.zeros((M, 4), dtype=np.float64)
    lib().orc_monopoles(_p(sbody), C.c_int64(M), _p(begin), _p(count), _p(first_child),
                        _p(child_mask), _p(mono))
    return mono


def group_starts(n, W, Gc, begin, count, first_child, parent) -> np.ndarray:
    """O7: group start indices [Ng+1] (last entry n)."""
    gstart = np.zeros(n + 1, dtype=np.uint32)
    lib().orc_group_starts.restype = C.c_int64
    ng = lib().orc_group_starts(C.c_int64(n), C.c_int64(begin.shape[0]), C.c_int32(W), C.c_int32(Gc),
                                _p(begin), _p(count), _p(first_child), _p(parent), _p(gstart))
    return gstart[:ng + 1].copy()


def group_boxes(sbody, gstart):
    ng = gstart.shape[0] - 1
    glo = np.zeros((ng, 3))
    ghi = np.zeros((ng, 3))
    lib().orc_group_boxes(_p(sbody), _p(gstart), C.c_int64(ng), _p(glo), _p(ghi))
    return glo, ghi


# Reading R6 ("each body is assigned to a thread ... neighbouring threads
# traverse similar sub-trees"): the method's two grouping parameters and the values the reading fixes
# when a caller names none.  They are parameters of the METHOD, owned by this oracle: the CUDA path
# takes them as run-time arguments (bh_create group_size, bh_set_group_cell) and is tested against
# this file at several (W, Gc), not only at the defaults.
R6_W = 32      # bodies that walk the tree together
R6_GC = 512    # group-cell capacity: a group never straddles a tree cell holding <= Gc bodies


def build(pos, mass, leaf_cap: int, W: int = R6_W, Gc: int = R6_GC, gstart=None) -> Tree:
    """O1..O7 in order: cube, keys, sort, gather, tree, monopoles, groups.  W = 1 (any Gc) is the
    paper's per-body walk."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    n = pos.shape[0]
    lo, L, e = cube(pos)
    key = morton(pos, lo, e)
    perm, skey = sort(key)
    sbody = np.zeros((n, 4), dtype=np.float64)
    lib().orc_gather(_p(pos), _p(mass), _p(perm), C.c_int64(n), _p(sbody))
    M, depth, level, begin, count, first_child, child_mask, parent = tree_from_keys(skey, leaf_cap)
    mono = monopoles(sbody, begin, count, first_child, child_mask)
    if gstart is None:
        gstart = group_starts(n, W, Gc, begin, count, first_child, parent)
    gstart = np.ascontiguousarray(gstart, dtype=np.uint32)
    glo, ghi = group_boxes(sbody, gstart)
    return Tree(n, leaf_cap, W, lo, L, e, key, perm, skey, sbody, M, depth, level, begin, count,
                first_child, child_mask, parent, mono, Gc, gstart, glo, ghi)


def walk_lists(t: Tree, g: int, theta: float):
    """O8 for one group -> (monopole node ids, direct sorted-body indices), in visit order."""
    lm = C.POINTER(C.c_int32)()
    ld = C.POINTER(C.c_int32)()
    nm = C.c_int64()
    nd = C.c_int64()
    lib().orc_walk_lists(C.c_double(t.L), C.c_int64(t.n), _p(t.gstart), _p(t.level), _p(t.begin),
                         _p(t.count), _p(t.first_child), _p(t.child_mask), _p(t.mono), _p(t.glo),
                         _p(t.ghi), C.c_int64(g), C.c_double(theta), C.byref(lm), C.byref(nm),
                         C.byref(ld), C.byref(nd))
    a = np.ctypeslib.as_array(lm, shape=(nm.value,)).copy() if nm.value else np.zeros(0, np.int32)
    b = np.ctypeslib.as_array(ld, shape=(nd.value,)).copy() if nd.value else np.zeros(0, np.int32)
    lib().orc_free(lm)
    lib().orc_free(ld)
    return a, b


def accel(t: Tree, theta: float, eps: float, G: float, g0: int = 0, g1: int | None = None,
          want_kappa: bool = False):
    """O8+O9 for groups [g0,g1) -> (acc[n,3] in ORIGINAL body order (rows of other groups are NaN),
    n_mono[g1-g0], n_direct[g1-g0], kappa[n] or None)."""
    if g1 is None:
        g1 = t.ngroups
    acc = np.full((t.n, 3), np.nan)
    n_mono = np.zeros(g1 - g0, dtype=np.uint32)
    n_direct = np.zeros(g1 - g0, dtype=np.uint32)
    kappa = np.full(t.n, np.nan) if want_kappa else None
    lib().orc_accel(C.c_double(t.L), C.c_int64(t.n), _p(t.gstart), _p(t.level), _p(t.begin),
                    _p(t.count), _p(t.first_child), _p(t.child_mask), _p(t.mono), _p(t.sbody),
                    _p(t.perm), _p(t.glo), _p(t.ghi), C.c_double(theta), C.c_double(eps),
                    C.c_double(G), C.c_int64(g0), C.c_int64(g1), _p(acc), _p(n_mono), _p(n_direct),
                    _p(kappa) if want_kappa else None)
    return acc, n_mono, n_direct, kappa


def direct(pos, mass, eps: float, G: float, targets=None, want_kappa: bool = False):
    """O10: Eq. (1). targets=None -> acc[n,3]; else acc[len(targets),3]."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    n = pos.shape[0]
    if targets is None:
        nt, tp = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int32)
        nt, tp = targets.shape[0], _p(targets)
    acc = np.zeros((nt, 3))
    kappa = np.zeros(nt) if want_kappa else None
    lib().orc_direct(_p(pos), _p(mass), C.c_int64(n), tp, C.c_int64(nt), C.c_double(eps),
                     C.c_double(G), _p(acc), _p(kappa) if want_kappa else None)
    return (acc, kappa) if want_kappa else acc


def kick(vel, acc, h: float):
    lib().orc_kick(_p(vel), _p(acc), C.c_int64(vel.shape[0]), C.c_double(h))


def drift(pos, vel, dt: float):
    lib().orc_drift(_p(pos), _p(vel), C.c_int64(pos.shape[0]), C.c_double(dt))


class Leapfrog:
    """O11: KDK state machine with the semantics of include/bh.h bh_kdk_step: the first step
    evaluates a(x0) once; each step is kick(dt/2), drift(dt), rebuild + accel, kick(dt/2)."""

    def __init__(self, pos, vel, mass, theta, eps, G, leaf_cap, W=R6_W, use_direct=False, Gc=R6_GC):
        self.pos = np.array(pos, dtype=np.float64, order="C")
        self.vel = np.array(vel, dtype=np.float64, order="C")
        self.mass = np.ascontiguousarray(mass, dtype=np.float64)
        self.theta, self.eps, self.G, self.C, self.W, self.Gc = theta, eps, G, leaf_cap, W, Gc
        self.use_direct = use_direct
        self.acc = None

    def _eval(self):
        if self.use_direct:
            return direct(self.pos, self.mass, self.eps, self.G)
        t = build(self.pos, self.mass, self.C, self.W, self.Gc)
        return accel(t, self.theta, self.eps, self.G)[0]

    def step(self, dt: float):
        if self.acc is None:
            self.acc = self._eval()
        kick(self.vel, self.acc, dt * 0.5)
        drift(self.pos, self.vel, dt)
        self.acc = self._eval()
        kick(self.vel, self.acc, dt * 0.5)


# ------------------------------------------------------------------ rows "next" of SURVEY.md §8(f)
def potential(t: Tree, theta: float, eps: float, G: float, g0: int = 0, g1: int | None = None):
    """O12: tree potential of the bodies of groups [g0,g1) -> phi[n] in ORIGINAL order (others NaN)."""
    if g1 is None:
        g1 = t.ngroups
    phi = np.full(t.n, np.nan)
    lib().orc_potential(C.c_double(t.L), C.c_int64(t.n), _p(t.gstart), _p(t.level), _p(t.begin),
                        _p(t.count), _p(t.first_child), _p(t.child_mask), _p(t.mono), _p(t.sbody),
                        _p(t.perm), _p(t.glo), _p(t.ghi), C.c_double(theta), C.c_double(eps),
                        C.c_double(G), C.c_int64(g0), C.c_int64(g1), _p(phi))
    return phi


def direct_potential(pos, mass, eps: float, G: float):
    """O13: phi_i = -G sum_{k != i} m_k / sqrt(|R_ik|^2 + eps^2)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    phi = np.zeros(pos.shape[0])
    lib().orc_direct_potential(_p(pos), _p(mass), C.c_int64(pos.shape[0]), C.c_double(eps),
                               C.c_double(G), _p(phi))
    return phi


def diagnostics(pos, vel, mass, phi=None):
    """O14 -> dict(ekin, epot, P[3], L[3])."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    vel = np.ascontiguousarray(vel, dtype=np.float64)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    out = np.zeros(8)
    if phi is not None:
        phi = np.ascontiguousarray(phi, dtype=np.float64)
    lib().orc_diagnostics(_p(pos), _p(vel), _p(mass), _p(phi) if phi is not None else None,
                          C.c_int64(pos.shape[0]), _p(out))
    return {"ekin": out[0], "epot": out[1], "P": out[2:5].copy(), "L": out[5:8].copy()}


def position_error(pos, ref) -> float:
    """O15: Eq. (7), max over bodies, per cent."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    ref = np.ascontiguousarray(ref, dtype=np.float64)
    lib().orc_position_error.restype = C.c_double
    return float(lib().orc_position_error(_p(pos), _p(ref), C.c_int64(pos.shape[0])))


def gravity_dt(G: float, rho: float) -> float:
    """O16: Eq. (8) bound 1 / (2 sqrt(G rho))."""
    lib().orc_gravity_dt.restype = C.c_double
    return float(lib().orc_gravity_dt(C.c_double(G), C.c_double(rho)))


class Stepper:
    """The paper's stepping variants (NEXT-2), composed of the C kick / drift / evaluation steps.

    euler(dt): semi-implicit (symplectic) Euler, the paper's preferred stepper:
        a = a(x_k);  v_{k+1} = fma(a, dt, v_k);  x_{k+1} = fma(v_{k+1}, dt, x_k).
    multirate(dt_c, n_sub): PAPER.md:338-340 — "we advance the simulation of dt_c ... but we evaluate
        gravity (through N^2 interactions or by building the octree) every dt_g": one evaluation
        a = a(x_k), then n_sub semi-implicit Euler sub-steps of dt_c with that same a (dt_g = n_sub dt_c;
        with contacts out of scope nothing else acts between evaluations).
    """

    def __init__(self, pos, vel, mass, theta, eps, G, leaf_cap, W=R6_W, use_direct=False, Gc=R6_GC):
        self.pos = np.array(pos, dtype=np.float64, order="C")
        self.vel = np.array(vel, dtype=np.float64, order="C")
        self.mass = np.ascontiguousarray(mass, dtype=np.float64)
        self.theta, self.eps, self.G, self.C, self.W, self.Gc = theta, eps, G, leaf_cap, W, Gc
        self.use_direct = use_direct
        self.acc = None

    def _eval(self):
        if self.use_direct:
            return direct(self.pos, self.mass, self.eps, self.G)
        t = build(self.pos, self.mass, self.C, self.W, self.Gc)
        return accel(t, self.theta, self.eps, self.G)[0]

    def euler(self, dt: float):
        self.acc = self._eval()
        kick(self.vel, self.acc, dt)
        drift(self.pos, self.vel, dt)

    def multirate(self, dt_c: float, n_sub: int):
        self.acc = self._eval()
        for _ in range(n_sub):
            kick(self.vel, self.acc, dt_c)
            drift(self.pos, self.vel, dt_c)


# ------------------------------------------------------------------ rows NEXT-3 / NEXT-4
def bound_radius(vel, radius, dt: float) -> np.ndarray:
    """O17 (R26): b_i = fma(|v_i|, dt, R_i); vel may be None (b = R)."""
    radius = np.ascontiguousarray(radius, dtype=np.float64)
    b = np.zeros_like(radius)
    if vel is not None:
        vel = np.ascontiguousarray(vel, dtype=np.float64)
    lib().orc_bound_radius(_p(vel) if vel is not None else None, _p(radius), C.c_int64(radius.shape[0]),
                           C.c_double(dt), _p(b))
    return b


def broadphase(pos, b) -> np.ndarray:
    """O17: all pairs i < j with |x_j - x_i|^2 <= (b_i + b_j)^2 -> int32 [P,2], lexicographic."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    n = pos.shape[0]
    f = lib().orc_broadphase
    f.restype = C.c_int64
    total = f(_p(pos), _p(b), C.c_int64(n), None, C.c_int64(0))
    pairs = np.zeros((max(total, 1), 2), dtype=np.int32)
    f(_p(pos), _p(b), C.c_int64(n), _p(pairs), C.c_int64(total))
    return pairs[:total]


def aggregates(n: int, pairs, mass=None):
    """O18 -> dict(label[n], size[n], mass[n] or None, components, aggregates)."""
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    label = np.zeros(n, dtype=np.int32)
    size = np.zeros(n, dtype=np.int32)
    out_mass = np.zeros(n) if mass is not None else None
    if mass is not None:
        mass = np.ascontiguousarray(mass, dtype=np.float64)
    counts = np.zeros(2, dtype=np.int64)
    rc = lib().orc_aggregates(C.c_int64(n), _p(pairs) if pairs.size else None, C.c_int64(pairs.shape[0]),
                              _p(mass) if mass is not None else None, _p(label), _p(size),
                              _p(out_mass) if mass is not None else None, _p(counts))
    if rc != 0:
        raise ValueError("pair index out of range")
    return dict(label=label, size=size, mass=out_mass, components=int(counts[0]), aggregates=int(counts[1]))
