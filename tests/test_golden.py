"""The oracle still reproduces the frozen c1 fixture written by tests/golden/make_golden.py."""
import json
import os

import numpy as np

from oracle import bh_oracle as orc
from paper_1912_04197_b200 import workloads as wl
from tests.golden.make_golden import sha


def test_c1_fixture():
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "c1_oracle.json")))
    w = wl.make("c1")
    assert sha(w.pos) == g["pos_sha256"]
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    assert [float(x).hex() for x in t.lo] == g["lo_hex"] and t.L == g["L"]
    assert (t.M, t.depth) == (g["M"], g["depth"])
    assert np.bincount(t.level).tolist() == g["nodes_per_level"]
    assert sha(t.key) == g["key_sha256"] and sha(t.perm) == g["perm_sha256"]
    assert sha(t.mono) == g["mono_sha256"]
    assert t.ngroups == g["n_groups"] and sha(t.gstart) == g["gstart_sha256"]
    acc, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G)
    assert (int(nm.sum()), int(nd.sum())) == (g["n_mono_sum"], g["n_direct_sum"])
    ref = np.array([[float.fromhex(x) for x in r] for r in g["acc_first3_hex"]])
    assert np.abs(acc[:3] - ref).max() <= 1e-15 * np.abs(ref).max()
