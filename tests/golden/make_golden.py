"""Writes tests/golden/c1_oracle.json from the ORACLE ALONE (never from the CUDA path).

A regression fixture: it freezes what oracle/ computes today for configs[0] (N=1024, C=8,
theta=0.5, eps=1e-3) so that a later, unannounced change to the oracle's
arithmetic or to the input generator shows up as a diff.  The paper prints no worked numeric
example for this path (PAPER.md has none for keys, tree or forces), so no value here is "the
paper's"; correctness pins live in tests/test_oracle_*.py.

    python tests/golden/make_golden.py
"""
import hashlib
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import bh_oracle as orc                      # noqa: E402
from paper_1912_04197_b200 import workloads as wl        # noqa: E402


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def main():
    w = wl.make("c1")
    t = orc.build(w.pos, w.mass, w.leaf_cap)
    acc, nm, nd, _ = orc.accel(t, w.theta, w.eps, w.G)
    ad = orc.direct(w.pos, w.mass, w.eps, w.G)
    out = {
        "config": "c1: N=1024 uniform unit ball, m=1/N, G=1, eps=1e-3, theta=0.5, C=8, W=32, Gc=512",
        "pos_sha256": sha(w.pos), "lo_hex": [float(x).hex() for x in t.lo], "L": t.L,
        "M": t.M, "depth": t.depth, "nodes_per_level": np.bincount(t.level).tolist(),
        "key_sha256": sha(t.key), "perm_sha256": sha(t.perm),
        "topology_sha256": sha(np.concatenate([t.level.astype(np.int64), t.begin, t.count, t.first_child,
                                               t.child_mask, t.parent]).astype(np.int64)),
        "mono_sha256": sha(t.mono), "n_groups": t.ngroups, "gstart_sha256": sha(t.gstart),
        "n_mono_sum": int(nm.sum()), "n_direct_sum": int(nd.sum()),
        "acc_first3_hex": [[float(x).hex() for x in r] for r in acc[:3]],
        "direct_first3_hex": [[float(x).hex() for x in r] for r in ad[:3]],
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(path)


if __name__ == "__main__":
    main()
