"""Writes tests/golden/oracle_tiny_case.json: the oracle's own output on a 24-particle case, frozen.

    python tests/golden/make_golden.py

The paper prints no key, tree or force of a worked example, so there is no paper value to store;
the oracle is pinned by closed forms and invariants (tests/test_oracle_*.py).  This fixture is a tripwire:
a later edit to oracle/ that changes its arithmetic shows up as a diff of this file and must name, in its
commit message, the passage or DESIGN.md reading that justifies it.  The script calls only oracle/ (and
numpy for the seeded input); nothing here ever comes from the CUDA path.
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402


def case():
    rng = np.random.Generator(np.random.PCG64(14072600))
    pos = rng.random((24, 3)).astype(np.float32)
    pos[5] = pos[4]                                   # a coincident pair
    mass = rng.uniform(0.5, 1.5, 24).astype(np.float32)
    return pos, mass


def compute():
    pos, mass = case()
    out = {"nleaf": 4, "ncrit": 8, "eps": 0.05, "theta": 0.5}
    t = oracle.OracleTree(pos, mass, 1.0, False, 4, 8)
    skey, order = t.sorted()
    c = t.cells()
    out["sorted_keys_hex"] = [format(int(k), "016x") for k in skey]
    out["order"] = [int(i) for i in order]
    out["cells"] = {k: [int(v) for v in c[k]] if k != "hotkey" else [format(int(v), "x") for v in c[k]]
                    for k in ("hotkey", "first", "count", "nchild")}
    for p in (2, 4):
        a, ph, n_p2p, n_m2p = t.accel(0.05, 0.5, p)
        out[f"tree_p{p}"] = {"acc": a.tolist(), "pot": ph.tolist(), "n_p2p": n_p2p, "n_m2p": n_m2p}
    a, ph = oracle.direct_iso(pos, mass, 0.05)
    out["direct"] = {"acc": a.tolist(), "pot": ph.tolist()}
    tp = oracle.OracleTree(pos, mass, 1.0, True, 4, 8)
    a = oracle.tree_force(pos, mass, 1.0, True, 0.05, 0.5, 4, tree=tp, ws=2, bg=False)[0]
    out["periodic_tree_p4_acc"] = a.tolist()                      # without background subtraction (the round-1 definition)
    a = oracle.tree_force(pos, mass, 1.0, True, 0.05, 0.5, 4, tree=tp, ws=2, bg=True)[0]
    out["periodic_tree_p4_bg_acc"] = a.tolist()                   # reading O4b
    a = oracle.tree_force(pos, mass, 1.0, True, 0.05, 0.5, 4, tree=tp, ws=1, bg=True)[0]
    out["periodic_tree_p4_bg_ws1_acc"] = a.tolist()               # the defaults: subtraction on, 27 images
    out["kdk_factors_eds"] = list(oracle.kdk_factors(True, 1.0, 1.0, 0.5, 0.01))
    out["kdk_factors_lcdm"] = list(oracle.kdk_factors(True, 1.0, 1.0, 0.5, 0.01, (0.295, 0.705)))
    return out


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny_case.json")
    with open(path, "w") as f:
        json.dump(compute(), f, indent=1)
    print(path)
