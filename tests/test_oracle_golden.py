"""The frozen oracle output of tests/golden/ (a tripwire against silent changes of the oracle's arithmetic)."""
import importlib.util
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def _load():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_oracle_matches_frozen_output():
    now = _load().compute()
    ref = json.load(open(os.path.join(HERE, "golden", "oracle_tiny_case.json")))
    assert now["sorted_keys_hex"] == ref["sorted_keys_hex"] and now["order"] == ref["order"]
    assert now["cells"] == ref["cells"]
    for k in ("tree_p2", "tree_p4"):
        assert now[k]["n_p2p"] == ref[k]["n_p2p"] and now[k]["n_m2p"] == ref[k]["n_m2p"]
        assert np.allclose(now[k]["acc"], ref[k]["acc"], rtol=1e-12, atol=1e-14)
        assert np.allclose(now[k]["pot"], ref[k]["pot"], rtol=1e-12, atol=1e-14)
    assert np.allclose(now["direct"]["acc"], ref["direct"]["acc"], rtol=1e-13, atol=1e-15)
    assert np.allclose(now["periodic_tree_p4_acc"], ref["periodic_tree_p4_acc"], rtol=1e-10, atol=1e-12)
    assert np.allclose(now["periodic_tree_p4_bg_acc"], ref["periodic_tree_p4_bg_acc"], rtol=1e-10, atol=1e-12)
    assert np.allclose(now["periodic_tree_p4_bg_ws1_acc"], ref["periodic_tree_p4_bg_ws1_acc"], rtol=1e-10, atol=1e-12)
    # the two periodic definitions approximate the same Ewald field: they agree to the tree error of this tiny, clumpy case
    a0, a1 = np.array(ref["periodic_tree_p4_acc"]), np.array(ref["periodic_tree_p4_bg_acc"])
    assert np.linalg.norm(a1 - a0) < 5e-3 * np.linalg.norm(a0)
    assert np.allclose(now["kdk_factors_eds"], ref["kdk_factors_eds"], rtol=1e-14)
    assert np.allclose(now["kdk_factors_lcdm"], ref["kdk_factors_lcdm"], rtol=1e-12)
    # the tree sum is an approximation of the direct sum: the frozen case shows the expected convergence in p
    d = np.array(ref["direct"]["acc"])
    e2 = np.linalg.norm(np.array(ref["tree_p2"]["acc"]) - d) / np.linalg.norm(d)
    e4 = np.linalg.norm(np.array(ref["tree_p4"]["acc"]) - d) / np.linalg.norm(d)
    assert e4 < e2 < 1e-2
