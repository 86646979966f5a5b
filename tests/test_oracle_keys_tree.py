"""Pins for the oracle's keys, sort, tree and groups."""
import numpy as np
import pytest

from paper_1407_2600_b200 import workloads


def _interleave_bruteforce(q):
    """bit loop, python ints: x most significant of each triple, placeholder at 2^63"""
    k = 1 << 63
    for b in range(21):
        k |= ((int(q[0]) >> b) & 1) << (3 * b + 2)
        k |= ((int(q[1]) >> b) & 1) << (3 * b + 1)
        k |= ((int(q[2]) >> b) & 1) << (3 * b)
    return k


def test_key_corners(orc):
    one_minus = np.nextafter(np.float32(1.0), np.float32(0.0))
    pos = np.array([[0, 0, 0], [one_minus] * 3], dtype=np.float32)
    k, _ = orc.keys(pos)
    assert int(k[0]) == 1 << 63
    assert int(k[1]) == (1 << 64) - 1


def test_key_single_axis_bits(orc):
    # stepping one axis by 2^-(b+1)... sets exactly bit 3*(20-b)+{2,1,0}
    for axis, off in ((0, 2), (1, 1), (2, 0)):
        for lvl in range(1, 22):
            pos = np.zeros((1, 3), dtype=np.float32)
            pos[0, axis] = 2.0 ** -lvl
            k, _ = orc.keys(pos)
            assert int(k[0]) == (1 << 63) | (1 << (3 * (21 - lvl) + off))


def test_key_bruteforce_random(orc):
    rng = np.random.default_rng(1)
    pos = rng.random((20000, 3), dtype=np.float32)
    k, _ = orc.keys(pos)
    q = np.floor(pos.astype(np.float64) * 2 ** 21).astype(np.int64)   # exact: pos*2^21 is exact
    for i in range(0, 20000, 97):
        assert int(k[i]) == _interleave_bruteforce(q[i])
    # vectorised magic-number-free check of all: de-interleave and compare
    kk = k.astype(np.uint64)
    for axis, off in ((0, 2), (1, 1), (2, 0)):
        v = np.zeros(len(kk), dtype=np.int64)
        for b in range(21):
            v |= (((kk >> np.uint64(3 * b + off)) & np.uint64(1)).astype(np.int64) << b)
        assert np.array_equal(v, q[:, axis])


def test_key_algebra(orc):
    rng = np.random.default_rng(2)
    pos = rng.random((100, 3), dtype=np.float32)
    k, _ = orc.keys(pos)
    for key in k[:20]:
        key = int(key)
        for lvl in range(0, 22):
            hot = key >> (3 * (21 - lvl))
            assert (hot.bit_length() - 1) // 3 == lvl
            if lvl > 0:
                parent = hot >> 3
                assert parent == key >> (3 * (21 - lvl + 1))
                assert (parent << 3) | (hot & 7) == hot
        assert key >> 63 == 1


def test_key_errors_and_wrap(orc):
    with pytest.raises(ValueError):
        orc.keys(np.array([[1.0, 0.5, 0.5]], dtype=np.float32))
    with pytest.raises(ValueError):
        orc.keys(np.array([[-1e-9, 0.5, 0.5]], dtype=np.float32))
    with pytest.raises(ValueError):
        orc.keys(np.array([[np.nan, 0.5, 0.5]], dtype=np.float32))
    pos = np.array([[1.25, -0.25, 3.0], [-1e-10, 0.999999, 1.0]], dtype=np.float32)
    k, w = orc.keys(pos, 1.0, True)
    assert np.allclose(w[0], [0.25, 0.75, 0.0])
    assert w[1, 0] == 0.0 and w[1, 2] == 0.0
    assert np.all((w >= 0) & (w < 1))
    k2, _ = orc.keys(w, 1.0, False)
    assert np.array_equal(k, k2)


def test_sort_stable(orc):
    rng = np.random.default_rng(3)
    for keys in (rng.integers(0, 50, 5000).astype(np.uint64) | np.uint64(1 << 63),      # many ties
                 np.full(1000, 1 << 63, dtype=np.uint64),                                  # all equal
                 (np.arange(3000, 0, -1).astype(np.uint64)),                               # reversed
                 np.where(np.arange(2000) % 2 == 0, np.uint64(7), np.uint64(3)).astype(np.uint64),
                 rng.integers(0, 2 ** 63, 10000).astype(np.uint64)):
        sk, order = orc.sort(keys)
        ref = np.argsort(keys, kind="stable")
        assert np.array_equal(order, ref.astype(np.uint32))
        assert np.array_equal(sk, keys[ref])


def _space_bruteforce(pos, idx, corner, side, level, nleaf, out, hot):
    """recursive subdivision of the point set IN SPACE (no keys): returns cells as (hot, sorted idx)"""
    out.append((hot, tuple(sorted(idx)), 0))
    if len(idx) <= nleaf or level == 21:
        return
    half = side / 2
    nchild = 0
    for o in range(8):
        ox, oy, oz = (o >> 2) & 1, (o >> 1) & 1, o & 1
        c = corner + half * np.array([ox, oy, oz])
        sel = [i for i in idx if np.all(pos[i] >= c) and np.all(pos[i] < c + half)]
        if sel:
            nchild += 1
            _space_bruteforce(pos, sel, c, half, level + 1, nleaf, out, (hot << 3) | o)
    out[[k for k, v in enumerate(out) if v[0] == hot][0]] = (hot, tuple(sorted(idx)), nchild)


@pytest.mark.parametrize("n,seed", [(1, 0), (17, 1), (64, 2), (300, 3)])
def test_tree_vs_spatial_bruteforce(orc, n, seed):
    rng = np.random.default_rng(seed)
    pos = rng.random((n, 3), dtype=np.float32)
    if n >= 64:
        pos[: n // 2] = 0.3 + 0.01 * pos[: n // 2]          # a clump => deeper levels
    mass = np.ones(n, dtype=np.float32)
    t = orc.OracleTree(pos, mass, nleaf=4)
    cells = t.cells()
    skey, order = t.sorted()
    ref = []
    _space_bruteforce(pos.astype(np.float64), list(range(n)), np.zeros(3), 1.0, 0, 4, ref, 1)
    ref.sort(key=lambda v: v[0])
    assert len(ref) == t.ncell
    for c, (hot, members, nchild) in enumerate(ref):
        assert int(cells["hotkey"][c]) == hot
        f, cnt = int(cells["first"][c]), int(cells["count"][c])
        assert tuple(sorted(order[f:f + cnt].tolist())) == members
        assert int(cells["nchild"][c]) == nchild


def test_tree_invariants(orc):
    pos, mass = workloads.plummer_sphere(20000, cfg=2)
    t = orc.OracleTree(pos, mass)
    c = t.cells()
    n = len(pos)
    assert c["first"][0] == 0 and c["count"][0] == n and c["hotkey"][0] == 1
    assert np.all(np.diff(c["hotkey"].astype(np.float64)) > 0) or np.all(c["hotkey"][1:] > c["hotkey"][:-1])
    leaf = c["nchild"] == 0
    assert c["count"][leaf].sum() == n                          # each particle in exactly one leaf
    assert np.all((c["count"][leaf] <= orc.NLEAF) | (c["level"][leaf] == 21))
    assert np.all(c["count"][~leaf] > orc.NLEAF)
    for i in np.nonzero(~leaf)[0][:2000]:
        ch = slice(c["child0"][i], c["child0"][i] + c["nchild"][i])
        assert c["count"][ch].sum() == c["count"][i]            # children tile the parent range
        assert c["first"][ch][0] == c["first"][i]
        assert np.array_equal(c["first"][ch][1:], c["first"][ch][:-1] + c["count"][ch][:-1])
        assert np.all(c["hotkey"][ch] >> np.uint64(3) == c["hotkey"][i])
        assert np.all(c["level"][ch] == c["level"][i] + 1)
    # hotkey of a cell == key >> 3(21-l) of each member
    skey, _ = t.sorted()
    for i in range(0, t.ncell, 37):
        f, cnt, l = int(c["first"][i]), int(c["count"][i]), int(c["level"][i])
        assert np.all(skey[f:f + cnt] >> np.uint64(3 * (21 - l)) == c["hotkey"][i])


def test_coincident_particles_level21(orc):
    nco = 2 * orc.NCRIT + 36                   # coincident particles: one over-full level-21 leaf
    pos = np.tile(np.array([[0.3, 0.4, 0.5]], dtype=np.float32), (nco, 1))
    pos = np.concatenate([pos, np.random.default_rng(0).random((50, 3), dtype=np.float32)])
    t = orc.OracleTree(pos, np.ones(nco + 50, dtype=np.float32))
    c = t.cells()
    deep = c["level"] == 21
    assert deep.any() and c["count"][deep].max() == nco and np.all(c["nchild"][deep] == 0)
    g = t.groups()
    assert g["count"].sum() == nco + 50 and g["count"].max() <= orc.NCRIT
    # the over-full level-21 leaf is cut in chunks of NCRIT
    big = g["cell"] == np.nonzero(deep & (c["count"] == nco))[0][0]
    assert sorted(g["count"][big].tolist()) == [36, orc.NCRIT, orc.NCRIT]


def test_groups(orc):
    pos, mass = workloads.uniform_box(5000)
    t = orc.OracleTree(pos, mass)
    c, g = t.cells(), t.groups()
    assert g["count"].sum() == 5000
    assert np.array_equal(g["first"][1:], g["first"][:-1] + g["count"][:-1]) and g["first"][0] == 0
    assert np.all(g["count"] <= orc.NCRIT)
    # a group is the first cell from the root with count <= NCRIT: its parent has more
    parent = np.full(t.ncell, -1)
    for i in range(t.ncell):
        if c["nchild"][i]:
            parent[c["child0"][i]:c["child0"][i] + c["nchild"][i]] = i
    for k in range(t.ngroup):
        cell = g["cell"][k]
        assert c["count"][cell] == g["count"][k] and c["first"][cell] == g["first"][k]
        assert parent[cell] < 0 or c["count"][parent[cell]] > orc.NCRIT
    # bbox = exact fp32 min/max of members
    _, order = t.sorted()
    for k in range(0, t.ngroup, 7):
        mem = pos[order[g["first"][k]:g["first"][k] + g["count"][k]]]
        assert np.array_equal(g["bbox"][k, :3], mem.min(0)) and np.array_equal(g["bbox"][k, 3:], mem.max(0))
