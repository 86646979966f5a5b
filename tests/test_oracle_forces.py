"""Pins for the oracle's moments, Taylor coefficients, M2P, direct sum and tree evaluation
(SURVEY.md §8(c) O4, O6, D-iso)."""
import itertools
import math

import numpy as np
import pytest

from paper_1407_2600_b200 import workloads


# ---- O4 moments ---------------------------------------------------------------------------------
def test_moments_m2m_equals_p2m(orc):
    pos, mass = workloads.plummer_sphere(3000, cfg=2)
    mass = (mass * np.random.default_rng(0).uniform(0.5, 1.5, len(mass))).astype(np.float32)
    t = orc.OracleTree(pos, mass)
    for p in (2, 4, 6, 8):
        cm, com, dl, mom = t.moments(p)
        m2m = t.moments_m2m(p)
        rank = np.array([sum(n) for n in orc.mtable(p)])
        scale = np.abs(mom).max(axis=0) + 1e-300
        assert np.max((np.abs(m2m - mom) / scale)[:, rank != 1]) < 1e-11
        assert np.max(np.abs(m2m[:, rank == 1])) < 1e-15         # dipole: pure roundoff
        assert abs(cm[0] - mass.astype(np.float64).sum()) < 1e-12
        tab = orc.mtable(p)
        for i, n in enumerate(tab):
            if sum(n) == 1:                                    # dipole about the COM vanishes
                assert np.max(np.abs(mom[:, i])) < 1e-15
        assert np.allclose(mom[:, 0], cm)


def test_moments_closed_forms(orc):
    # single particle: every moment of rank >= 1 is 0; two particles: closed form
    t = orc.OracleTree(np.array([[0.2, 0.3, 0.4]], np.float32), np.array([2.0], np.float32))
    cm, com, dl, mom = t.moments(4)
    assert np.all(mom[0, 1:] == 0) and mom[0, 0] == 2.0
    x1 = np.array([0.25, 0.5, 0.5], np.float32); x2 = np.array([0.75, 0.5, 0.25], np.float32)
    m1, m2 = 1.0, 3.0
    t = orc.OracleTree(np.stack([x1, x2]), np.array([m1, m2], np.float32))
    cm, com, dl, mom = t.moments(6)
    z = (m1 * x1.astype(np.float64) + m2 * x2.astype(np.float64)) / (m1 + m2)
    assert np.allclose(com[0], z)
    assert np.isclose(dl[0], np.linalg.norm(z - 0.5))
    d1, d2 = x1 - z, x2 - z
    for i, (a, b, c) in enumerate(orc.mtable(6)):
        ref = m1 * d1[0] ** a * d1[1] ** b * d1[2] ** c + m2 * d2[0] ** a * d2[1] ** b * d2[2] ** c
        assert np.isclose(mom[0, i], ref, rtol=1e-12, atol=1e-18)


# ---- O6 Taylor coefficients ---------------------------------------------------------------------
def test_bn_closed_forms(orc):
    r = np.array([0.3, -0.7, 0.45]); e2 = 0.01
    R = math.sqrt(r @ r + e2)
    b = orc.bn(3, r, e2)
    I = np.eye(3)
    assert np.isclose(b[0], 1 / R)
    for i in range(3):
        n = [0, 0, 0]; n[i] = 1
        assert np.isclose(b[orc.midx(*n)], -r[i] / R ** 3)
    for i, j in itertools.product(range(3), repeat=2):
        n = [0, 0, 0]; n[i] += 1; n[j] += 1
        d2 = 3 * r[i] * r[j] / R ** 5 - I[i, j] / R ** 3
        fact = math.prod(math.factorial(k) for k in n)
        assert np.isclose(b[orc.midx(*n)], d2 / fact)
    for i, j, k in itertools.product(range(3), repeat=3):
        n = [0, 0, 0]; n[i] += 1; n[j] += 1; n[k] += 1
        d3 = -15 * r[i] * r[j] * r[k] / R ** 7 + 3 * (I[i, j] * r[k] + I[i, k] * r[j] + I[j, k] * r[i]) / R ** 5
        fact = math.prod(math.factorial(q) for q in n)
        assert np.isclose(b[orc.midx(*n)], d3 / fact)


def test_bn_is_taylor_series(orc):
    """g(r + h) = sum_n b_n(r) h^n: check against the function itself, all ranks to 9 at once"""
    r = np.array([0.8, -0.5, 0.6]); e2 = 0.02
    b = orc.bn(9, r, e2)
    tab = orc.mtable(9)
    for hs in (0.02, 0.04):
        h = hs * np.array([0.6, -0.3, 0.74])
        series = sum(b[i] * h[0] ** a * h[1] ** bb * h[2] ** c for i, (a, bb, c) in enumerate(tab))
        exact = 1 / math.sqrt((r + h) @ (r + h) + e2)
        assert abs(series - exact) < 50 * (hs / 1.1) ** 10
    # finite-difference check of one high-rank relation: d/dx b_n = (n_x+1) b_{n+e_x}
    d = 1e-5
    bp = orc.bn(8, r + [d, 0, 0], e2); bm = orc.bn(8, r - [d, 0, 0], e2)
    for i, (a, bb, c) in enumerate(orc.mtable(8)):
        fd = (bp[i] - bm[i]) / (2 * d)
        assert np.isclose(fd, (a + 1) * b[orc.midx(a + 1, bb, c)], rtol=1e-5, atol=1e-7)


def test_m2p_converges_at_rate(orc):
    """error of the order-p expansion falls as (size/distance)^(p+1): doubling d => 2^(p+1)"""
    rng = np.random.default_rng(5)
    src = (0.5 + 0.05 * (rng.random((50, 3)) - 0.5)).astype(np.float32)
    m = rng.uniform(0.5, 1.5, 50).astype(np.float32)
    eps = 1e-3
    t = orc.OracleTree(src, m, nleaf=64)
    for p in (2, 4, 6, 8):
        cm, com, dl, mom = t.moments(p)
        errs = []
        for dist in (0.2, 0.4):
            x = com[0] + dist * np.array([0.6, 0.64, 0.48])
            acc, pot = orc.m2p(p, mom[0], x - com[0], eps * eps)
            d = x - src.astype(np.float64)
            R2 = (d * d).sum(1) + eps * eps
            ref = -(m[:, None] * d / R2[:, None] ** 1.5).sum(0)
            refp = -(m / np.sqrt(R2)).sum()
            errs.append(np.linalg.norm(acc - ref) / np.linalg.norm(ref))
            assert abs(pot - refp) / abs(refp) < 10 * (0.05 / dist) ** (p + 1)
        ratio = errs[0] / errs[1]
        assert 2 ** (p + 1) / 2.5 < ratio < 2 ** (p + 1) * 2.5, (p, ratio)


def test_m2p_single_offcentre_mass(orc):
    """one point mass expanded about a shifted centre reproduces its exact field as p grows"""
    y = np.array([0.05, -0.03, 0.02]); x = np.array([0.5, 0.4, -0.3]); eps2 = 1e-4
    d = x - y; R = math.sqrt(d @ d + eps2)
    ref = -d / R ** 3
    prev = None
    for p in (2, 4, 6, 8):
        mom = np.array([y[0] ** a * y[1] ** b * y[2] ** c for a, b, c in orc.mtable(p)])
        acc, pot = orc.m2p(p, mom, x, eps2)
        err = np.linalg.norm(acc - ref) / np.linalg.norm(ref)
        assert prev is None or err < prev / 20
        prev = err
    assert prev < 1e-7 and abs(pot + 1 / R) < 1e-8


# ---- D-iso --------------------------------------------------------------------------------------
def test_direct_two_body_and_coincident(orc):
    pos = np.array([[0.25, 0.5, 0.5], [0.75, 0.5, 0.5], [0.75, 0.5, 0.5]], np.float32)
    mass = np.array([1.0, 2.0, 0.0], np.float32)
    eps = 0.1
    acc, pot = orc.direct_iso(pos[:2], mass[:2], eps)
    R = math.sqrt(0.25 + 0.01)
    assert np.allclose(acc[0], [2.0 * 0.5 / R ** 3, 0, 0]) and np.allclose(acc[1], [-1.0 * 0.5 / R ** 3, 0, 0])
    assert np.isclose(pot[0], -2.0 / R) and np.isclose(pot[1], -1.0 / R)
    # coincident distinct pair: zero force, -m/eps potential (reading A10)
    pos2 = np.array([[0.5, 0.5, 0.5], [0.5, 0.5, 0.5]], np.float32)
    acc, pot = orc.direct_iso(pos2, np.array([1.0, 3.0], np.float32), eps)
    assert np.all(acc == 0) and np.isclose(pot[0], -3.0 / eps) and np.isclose(pot[1], -1.0 / eps)


def test_direct_momentum(orc):
    pos, mass = workloads.uniform_box(2000)
    mass = (mass * np.random.default_rng(1).uniform(0.5, 2, 2000)).astype(np.float32)
    acc, _ = orc.direct_iso(pos, mass, 1e-3)
    f = (mass.astype(np.float64)[:, None] * acc)
    assert np.linalg.norm(f.sum(0)) < 1e-13 * np.abs(f).sum()


def test_direct_uniform_and_plummer_sphere(orc):
    rng = np.random.default_rng(7)
    n = 40000
    # uniform sphere radius 0.4 about the centre, M = 1
    r = 0.4 * rng.random(n) ** (1 / 3)
    u = rng.standard_normal((n, 3)); u /= np.linalg.norm(u, axis=1)[:, None]
    pos = (0.5 + r[:, None] * u).astype(np.float32)
    mass = np.full(n, 1.0 / n, np.float32)
    # probes: radial field averaged over shells, inside and outside
    # Gauss's law: the shell-averaged radial field is -M_enclosed/r^2; M_enclosed of a uniform
    # sphere is (r/R)^3 up to Poisson noise of this realisation (checked separately at 3 sigma)
    for rad, smooth in ((0.2, -0.2 / 0.4 ** 3), (0.3, -0.3 / 0.4 ** 3), (0.45, -1 / 0.45 ** 2)):
        nenc = np.count_nonzero(r < rad)
        expect = -(nenc / n) / rad ** 2
        assert abs(expect - smooth) / abs(smooth) < 3.0 / math.sqrt(nenc) + 1e-12
        d = rng.standard_normal((1000, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
        probes = (0.5 + rad * d).astype(np.float32)
        allpos = np.concatenate([pos, probes]); allm = np.concatenate([mass, np.zeros(1000, np.float32)])
        acc, _ = orc.direct_iso(allpos, allm, 5e-3, np.arange(n, n + 1000))
        ar = (acc * d).sum(1).mean()
        assert abs(ar - expect) / abs(expect) < 0.01
    # Plummer sphere, a = 0.01 cut at 20a: a_r = -M_enc-renormalised r/(r^2+a^2)^1.5
    pos, mass = workloads.plummer_sphere(n, a=0.01, cut=20.0, cfg=2)
    a = 0.01
    frac = (20.0 ** 2 / (1 + 20.0 ** 2)) ** 1.5                  # mass fraction inside 20a = 0.99626
    assert abs(frac - 0.99626) < 1e-5
    for rad in (0.005, 0.01, 0.03):
        d = rng.standard_normal((1000, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
        probes = (0.5 + rad * d).astype(np.float32)
        allpos = np.concatenate([pos, probes]); allm = np.concatenate([mass, np.zeros(1000, np.float32)])
        acc, _ = orc.direct_iso(allpos, allm, 3e-4, np.arange(n, n + 1000))
        ar = (acc * d).sum(1).mean()
        smooth = -(1 / frac) * rad / (rad ** 2 + a ** 2) ** 1.5
        nenc = np.count_nonzero(np.linalg.norm(pos.astype(np.float64) - 0.5, axis=1) < rad)
        expect = -(nenc / n) / rad ** 2
        assert abs(expect - smooth) / abs(smooth) < 3.0 / math.sqrt(nenc)
        assert abs(ar - expect) / abs(expect) < 0.02


# ---- Tr vs D ------------------------------------------------------------------------------------
def test_tree_equals_direct_as_theta_to_zero(orc):
    pos, mass = workloads.uniform_box(1500)
    t = orc.OracleTree(pos, mass)
    ref, refp = orc.direct_iso(pos, mass, 1e-3)
    acc, pot, n_p2p, n_m2p = t.accel(1e-3, 1e-6, 4)
    assert n_m2p == 0 and n_p2p == 1500 * 1499
    assert np.max(np.abs(acc - ref)) < 1e-13 * np.abs(ref).max()
    assert np.max(np.abs(pot - refp)) < 1e-13 * np.abs(refp).max()


def _erms(a, b):
    return math.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


def test_tree_error_monotone_in_p_and_theta(orc):
    pos, mass = workloads.plummer_sphere(6000, cfg=2)
    sink = workloads.subsample(2, 6000, 500)
    ref, _ = orc.direct_iso(pos, mass, 1e-4, sink)
    t = orc.OracleTree(pos, mass)
    table = {}
    for p in (2, 4, 6, 8):
        for theta in (0.3, 0.5, 0.7, 1.0):
            acc, pot, n_p2p, n_m2p = t.accel(1e-4, theta, p, sink)
            table[(p, theta)] = _erms(acc, ref)
    for theta in (0.3, 0.5, 0.7, 1.0):
        e = [table[(p, theta)] for p in (2, 4, 6, 8)]
        assert all(e[i + 1] < e[i] for i in range(3)), (theta, e)
    for p in (2, 4, 6, 8):
        e = [table[(p, th)] for th in (0.3, 0.5, 0.7, 1.0)]
        assert all(e[i + 1] > e[i] for i in range(3)), (p, e)
        # roughly theta^(p+1): between theta=0.3 and 0.7 expect a factor >~ (0.7/0.3)^(p) at least
        assert e[2] / e[0] > (0.7 / 0.3) ** (p - 1)
    assert table[(4, 0.5)] < 2e-4 and table[(8, 0.3)] < 1e-8


def test_tree_subset_equals_full(orc):
    pos, mass = workloads.uniform_box(3000)
    t = orc.OracleTree(pos, mass)
    full, fp, _, _ = t.accel(1e-3, 0.5, 4)
    sink = np.array([5, 17, 2999, 1234, 0])
    sub, sp, _, _ = t.accel(1e-3, 0.5, 4, sink)
    assert np.array_equal(sub, full[sink]) and np.array_equal(sp, fp[sink])


# ---- O5: the acceptance rule itself (PAPER.md:61 traversal, :73 "grouping and multipole acceptance tests") --------
def _lists_case(orc, periodic):
    rng = np.random.default_rng(21 + int(periodic))
    n = 5000
    c = rng.random((12, 3))
    pos = c[rng.integers(12, size=n)] + 0.03 * rng.standard_normal((n, 3))
    pos[: n // 4] = rng.random((n // 4, 3))
    pos = (np.mod(pos, 1.0) if periodic else np.clip(pos, 0.0, 0.999999)).astype(np.float32)
    pos[pos >= 1.0] = 0.0
    mass = rng.uniform(0.5, 1.5, n).astype(np.float32) / n
    t = orc.OracleTree(pos, mass, 1.0, periodic, nleaf=16, ncrit=32)
    return pos, mass, t


@pytest.mark.parametrize("periodic", [False, True])
@pytest.mark.parametrize("theta", [0.3, 0.7, 1.0])
def test_lists_partition_and_validity(orc, periodic, theta):
    """What the mathematics fixes about the lists of reading O5, whatever the MAC's exact form:
    PARTITION  per group and image, the listed leaves' particles plus the accepted cells' particles are all N
               particles exactly once (every source is summed once, either directly or inside one expansion);
    VALIDITY   for every accepted (cell, image) every sink of the group is farther from the expansion centre
               z_c + nL than every source of the cell (the expansion converges), with the margin the rule promises:
               min sink distance >= d_AABB > s/theta + delta >= max source distance + s (1/theta - sqrt(3)/2);
    RULE       recomputed here from cells(), moments() and the group's box: every accepted entry satisfies
               d^2 > (s/theta + delta)^2 and every listed leaf and every opened ancestor fails it."""
    ws = 1
    pos, mass, t = _lists_case(orc, periodic)
    n = len(pos)
    cm, com, dl, _ = t.moments(2)
    cells, grp = t.cells(), t.groups()
    _, order = t.sorted()
    wp = t.wrapped_pos().astype(np.float64)
    spos = wp[order]
    side = 2.0 ** (-cells["level"].astype(np.float64))
    nimg = (2 * ws + 1) ** 3 if periodic else 1
    # farthest source of every cell from its centre of mass
    rmax = np.array([np.linalg.norm(spos[f:f + c] - com[i], axis=1).max() for i, (f, c) in enumerate(zip(cells["first"], cells["count"]))])
    parent = np.full(t.ncell, -1)
    for c in range(t.ncell):
        for k in range(cells["nchild"][c]):
            parent[cells["child0"][c] + k] = c

    def d2_aabb(bb, z):
        lo = bb[:3].astype(np.float64) - z; hi = z - bb[3:].astype(np.float64)
        d = np.maximum(np.maximum(lo, hi), 0.0)
        return float(d @ d)

    for g in np.random.default_rng(5).choice(t.ngroup, 40, replace=False):
        mc, mi, pc, pi = t.lists(theta, int(g), ws)
        sinks = spos[grp["first"][g]:grp["first"][g] + grp["count"][g]]
        bb = grp["bbox"][g]
        per_img = np.zeros(nimg, np.int64)
        np.add.at(per_img, mi, cells["count"][mc])
        np.add.at(per_img, pi, cells["count"][pc])
        assert np.all(per_img == n), (g, per_img)
        opened = set()
        for c, im in zip(mc, mi):
            z = com[c] + orc.image_shift(int(im), 1.0, periodic, ws)
            dmin = np.linalg.norm(sinks - z, axis=1).min()
            assert dmin > rmax[c] + side[c] * (1.0 / theta - math.sqrt(3) / 2) * (1 - 1e-12) - 1e-15
            assert d2_aabb(bb, z) > (side[c] / theta + dl[c]) ** 2
            a = parent[c]
            while a >= 0 and (a, int(im)) not in opened:
                opened.add((int(a), int(im))); a = parent[a]
        for c, im in zip(pc, pi):
            assert cells["nchild"][c] == 0
            z = com[c] + orc.image_shift(int(im), 1.0, periodic, ws)
            assert not d2_aabb(bb, z) > (side[c] / theta + dl[c]) ** 2
            a = parent[c]
            while a >= 0 and (a, int(im)) not in opened:
                opened.add((int(a), int(im))); a = parent[a]
        for a, im in opened:
            z = com[a] + orc.image_shift(im, 1.0, periodic, ws)
            assert not d2_aabb(bb, z) > (side[a] / theta + dl[a]) ** 2
        # counts agree with the separate counter
        assert t.list_counts(theta, int(g), ws) == (len(mc), len(pc), int(cells["count"][pc].sum()))


def test_lists_hand_built_case(orc):
    """Four particles whose tree and lists are worked out by hand (all coordinates are exact binary fractions):
        S  = (1/16, 1/8, 1/8)  m 1     S' = (3/8, 1/8, 1/8)  m 1     A1 = (13/16, 1/8, 1/8)  m 1     A2 = (15/16, 1/8, 1/8)  m 3
    NLEAF = NCRIT = 1, so every particle is a leaf and a group.  Cells (hotkey): root 1; octant 0 = 8 {S, S'} with leaves
    64 (S) and 68 (S'); octant 4 = 12 {A1, A2} -> its only child 100 (side 1/4, centre (7/8, 1/8, 1/8)) -> leaves 803 (A1), 807 (A2).
    Cell 100: centre of mass x = (13/16 + 3 * 15/16)/4 = 29/32, so delta = 1/32 and s/theta + delta = 1/(4 theta) + 1/32.
    Sink S (group box = the point S, 1/16 off the centre of its own cell): d = 29/32 - 1/16 = 27/32 = 0.84375 from 100's centre of mass.
      theta = 0.30: 0.8333 + 0.03125 = 0.8646 > d  -> 100 is opened, its leaves (d = 0.75, 0.875 > 0.4167 + 0.0884) are accepted.
                    Dropping delta (0.8333 < d) would accept 100 instead.
      theta = 0.31: 0.8065 + 0.03125 = 0.8377 < d  -> 100 is accepted.  Measuring d to the centre of S's cell (1/8, 1/8, 1/8),
                    d = 25/32 = 0.78125 < 0.8377, would open it instead.
    Sink S': d = 29/32 - 3/8 = 17/32 = 0.53125 = 1/(4 * 0.5) + 1/32 EXACTLY at theta = 0.5: the test is strict, 100 is opened
                    (its leaves, d = 0.4375 and 0.5625 > 0.25 + 0.0884, are accepted); '>=' would accept 100."""
    pos = np.array([[1 / 16, 1 / 8, 1 / 8], [3 / 8, 1 / 8, 1 / 8], [13 / 16, 1 / 8, 1 / 8], [15 / 16, 1 / 8, 1 / 8]], np.float32)
    mass = np.array([1, 1, 1, 3], np.float32)
    t = orc.OracleTree(pos, mass, 1.0, False, nleaf=1, ncrit=1)
    cells, grp = t.cells(), t.groups()
    assert [int(h) for h in cells["hotkey"]] == [1, 8, 12, 64, 68, 100, 803, 807]
    cm, com, dl, _ = t.moments(2)
    c100 = list(cells["hotkey"]).index(100)
    assert com[c100][0] == 29 / 32 and dl[c100] == 1 / 32
    assert t.ngroup == 4 and list(grp["first"]) == [0, 1, 2, 3]          # Morton order: S, S', A1, A2
    hk = lambda idx: sorted(int(cells["hotkey"][i]) for i in idx)       # noqa: E731

    mc, _, pc, _ = t.lists(0.30, 0)
    assert hk(mc) == [803, 807] and hk(pc) == [64, 68]
    mc, _, pc, _ = t.lists(0.31, 0)
    assert hk(mc) == [100] and hk(pc) == [64, 68]
    mc, _, pc, _ = t.lists(0.5, 1)
    assert hk(mc) == [803, 807] and hk(pc) == [64, 68]
    # and the sources' side: A1 at theta = 0.5 sees octant 0 as one cell?  cell 8: centre of mass x = 7/32, centre 1/4,
    # delta = 1/32; d = 13/16 - 7/32 = 19/32 = 0.594 < 1.0 + 0.031 -> opened; leaves 64 (delta 1/16, d 0.75 > 0.5625) and
    # 68 (delta 0, d 0.4375 < 0.5) -> 64 accepted, 68 direct; its own cell 12 and sibling leaf 807 are direct.
    mc, _, pc, _ = t.lists(0.5, 2)
    assert hk(mc) == [64] and hk(pc) == [68, 803, 807]


# ---- O5b: the absolute-error acceptance rule ("limit absolute errors ...") ---------------------------------
@pytest.mark.parametrize("p", [2, 4, 6, 8])
def test_mac_bound_holds_for_every_cell(orc, p):
    """E_c(d) = (p+2) Q b^(p-1) / (d^(p+1) (d-b)^2) is an UPPER BOUND: for random cells and random field points at distance
    d > s + delta from the expansion centre, the error of the order-p expansion against the direct sum over the cell's particles
    stays below it (and is not absurdly below: the bound is within a few orders of magnitude for compact cells)."""
    rng = np.random.default_rng(p)
    pos, mass, t = _lists_case(orc, False)
    cm, com, dl, mom = t.moments(p)
    cells = t.cells()
    _, order = t.sorted()
    spos = t.wrapped_pos().astype(np.float64)[order]
    smass = mass.astype(np.float64)[order]
    side = 2.0 ** (-cells["level"].astype(np.float64))
    eps2 = 1e-16
    worst, n = 0.0, 0
    for c in rng.choice(t.ncell, 400, replace=False):
        if cells["count"][c] < 2:
            continue
        f, k = cells["first"][c], cells["count"][c]
        for _ in range(5):
            d = (side[c] + dl[c]) * (1.0 + 3.0 * rng.random() ** 2)
            u = rng.standard_normal(3); u /= np.linalg.norm(u)
            x = com[c] + d * u
            r = x - spos[f:f + k]
            exact = -(smass[f:f + k, None] * r / ((r * r).sum(1) + eps2)[:, None] ** 1.5).sum(0)
            approx, _ = orc.m2p(p, mom[c], x - com[c], eps2)
            err = np.linalg.norm(approx - exact)
            bound = t.mac_bound(int(c), d)
            assert err <= bound * (1 + 1e-9) + 1e-13 * np.linalg.norm(exact), (c, d, err, bound)
            worst = max(worst, err / bound); n += 1
    assert n > 500 and worst > 1e-4                        # the bound is not vacuous


def test_mac_bound_holds_for_subtracted_cells(orc):
    """the same for the background-subtracted copies (O4b): sources = particles - rho_bar over the cube, exact field = direct sum
    minus rho_bar times the closed-form cuboid field; Q' = Q + rho_bar tr C in the bound"""
    rng = np.random.default_rng(9)
    pos, mass = workloads.clustered_box(20, 10, cfg=4)
    t = orc.OracleTree(pos, mass, 1.0, True)
    p = 4
    cm, com, dl, mom = t.moments(p)
    lb, rho, mb = t.moments_bg(p)
    cells = t.cells()
    _, order = t.sorted()
    spos = t.wrapped_pos().astype(np.float64)[order]
    smass = mass.astype(np.float64)[order]
    n = 0
    for c in rng.choice(len(mb), min(len(mb), 150), replace=False):
        lev = int(cells["level"][c]); s = 2.0 ** -lev
        hot = int(cells["hotkey"][c]) & ~(1 << (3 * lev))
        q = [sum(((hot >> (3 * b + sh)) & 1) << b for b in range(lev)) for sh in (2, 1, 0)]
        lo = np.array(q, float) * s; hi = lo + s
        f, k = cells["first"][c], cells["count"][c]
        for _ in range(4):
            d = (s + dl[c]) * (1.0 + 2.0 * rng.random())
            u = rng.standard_normal(3); u /= np.linalg.norm(u)
            x = com[c] + d * u
            r = x - spos[f:f + k]
            exact = -(smass[f:f + k, None] * r / ((r * r).sum(1) + 1e-16)[:, None] ** 1.5).sum(0) - rho * orc.cuboid_field(lo, hi, x)[1]
            approx, _ = orc.m2p(p, mb[c], x - com[c], 1e-16)
            err = np.linalg.norm(approx - exact)
            assert err <= t.mac_bound(int(c), d, sub=True) * (1 + 1e-9) + 1e-13, (c, d, err)
            n += 1
    assert n > 200


@pytest.mark.parametrize("periodic", [False, True])
def test_abs_mac_lists_and_error(orc, periodic):
    """Lists under the absolute-error rule: the particle partition holds; every accepted entry has d > s + delta and
    E_c(d_AABB) <= tol, every listed leaf fails one of the two (recomputed from mac_bound and the group's box); and the
    force error against the direct sum falls with tol."""
    ws = 1
    pos, mass, t = _lists_case(orc, periodic)
    n = len(pos)
    cm, com, dl, _ = t.moments(4)
    cells, grp = t.cells(), t.groups()
    side = 2.0 ** (-cells["level"].astype(np.float64))
    tol = 5.0

    def d_aabb(bb, z):
        lo = bb[:3].astype(np.float64) - z; hi = z - bb[3:].astype(np.float64)
        d = np.maximum(np.maximum(lo, hi), 0.0)
        return math.sqrt(float(d @ d))

    t.set_mac("abs", tol)
    nimg = (2 * ws + 1) ** 3 if periodic else 1
    for g in np.random.default_rng(6).choice(t.ngroup, 25, replace=False):
        mc, mi, pc, pi = t.lists(0.5, int(g), ws)
        per_img = np.zeros(nimg, np.int64)
        np.add.at(per_img, mi, cells["count"][mc]); np.add.at(per_img, pi, cells["count"][pc])
        assert np.all(per_img == n)
        bb = grp["bbox"][g]
        for c, im in zip(mc, mi):
            d = d_aabb(bb, com[c] + orc.image_shift(int(im), 1.0, periodic, ws))
            assert d > side[c] + dl[c] and t.mac_bound(int(c), d) <= tol
        for c, im in zip(pc, pi):
            d = d_aabb(bb, com[c] + orc.image_shift(int(im), 1.0, periodic, ws))
            assert not (d > side[c] + dl[c] and t.mac_bound(int(c), d) <= tol)
    if not periodic:
        sink = np.arange(0, n, 10)
        ref = orc.direct_iso(pos, mass, 1e-3, sink)[0]
        errs, work = [], []
        for tl in (50.0, 5.0, 0.5):
            t.set_mac("abs", tl)
            a, _, n_p2p, n_m2p = t.accel(1e-3, 0.5, 4, sink)
            errs.append(_erms(a, ref)); work.append(n_p2p + n_m2p)
        assert errs[0] > errs[1] > errs[2] and work[0] < work[1] < work[2], (errs, work)
    t.set_mac("theta")
