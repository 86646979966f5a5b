"""Pins for the oracle's background-subtraction pieces (reading O4b of DESIGN.md; "a technique to subtract
the uniform background density"): the closed-form field of a homogeneous cuboid and the moments of a homogeneous cube."""
import math

import numpy as np
import pytest

from paper_1407_2600_b200 import workloads


def _gl3(lo, hi, n):
    """Gauss-Legendre product rule on the cuboid: nodes [m,3] and weights [m]"""
    x, w = np.polynomial.legendre.leggauss(n)
    ax = [0.5 * (hi[d] - lo[d]) * x + 0.5 * (hi[d] + lo[d]) for d in range(3)]
    aw = [0.5 * (hi[d] - lo[d]) * w for d in range(3)]
    X, Y, Z = np.meshgrid(*ax, indexing="ij")
    W = aw[0][:, None, None] * aw[1][None, :, None] * aw[2][None, None, :]
    return np.stack([X.ravel(), Y.ravel(), Z.ravel()], 1), W.ravel()


def test_cuboid_field_known_values_and_symmetry(orc):
    lo, hi = np.array([-0.5, -0.5, -0.5]), np.array([0.5, 0.5, 0.5])
    # potential of the unit cube at its centre: the classical closed form 3 ln(2 + sqrt 3) - pi/2 = 2.38007736...
    centre = 3 * math.log(2 + math.sqrt(3)) - math.pi / 2
    I0, g0 = orc.cuboid_field(lo, hi, [0, 0, 0])
    assert abs(I0 - centre) < 1e-13 and np.max(np.abs(g0)) < 1e-14
    Ic, gc = orc.cuboid_field(lo, hi, [0.5, 0.5, 0.5])
    assert abs(Ic - centre / 2) < 1e-13                            # a corner sees one octant of the cube of side 2: (1/8) 2^2 I0
    assert np.allclose(gc, gc[0]) and gc[0] < 0                    # pulled back towards the cube, equally along the three axes
    # face centre and edge centre are finite; the field is odd, the potential even, cubic symmetry
    for x in ([0.5, 0, 0], [0.5, 0.5, 0], [0.3, -0.2, 0.1], [0.9, 0.4, -1.3]):
        I, g = orc.cuboid_field(lo, hi, x)
        I2, g2 = orc.cuboid_field(lo, hi, [-x[0], -x[1], -x[2]])
        assert np.isfinite(I) and np.all(np.isfinite(g))
        assert abs(I - I2) < 1e-13 and np.max(np.abs(g + g2)) < 1e-13
        I3, g3 = orc.cuboid_field(lo, hi, [x[1], x[2], x[0]])
        assert abs(I - I3) < 1e-13 and np.allclose(g3, [g[1], g[2], g[0]], atol=1e-13)
    # scaling: a cuboid twice as large seen from twice as far: I scales with length^2, g with length
    I, g = orc.cuboid_field([0, 0, 0], [1, 2, 3], [1.5, -0.5, 2.0])
    I2, g2 = orc.cuboid_field([0, 0, 0], [2, 4, 6], [3.0, -1.0, 4.0])
    assert abs(I2 - 4 * I) < 1e-12 * I2 and np.allclose(g2, 2 * g, rtol=1e-12)


def test_cuboid_field_outside_against_quadrature(orc):
    """outside the cuboid the integrand is smooth: a 48^3 Gauss-Legendre rule is exact to ~1e-12"""
    rng = np.random.default_rng(1)
    lo, hi = np.array([0.1, -0.3, 0.2]), np.array([0.6, 0.4, 0.45])          # a genuine cuboid, not a cube
    y, w = _gl3(lo, hi, 48)
    for _ in range(6):
        x = rng.uniform(-1, 1, 3)
        x[rng.integers(3)] = rng.choice([-0.9, 1.1])                          # certainly outside
        d = y - x
        r = np.linalg.norm(d, axis=1)
        Iq, gq = (w / r).sum(), (w[:, None] * d / r[:, None] ** 3).sum(0)
        I, g = orc.cuboid_field(lo, hi, x)
        assert abs(I - Iq) < 1e-10 * Iq and np.max(np.abs(g - gq)) < 1e-10 * np.linalg.norm(gq)
    # far away it is a point mass of the cuboid's volume at its centre (corrections ~ (size/d)^2)
    x = np.array([40.0, -30.0, 20.0]); c = 0.5 * (lo + hi); V = np.prod(hi - lo)
    I, g = orc.cuboid_field(lo, hi, x)
    dd = c - x; r = np.linalg.norm(dd)
    assert abs(I - V / r) < 1e-4 * V / r and np.max(np.abs(g - V * dd / r ** 3)) < 1e-4 * V / r ** 2


def test_cuboid_field_against_its_own_multipole_series(orc):
    """A second route that shares nothing with the closed form: the cube's moments (orc_cube_moments) contracted with the
    Taylor coefficients of 1/r (orc_bn, eps = 0) converge to the closed form as (cube size / distance)^(p+1)."""
    s = 0.25
    ctr = np.array([0.375, 0.125, 0.625])
    lo, hi = ctr - s / 2, ctr + s / 2
    z = ctr + np.array([0.03, -0.05, 0.02])                      # expansion centre off the cube's centre: odd moments too
    errs = []
    for dist in (1.0, 2.0):
        x = z + dist * np.array([0.6, -0.64, 0.48])
        I, g = orc.cuboid_field(lo, hi, x)
        C8 = orc.cube_moments(s, ctr, z, 8)
        acc, pot = orc.m2p(8, C8, x - z, 0.0)                    # field of unit positive density: acc = g, pot = -I
        errs.append(np.linalg.norm(acc - g) / np.linalg.norm(g))
        assert abs(pot + I) < 1e-6 * I
    assert errs[0] < 1e-6 and errs[1] < errs[0] / 2 ** 8        # order 8: the error falls at least as 2^-9 per doubling


def test_cuboid_field_inside_poisson_and_gradient(orc):
    """inside: g = grad I and div g = -4 pi (unit density); across a face both are continuous"""
    lo, hi = np.array([0.0, 0.0, 0.0]), np.array([1.0, 0.5, 0.75])
    h = 1e-4
    for x in ([0.3, 0.2, 0.4], [0.9, 0.45, 0.1], [0.5, 0.25, 0.375]):
        x = np.array(x)
        I, g = orc.cuboid_field(lo, hi, x)
        div = 0.0
        for k in range(3):
            e = np.zeros(3); e[k] = h
            Ip, gp = orc.cuboid_field(lo, hi, x + e); Im, gm = orc.cuboid_field(lo, hi, x - e)
            assert abs((Ip - Im) / (2 * h) - g[k]) < 1e-6
            div += (gp[k] - gm[k]) / (2 * h)
        assert abs(div + 4 * math.pi) < 1e-5
    x = np.array([1.0, 0.2, 0.3])                                # on a face
    Im, gm = orc.cuboid_field(lo, hi, x - [1e-9, 0, 0]); Ip, gp = orc.cuboid_field(lo, hi, x + [1e-9, 0, 0])
    I, g = orc.cuboid_field(lo, hi, x)
    assert abs(Ip - Im) < 1e-7 and np.max(np.abs(gp - gm)) < 1e-7 and np.max(np.abs(g - gm)) < 1e-7
    # outside the Laplacian vanishes
    x = np.array([1.4, 0.2, 0.3]); div = 0.0
    for k in range(3):
        e = np.zeros(3); e[k] = h
        div += (orc.cuboid_field(lo, hi, x + e)[1][k] - orc.cuboid_field(lo, hi, x - e)[1][k]) / (2 * h)
    assert abs(div) < 1e-5


def test_cuboid_field_additive_and_on_grid_points(orc):
    """two halves add up to the whole, also seen from points that lie exactly on the planes, edges and corner lines of the
    pieces (a perfect lattice puts particles there): the dropped 0 * ln(0) terms are really 0"""
    lo, hi = np.array([0.0, 0.0, 0.0]), np.array([1.0, 1.0, 1.0])
    mid = np.array([0.5, 1.0, 1.0])
    for x in ([0.5, 0.5, 0.5], [0.5, 0.0, 0.0], [0.5, 1.0, 2.0], [0.0, 0.0, 3.0], [2.0, 1.0, 1.0], [0.25, 0.25, 0.25], [0.5, 1.0, 1.0]):
        I, g = orc.cuboid_field(lo, hi, x)
        I1, g1 = orc.cuboid_field(lo, mid, x)
        I2, g2 = orc.cuboid_field([0.5, 0.0, 0.0], hi, x)
        assert np.isfinite(I) and np.all(np.isfinite(g))
        assert abs(I - I1 - I2) < 1e-13 and np.max(np.abs(g - g1 - g2)) < 1e-13


def test_cube_moments_against_quadrature(orc):
    s = 0.125
    ctr = np.array([0.4375, 0.0625, 0.8125]); z = ctr + np.array([0.02, 0.05, -0.0625])
    y, w = _gl3(ctr - s / 2, ctr + s / 2, 6)                      # exact for polynomials of degree <= 11 per axis
    C = orc.cube_moments(s, ctr, z, 8)
    d = y - z
    for i, (a, b, c) in enumerate(orc.mtable(8)):
        ref = (w * d[:, 0] ** a * d[:, 1] ** b * d[:, 2] ** c).sum()
        assert abs(C[i] - ref) < 1e-13 * s ** 3 * (0.13) ** (a + b + c) + 1e-300, (a, b, c)
    C0 = orc.cube_moments(s, ctr, ctr, 4)                         # about its own centre: volume, no odd moments, s^2/12 per axis
    assert abs(C0[0] - s ** 3) < 1e-18
    for i, (a, b, c) in enumerate(orc.mtable(4)):
        if a % 2 or b % 2 or c % 2:
            assert C0[i] == 0.0
    assert abs(C0[orc.midx(2, 0, 0)] - s ** 5 / 12) < 1e-18 and abs(C0[orc.midx(2, 2, 0)] - s ** 7 / 144) < 1e-20


def test_bg_level_and_halfwidth(orc):
    assert [orc.bg_level(n) for n in (1, 100, 32768, 2 ** 21, 2 ** 24, 2 ** 27)] == [2, 2, 3, 5, 6, 7]
    assert orc.bg_halfwidth(0.5, 5, ws=2) == 2 and orc.bg_halfwidth(1.0, 5, ws=2) == 1 and orc.bg_halfwidth(0.3, 5, ws=2) == 4
    assert orc.bg_halfwidth(0.3, 2, ws=1) == 4 and orc.bg_halfwidth(0.2, 2, ws=1) == 4 and orc.bg_halfwidth(1e-6, 3, ws=2) == 16   # clamped: the window stays in the block


# ---- the whole reading O4b -------------------------------------------------------------------------------
def _clumpy(n, seed, nclump=3, spread=0.02):
    rng = np.random.default_rng(seed)
    c = rng.random((nclump, 3))
    pos = np.mod(c[rng.integers(nclump, size=n)] + spread * rng.standard_normal((n, 3)), 1.0).astype(np.float32)
    pos[pos >= 1.0] = 0.0
    mass = (rng.uniform(0.5, 1.5, n) / n).astype(np.float32)
    return pos, mass


def _erms(a, b):
    return math.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


@pytest.mark.parametrize("case", ["lattice", "clumpy", "three"])
def test_bg_everything_direct_equals_ewald(orc, case):
    """theta -> 0: nothing is accepted, every leaf and every empty octant of the image block is an exposed cube, the window
    and the cubes kept outside it tile the block; what is left is the direct sum over the block's particles, the exact
    background of the block and the order-8 far field of the NEUTRAL box.  Must equal the Ewald direct sum D-per up to the
    far-field truncation, which subtraction makes ~10x smaller than without (WS = 2: 3.9e-6 -> 3.4e-7 on the 16^3 lattice;
    WS = 1: 2.5e-3 -> 1.9e-4)."""
    if case == "lattice":
        pos, mass = workloads.perturbed_lattice(16, cfg=3)
        tol = 1e-6
    elif case == "clumpy":                    # shallow, lopsided tree: coarse leaves and empty octants everywhere
        pos, mass = _clumpy(300, 5)
        tol = 2e-7
    else:                                     # three particles: as far from uniform as it gets (far-field floor 6e-7)
        pos, mass = _clumpy(3, 7)
        tol = 2e-6
    n = len(pos)
    eps = 1.0 / 640
    sink = np.arange(0, n, max(1, n // 48))
    ref, refp = orc.direct_per(pos, mass, 1.0, eps, sink, ws=2)
    acc, pot, _, nm, _ = orc.tree_force(pos, mass, 1.0, True, eps, 1e-6, 4, sink, ws=2, bg=True)
    assert nm == 0
    assert _erms(acc, ref) < tol, _erms(acc, ref)
    assert np.max(np.abs(pot - refp)) < 10 * tol * np.abs(refp).max()
    if case == "lattice":
        plain = orc.tree_force(pos, mass, 1.0, True, eps, 1e-6, 4, sink, ws=2, bg=False)[0]
        assert _erms(acc, ref) < 0.3 * _erms(plain, ref)
    # WS = 1 (the default): the same identity, with the larger far-field floor that goes with the smaller block
    ref1 = orc.direct_per(pos, mass, 1.0, eps, sink, ws=1)[0]
    acc1 = orc.tree_force(pos, mass, 1.0, True, eps, 1e-6, 4, sink, ws=1, bg=True)[0]
    assert _erms(acc1, ref1) < {"lattice": 5e-4, "clumpy": 2e-5, "three": 1e-3}[case], _erms(acc1, ref1)   # measured 3.1e-4, <2e-5, 3.6e-4


@pytest.mark.parametrize("case", ["lattice", "clustered", "clumpy"])
@pytest.mark.parametrize("theta", [0.4, 0.7, 1.0])
def test_bg_lists_tile_the_block(orc, case, theta):
    """The bookkeeping of reading O4b, checked with integers: per group, the cubes of the accepted cells that carry
    subtracted moments, the window, and the cubes kept outside it (minus their overlap with the window) have exactly the
    volume of the image block, (2 WS + 1)^3 boxes - the background of every point is counted once.  Subtracted entries are
    cells of level <= l_b that do not touch the window; no other accepted cell of level <= l_b lies outside it or sticks
    out of it; the particle partition of the lists is untouched."""
    ws = 2
    if case == "lattice":
        pos, mass = workloads.perturbed_lattice(20, cfg=3)
    elif case == "clustered":
        pos, mass = workloads.clustered_box(20, 10, cfg=4)
    else:
        pos, mass = _clumpy(700, 11, nclump=4)
    n = len(pos)
    t = orc.OracleTree(pos, mass, 1.0, True, nleaf=16, ncrit=32)
    t.moments(2)
    lb = orc.bg_level(n)
    cells = t.cells()
    hot = cells["hotkey"]
    lev = cells["level"].astype(np.int64)
    coords = np.zeros((t.ncell, 3), np.int64)
    for c in range(t.ncell):
        pre = int(hot[c]) & ~(1 << (3 * int(lev[c])))
        for b in range(int(lev[c])):
            coords[c, 0] |= ((pre >> (3 * b + 2)) & 1) << b
            coords[c, 1] |= ((pre >> (3 * b + 1)) & 1) << b
            coords[c, 2] |= ((pre >> (3 * b)) & 1) << b
    nimg = (2 * ws + 1) ** 3
    seen_left = 0
    for g in np.random.default_rng(3).choice(t.ngroup, min(40, t.ngroup), replace=False):
        mc, mi, pc, pi, sub, left, win = t.lists(theta, int(g), ws, bg=True, full=True)
        per_img = np.zeros(nimg, np.int64)
        np.add.at(per_img, mi, cells["count"][mc]); np.add.at(per_img, pi, cells["count"][pc])
        assert np.all(per_img == n)
        vol = int(np.prod(win[3:] - win[:3] + 1))
        for c, im, sb in zip(mc, mi, sub):
            if lev[c] > lb:
                assert not sb
                continue
            sh = (orc.image_shift(int(im), 1.0, True, ws)).astype(np.int64)
            lo = (coords[c] << (lb - lev[c])) + (sh << lb)
            hi = lo + (1 << (lb - lev[c])) - 1
            inter = bool(np.all(lo <= win[3:]) and np.all(hi >= win[:3]))
            inside = bool(np.all(lo >= win[:3]) and np.all(hi <= win[3:]))
            assert inter == inside                     # an accepted cell never sticks out of the window
            assert bool(sb) == (not inter)
            if sb:
                vol += 8 ** int(lb - lev[c])
        for lo6 in left:
            lo, hi = lo6[:3], lo6[3:]
            vol += int(np.prod(hi - lo + 1))
            ol, oh = np.maximum(lo, win[:3]), np.minimum(hi, win[3:])
            if np.all(ol <= oh):
                vol -= int(np.prod(oh - ol + 1))
            assert not (np.all(lo >= win[:3]) and np.all(hi <= win[3:]))        # cubes inside the window are not kept
        seen_left += len(left)
        assert vol == nimg * 8 ** lb, (g, vol, nimg * 8 ** lb)
    if case == "clumpy":
        assert seen_left > 0                             # the case does exercise the cubes kept outside the window


def test_bg_moments_of_a_perfect_lattice_vanish(orc):
    """A perfect k^3 lattice IS the uniform background as far as whole lattice cells go: the subtracted monopole of every
    cell that holds whole lattice cells is 0 to roundoff, and so is its dipole; the quadrupole is the discreteness term
    -(M/12) d^2 per axis (d = lattice spacing), the difference between a point lattice and the continuum."""
    kk = 16
    pos, mass = workloads.perfect_lattice(kk)
    t = orc.OracleTree(pos, mass, 1.0, True)
    lb, rho, mb = t.moments_bg(2)
    cm, com, dl, mom = t.moments(2)
    assert lb == orc.bg_level(kk ** 3) and abs(rho - 1.0) < 1e-12
    lev = t.cells()["level"][:len(mb)]
    assert len(mb) == int((t.cells()["level"] <= lb).sum())
    assert np.max(np.abs(mb[:, 0])) < 1e-15 and np.max(np.abs(mb[:, 1:4])) < 1e-16
    i200 = orc.midx(2, 0, 0)
    assert np.allclose(mb[:, i200], -cm[:len(mb)] / 12.0 / kk ** 2, rtol=1e-9, atol=1e-18)


def test_bg_improves_the_near_lattice_error(orc):
    """What the paper says subtraction is for: on a near-uniform periodic box the tree error at fixed theta and
    p drops (measured 1.9x at 20^3 and 3.3x at 32^3 for theta 0.5, p 4); on a clustered box, where the error comes from the halos, it does not
    get worse."""
    for (pos, mass), gain in ((workloads.perturbed_lattice(20, cfg=3), 1.5), (workloads.clustered_box(20, 10, cfg=4), 0.9)):
        n = len(pos)
        eps = 1.0 / 800
        sink = workloads.subsample(3, n, 96)
        ref = orc.direct_per(pos, mass, 1.0, eps, sink)[0]
        t = orc.OracleTree(pos, mass, 1.0, True)
        for theta, p in ((0.5, 4), (0.7, 4)):
            e0 = _erms(orc.tree_force(pos, mass, 1.0, True, eps, theta, p, sink, tree=t, bg=False)[0], ref)
            e1 = _erms(orc.tree_force(pos, mass, 1.0, True, eps, theta, p, sink, tree=t, bg=True)[0], ref)
            assert e1 * gain < e0, (theta, p, e0, e1)
