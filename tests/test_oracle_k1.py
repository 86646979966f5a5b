"""Pins for the oracle's Dehnen K1 compensating softening kernel (reading O6b of DESIGN.md; "using a Dehnen K1
compensating smoothing kernel (Dehnen 2001) for small-scale force softening").  Dehnen (2001) is not available: the kernel is rebuilt
from the properties that define it, and these tests pin exactly those properties."""
import math

import numpy as np
import pytest

from paper_1407_2600_b200 import workloads


def _erms(a, b):
    return math.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


def test_k1_defining_properties(orc):
    h = 0.37
    with orc.softening("k1"):
        f = lambda r: orc.soft_pair(r * r, h)[0]          # noqa: E731   acc = -m d f  ->  radial force per unit mass = -r f(r)
        phi = lambda r: orc.soft_pair(r * r, h)[1]        # noqa: E731
        # exactly Newtonian outside the support
        for r in (h, 1.0001 * h, 2 * h, 10 * h):
            assert abs(f(r) * r ** 3 - 1.0) < 1e-14 and abs(phi(r) * r - 1.0) < 1e-14
        # continuity at h of the force, of its derivative (the density vanishes at h) and of the potential
        d = 1e-6 * h
        assert abs(f(h - d) * (h - d) - f(h + d) * (h + d)) < 1.01 * 2 * d * 2 / h ** 3     # no jump: only the slope -2/h^3 times 2d
        dF_in = (f(h - d) * (h - d) - f(h - 2 * d) * (h - 2 * d)) / d
        dF_out = (f(h + 2 * d) * (h + 2 * d) - f(h + d) * (h + d)) / d
        assert abs(dF_in - dF_out) < 1e-4 * abs(dF_out)
        assert abs(phi(h - d) - phi(h + d)) < 1e-5 / h
        # the force is minus the gradient of the potential inside
        for r in (0.1 * h, 0.5 * h, 0.9 * h):
            g = (phi(r + d) - phi(r - d)) / (2 * d)       # d phi/dr, with pot = -m phi: a_r = +m dphi/dr = -m r f
            assert abs(g + r * f(r)) < 1e-6 / h ** 2
        assert abs(phi(0.0) * h - 105.0 / 32.0) < 1e-14   # central potential -(105/32) m/h
        # enclosed mass M(r) = r^3 f(r) (Gauss): density from its derivative; unit mass and ZERO SECOND MOMENT (the compensation)
        x, w = np.polynomial.legendre.leggauss(40)
        r = 0.5 * h * (x + 1.0); wr = 0.5 * h * w
        M = lambda rr: rr ** 3 * f(rr)                      # noqa: E731
        rho = np.array([(M(ri + 1e-6 * h) - M(ri - 1e-6 * h)) / (2e-6 * h) / (4 * math.pi * ri * ri) for ri in r])
        u = (r / h) ** 2
        assert np.max(np.abs(rho - 105.0 / (64 * math.pi * h ** 3) * (1 - u) * (5 - 9 * u))) < 1e-5 * np.abs(rho).max()      # finite differences of M(r)
        assert abs((wr * 4 * math.pi * r ** 2 * rho).sum() - 1.0) < 1e-6
        assert abs((wr * 4 * math.pi * r ** 4 * rho).sum()) < 1e-6 * h ** 2
        assert rho[-1] < 0 < rho[0]                       # positive core, negative skirt
    # and the default law is untouched afterwards
    fp, pp = orc.soft_pair(0.25, 0.1)
    assert abs(pp - 1 / math.sqrt(0.26)) < 1e-15


def test_k1_direct_sum_two_body_and_momentum(orc):
    h = 0.2
    pos = np.array([[0.25, 0.5, 0.5], [0.35, 0.5, 0.5], [0.9, 0.5, 0.5], [0.9, 0.5, 0.5]], np.float32)
    mass = np.array([1.0, 2.0, 0.5, 0.0], np.float32)
    with orc.softening("k1"):
        acc, pot = orc.direct_iso(pos, mass, h)
        r = float(pos[1, 0]) - float(pos[0, 0]); u = (r / h) ** 2
        fin = (175 / 16 - 147 / 8 * u + 135 / 16 * u * u) / h ** 3
        far = lambda d: 1.0 / d ** 2                       # noqa: E731
        d02 = float(pos[2, 0]) - float(pos[0, 0])
        assert np.isclose(acc[0, 0], 2.0 * r * fin + 0.5 * far(d02), rtol=1e-12)       # inside h from particle 1, Newtonian from 2
        f = mass.astype(np.float64)[:, None] * acc
        assert np.linalg.norm(f.sum(0)) < 1e-13 * np.abs(f).sum()
        # a coincident distinct pair: zero force, central potential
        assert acc[3, 1] == 0 and np.isclose(pot[3] - (-1.0 / (0.9 - 0.25) - 2.0 / (0.9 - 0.35)), -0.5 * 105 / 32 / h, rtol=1e-6)
        pos2, mass2 = workloads.uniform_box(1500)
        a2, _ = orc.direct_iso(pos2, mass2, 0.05)
        f2 = mass2.astype(np.float64)[:, None] * a2
        assert np.linalg.norm(f2.sum(0)) < 1e-13 * np.abs(f2).sum()


@pytest.mark.parametrize("periodic", [False, True])
def test_k1_tree_equals_direct_and_is_newtonian_far(orc, periodic):
    """theta -> 0: the tree's P2P with the K1 law is the direct sum; at theta = 0.5 the far cells are expanded with the NEWTONIAN
    Green's function, which is exact for K1 outside its support because the walk accepts a cell only beyond d - b > h: the error stays
    at the tree-truncation level even with h as large as a cell."""
    h = 0.03
    if periodic:
        pos, mass = workloads.clustered_box(12, 6, cfg=4)
    else:
        pos, mass = workloads.plummer_sphere(4000, a=0.02, cfg=2)
    n = len(pos)
    sink = np.arange(0, n, max(1, n // 200))
    with orc.softening("k1"):
        ref = (orc.direct_per(pos, mass, 1.0, h, sink) if periodic else orc.direct_iso(pos, mass, h, sink))[0]
        t = orc.OracleTree(pos, mass, 1.0, periodic)
        a0, _, _, nm0, _ = orc.tree_force(pos, mass, 1.0, periodic, h, 1e-6, 4, sink, tree=t)
        assert nm0 == 0 and _erms(a0, ref) < (3e-4 if periodic else 1e-12)          # periodic: the WS = 1 far-field floor
        a1, _, _, nm1, _ = orc.tree_force(pos, mass, 1.0, periodic, h, 0.5, 4, sink, tree=t)
        assert nm1 > 0 and _erms(a1, ref) < 2e-3
        # with Plummer's softened expansion switched in by mistake the same lists would be wrong at the level (h/d)^2 ~ 1e-2: the gap
        # between the two laws on this input is far above the tree error, so the test sees a mix-up
    plum = (orc.direct_per(pos, mass, 1.0, h, sink) if periodic else orc.direct_iso(pos, mass, h, sink))[0]
    assert _erms(plum, ref) > 10 * _erms(a1, ref)


def test_k1_direct_per_lattice_and_pairwise(orc):
    rng = np.random.default_rng(3)
    n = 30
    pos = rng.random((n, 3), dtype=np.float32)
    mass = rng.uniform(0.5, 1.5, n).astype(np.float32)
    with orc.softening("k1"):
        a1, p1 = orc.direct_per(pos, mass, 1.0, 0.3, pairwise=True)
        a2, p2 = orc.direct_per(pos, mass, 1.0, 0.3)
        assert np.max(np.abs(a1 - a2)) < 1e-10 * np.abs(a1).max() and np.max(np.abs(p1 - p2)) < 1e-10 * np.abs(p1).max()
        lp, lm = workloads.perfect_lattice(4)
        acc, _ = orc.direct_per(lp, lm, 1.0, 0.05)            # compact kernel: the lattice stays exactly force-free
        assert np.max(np.abs(acc)) < 1e-11
