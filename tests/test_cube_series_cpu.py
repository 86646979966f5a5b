"""The table the CUDA path uses for the window's background (paper_1407_2600_b200/csrc/cube_series.inc: Taylor coefficients of the
interior potential of the homogeneous cube, reading O4b of DESIGN.md) against what the mathematics fixes and against the oracle's
closed form.  The table belongs to the CUDA path; the oracle (orc_bg.c) sums the closed form and knows nothing of it."""
import math
import os
import re

import numpy as np

import oracle

INC = os.path.join(os.path.dirname(__file__), "..", "paper_1407_2600_b200", "csrc", "cube_series.inc")


def _table():
    txt = open(INC).read()
    h = int(re.search(r"#define BG_SER_H (\d+)", txt).group(1))
    body = txt[txt.index("{") + 1: txt.rindex("}")]
    v = np.array([float(t) for t in body.replace("\n", " ").split(",") if t.strip()])
    assert v.size == (h + 1) ** 3
    return h, v.reshape(h + 1, h + 1, h + 1)


def test_table_closed_forms_symmetry_and_laplace():
    h, C = _table()
    assert h >= 11
    # the potential at the centre of the cube [-1,1]^3 and the uniform-sphere term
    assert abs(C[0, 0, 0] - 4.0 * (3.0 * math.log(2.0 + math.sqrt(3.0)) - math.pi / 2.0)) < 1e-14
    assert abs(C[1, 0, 0] + 2.0 * math.pi / 3.0) < 1e-15
    for i in range(h + 1):
        for j in range(h + 1):
            for k in range(h + 1):
                if i + j + k > h:
                    assert C[i, j, k] == 0.0
                else:
                    assert C[i, j, k] == C[j, i, k] == C[k, j, i] == C[i, k, j]
    # lap Phi = -4 pi: sum over the axes of (2i+2)(2i+1) C_(i+1,j,k) = -4 pi at (0,0,0), 0 elsewhere
    for i in range(h):
        for j in range(h - i):
            for k in range(h - i - j):
                lap = ((2 * i + 2) * (2 * i + 1) * C[i + 1, j, k] + (2 * j + 2) * (2 * j + 1) * C[i, j + 1, k]
                       + (2 * k + 2) * (2 * k + 1) * C[i, j, k + 1])
                want = -4.0 * math.pi if (i, j, k) == (0, 0, 0) else 0.0
                scale = max(abs((2 * i + 2) * (2 * i + 1) * C[i + 1, j, k]), 1e-3)
                assert abs(lap - want) < 1e-12 * max(scale, 1.0) + 1e-13, (i, j, k, lap)


def _series(C, hh, u):
    a, b, c = u[0] ** 2, u[1] ** 2, u[2] ** 2
    phi, g = 0.0, np.zeros(3)
    for i in range(hh + 1):
        for j in range(hh + 1 - i):
            for k in range(hh + 1 - i - j):
                t = C[i, j, k]
                phi += t * a ** i * b ** j * c ** k
                if i:
                    g[0] += t * 2 * i * u[0] ** (2 * i - 1) * b ** j * c ** k
                if j:
                    g[1] += t * 2 * j * a ** i * u[1] ** (2 * j - 1) * c ** k
                if k:
                    g[2] += t * 2 * k * a ** i * b ** j * u[2] ** (2 * k - 1)
    return phi, g


def test_series_equals_the_oracle_closed_form_where_the_kernel_uses_it():
    """order 14 for |u|_inf <= 0.21, order 22 for |u|_inf <= 0.36 (k_bg_window), on a cube of another size and place"""
    h, C = _table()
    rng = np.random.default_rng(4)
    ctr, half = np.array([0.3, -1.2, 2.5]), 0.37
    lo, hi = ctr - half, ctr + half
    for order, lim in ((7, 0.21), (h, 0.36)):
        pts = list((rng.random((40, 3)) * 2 - 1) * lim) + [np.array([lim, lim, lim]), np.array([lim, -lim, 0.0]), np.zeros(3)]
        for u in pts:
            I, g = oracle.cuboid_field(lo, hi, ctr + half * u)
            phi, gu = _series(C, order, u)
            assert abs(half * half * phi - I) < 2e-12 * I
            assert np.max(np.abs(half * gu - g)) < 1e-11 * half * 4.0 * math.pi / 3.0 + 1e-13
