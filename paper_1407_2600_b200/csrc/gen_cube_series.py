"""Writes cube_series.inc: Taylor coefficients about the centre of the Newtonian potential of the homogeneous unit-density cube
[-1, 1]^3,   Phi(u) = int d^3y / |y - u| = sum_{i,j,k} C_ijk u1^(2i) u2^(2j) u3^(2k),   used by background.cu for the window's
background (reading O4b of DESIGN.md) where the sinks sit well inside the window.  Run by hand when the order changes:

    python paper_1407_2600_b200/csrc/gen_cube_series.py

The .inc is committed, so the build needs neither this script nor mpmath.  Nothing here is shared with oracle/ (which sums
the closed form, orc_bg.c); the script checks its own series against its own closed form before writing.

Derivation.  With f = 1/|y| and T_n = d^n Phi / du^n at 0 (n even in every component, by symmetry):
  * one derivative per axis turns the volume integral into corner values, d^3 Phi/du1 du2 du3 (u) = - sum_corners sigma f(corner - u)
    (sigma = +1 for an even number of lower corners); the remaining derivatives act on f, and D^m f for m = n - (1,1,1), odd in
    every coordinate, takes the value sigma D^m f(1,1,1) at the corners:      T_n = 8 D^(n-(1,1,1)) f (1,1,1)          (n1, n2, n3 >= 2)
  * with n3 = 0 one integral is left:                                          T_n = 4 int_-1^1 D^(n1-1,n2-1,0) f (1,1,z) dz   (n1, n2 >= 2)
  * Laplace: d^m (lap Phi) = 0 for |m| >= 1, lap Phi = -4 pi, hence           T_(l,0,0) = -2 T_(l-2,2,0),  T_(2,0,0) = -4 pi / 3.
  * D^m (1/r) = P_m / r^(2|m|+1),  P_0 = 1,  P_(m+e_x) = r^2 dP_m/dx - (2|m|+1) x P_m   (integer polynomials, exact).
"""
import os
from functools import lru_cache

import mpmath as mp

mp.mp.dps = 50
LMAX = 22                      # highest total degree kept (window half-width k = 1 needs it; k >= 2 uses 14)
HERE = os.path.dirname(os.path.abspath(__file__))


def padd(a, b, s=1):
    r = dict(a)
    for k, v in b.items():
        r[k] = r.get(k, 0) + s * v
        if r[k] == 0:
            del r[k]
    return r


def pmul_mono(a, e, c):
    return {(k[0] + e[0], k[1] + e[1], k[2] + e[2]): v * c for k, v in a.items()}


def pdiff(a, ax):
    r = {}
    for k, v in a.items():
        if k[ax]:
            kk = list(k); kk[ax] -= 1
            r[tuple(kk)] = r.get(tuple(kk), 0) + v * k[ax]
    return r


@lru_cache(maxsize=None)
def P(m):
    """numerator polynomial of D^m (1/r) (dict exponent triple -> int)"""
    if m == (0, 0, 0):
        return {(0, 0, 0): 1}
    ax = max(range(3), key=lambda i: m[i])
    mm = list(m); mm[ax] -= 1; mm = tuple(mm)
    k = sum(mm)
    p = P(mm)
    dp = pdiff(p, ax)
    r = {}
    for e in ((2, 0, 0), (0, 2, 0), (0, 0, 2)):
        r = padd(r, pmul_mono(dp, e, 1))
    ex = [0, 0, 0]; ex[ax] = 1
    return padd(r, pmul_mono(p, tuple(ex), 2 * k + 1), -1)


def Df(m, x, y, z):
    p = P(m)
    val = mp.mpf(0)
    for (a, b, c), v in p.items():
        val += v * mp.mpf(x) ** a * mp.mpf(y) ** b * mp.mpf(z) ** c
    r2 = mp.mpf(x) ** 2 + mp.mpf(y) ** 2 + mp.mpf(z) ** 2
    return val / r2 ** (mp.mpf(2 * sum(m) + 1) / 2)


@lru_cache(maxsize=None)
def T(n):
    n = tuple(sorted(n, reverse=True))
    if n == (0, 0, 0):
        return phi_closed(0, 0, 0)
    if n == (2, 0, 0):
        return -4 * mp.pi / 3
    if n[1] == 0:
        return -2 * T((n[0] - 2, 2, 0))
    if n[2] == 0:
        m = (n[0] - 1, n[1] - 1, 0)
        return 4 * mp.quad(lambda z: Df(m, 1, 1, z), [-1, 0, 1])
    return 8 * Df((n[0] - 1, n[1] - 1, n[2] - 1), 1, 1, 1)


def phi_closed(x, y, z):
    """closed form (MacMillan 1930), for the self-check only"""
    tot = mp.mpf(0)
    for i in (0, 1):
        for j in (0, 1):
            for k in (0, 1):
                X, Y, Z = (1 if i else -1) - mp.mpf(x), (1 if j else -1) - mp.mpf(y), (1 if k else -1) - mp.mpf(z)
                r = mp.sqrt(X * X + Y * Y + Z * Z)
                F = (X * Y * mp.log(Z + r) + Y * Z * mp.log(X + r) + Z * X * mp.log(Y + r)
                     - X * X / 2 * mp.atan(Y * Z / (X * r)) - Y * Y / 2 * mp.atan(Z * X / (Y * r)) - Z * Z / 2 * mp.atan(X * Y / (Z * r)))
                tot += (-1 if (i + j + k) % 2 else 1) * -F
    return tot


def coefficients(lmax):
    h = lmax // 2
    C = {}
    for i in range(h + 1):
        for j in range(h + 1 - i):
            for k in range(h + 1 - i - j):
                C[(i, j, k)] = T((2 * i, 2 * j, 2 * k)) / (mp.factorial(2 * i) * mp.factorial(2 * j) * mp.factorial(2 * k))
    return C


def series(C, x, y, z, lmax):
    return sum(v * mp.mpf(x) ** (2 * i) * mp.mpf(y) ** (2 * j) * mp.mpf(z) ** (2 * k) for (i, j, k), v in C.items() if 2 * (i + j + k) <= lmax)


def main():
    C = coefficients(LMAX)
    # self-check: the series against the closed form where background.cu uses it (|u|_inf <= 0.36 with LMAX, <= 0.21 with 14)
    worst = {14: 0, LMAX: 0}
    pts = [(0.0, 0.0, 0.0), (0.2, 0.1, 0.05), (0.21, 0.21, 0.21), (-0.21, 0.2, -0.13), (0.36, 0.36, 0.36), (0.36, -0.3, 0.1), (0.0, 0.36, 0.0)]
    for p in pts:
        ref = phi_closed(*[v + mp.mpf(10) ** -30 for v in p])          # off the planes where a prefactor vanishes
        for L in (14, LMAX):
            if L == 14 and max(abs(v) for v in p) > 0.21:
                continue
            worst[L] = max(worst[L], abs(series(C, *p, L) - ref))
    print("max |series - closed form|: order 14 on |u| <= 0.21:", mp.nstr(worst[14], 3), " order", LMAX, "on |u| <= 0.36:", mp.nstr(worst[LMAX], 3))
    assert worst[14] < 1e-9 and worst[LMAX] < 1e-9
    h = LMAX // 2
    with open(os.path.join(HERE, "cube_series.inc"), "w") as f:
        f.write("// written by gen_cube_series.py: C_ijk of Phi(u) = sum C_ijk u1^(2i) u2^(2j) u3^(2k), the potential int d^3y/|y - u| of the\n")
        f.write("// unit-density cube [-1,1]^3 about its centre; i + j + k <= %d, index ((i * %d) + j) * %d + k; 0 where i + j + k > %d.\n" % (h, h + 1, h + 1, h))
        f.write("#define BG_SER_H %d\n" % h)
        f.write("static const double bg_series_host[%d] = {\n" % ((h + 1) ** 3))
        for i in range(h + 1):
            for j in range(h + 1):
                f.write("    " + ", ".join(mp.nstr(C.get((i, j, k), mp.mpf(0)), 20, strip_zeros=False, min_fixed=0, max_fixed=0) for k in range(h + 1)) + ",\n")
        f.write("};\n")


if __name__ == "__main__":
    main()
