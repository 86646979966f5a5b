/* orc_soft.c — ORACLE (test infrastructure): the pair softening law.
 * Kind 0, Plummer (BASELINE.json; reading A8): phi = -m (r^2 + eps^2)^(-1/2).
 * Kind 1, Dehnen's K1 compensating kernel ("using a Dehnen K1 compensating smoothing kernel (Dehnen 2001) for
 * small-scale force softening"; reading O6b of DESIGN.md).  Dehnen (2001) is not available; the kernel is rebuilt from the properties
 * that define the family K_n: the point mass is replaced by a density of COMPACT support h,
 *     rho(r) = C (1 - u)^n (A - B u),  u = (r/h)^2 < 1,   n = 1,
 * with unit mass and VANISHING SECOND MOMENT int rho r^2 d^3r = 0 (the "compensation": the leading, O(h^2) force bias of softening
 * cancels; the density is negative in the outer part).  Two conditions, two constants:
 *     int_0^1 x^4 (1-x^2)(A - B x^2) dx = 0   =>  A (2/35) = B (2/63)  =>  A : B = 5 : 9
 *     4 pi C int_0^1 x^2 (1-x^2)(5 - 9 x^2) dx = 4 pi C (16/105) = 1  =>  C = 105 / (64 pi)
 * so rho = 105/(64 pi h^3) (1 - u)(5 - 9 u), enclosed mass M(x) = (105/16)(5 x^3/3 - 14 x^5/5 + 9 x^7/7), and for r < h
 *     acc = -m d / h^3 (175/16 - 147/8 u + 135/16 u^2),      (= -m d / r^3 at u = 1 and beyond: exactly Newtonian outside h)
 *     phi = -(m/h) [ 1 + ( c0 (1-u) + c1 (1-u^2)/2 + c2 (1-u^3)/3 ) / 2 ],  c = (175/16, -147/8, 135/16);  phi(0) = -(105/32) m/h.
 * The tests pin exactly these properties (unit mass, zero second moment, Newtonian outside, continuity of force, its derivative and
 * the potential at h), so a wrong coefficient cannot pass.
 * Returned: f and phi with  acc = -m d f,  pot = -m phi  for separation d, r2 = |d|^2, softening length len (eps or h).
 */
#include "orc.h"
#include <math.h>

static int g_soft_kind = 0;
void orc_set_softening(int kind) { g_soft_kind = kind; }
int orc_get_softening(void) { return g_soft_kind; }

void orc_soft_pair(double r2, double len, double *f, double *phi)
{
    if (g_soft_kind == 0) {
        double R2 = r2 + len * len, ri = 1.0 / sqrt(R2);
        *f = ri / R2; *phi = ri;
        return;
    }
    const double c0 = 175.0 / 16.0, c1 = -147.0 / 8.0, c2 = 135.0 / 16.0;
    double u = r2 / (len * len);
    if (u >= 1.0) {
        double ri = 1.0 / sqrt(r2);
        *f = ri / r2; *phi = ri;
    } else {
        *f = (c0 + u * (c1 + c2 * u)) / (len * len * len);
        *phi = (1.0 + 0.5 * (c0 * (1.0 - u) + 0.5 * c1 * (1.0 - u * u) + c2 * (1.0 - u * u * u) / 3.0)) / len;
    }
}
