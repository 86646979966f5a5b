/* orc_bg.c — ORACLE (test infrastructure): the pieces of background subtraction, reading O4b of DESIGN.md.
 * PAPER.md:63 "Accuracy and error behavior have been improved significantly for cosmological volumes through the use
 * of a technique to subtract the uniform background density (Warren 2013)".  Warren (2013) is not available; what is
 * implemented is the reading stated in DESIGN.md: in a periodic box the sources are delta rho = particles - rho_bar, and
 *   - cells of level <= l_b that are accepted outside the group's window carry the moments of delta rho over their cube
 *     (orc_cube_moments: closed-form moments of the homogeneous cube about the cell's expansion centre);
 *   - the background of everything else inside the image block is summed exactly: the window, one homogeneous cuboid
 *     around the sink group, plus the few coarse cubes that stick out of it (orc_cuboid_field: the closed-form Newtonian
 *     potential and field of a homogeneous cuboid).
 * Plain fp64, shares nothing with the CUDA path.  G = 1.
 */
#include "orc.h"
#include <math.h>

/* Antiderivatives.  With r = sqrt(X^2 + Y^2 + Z^2):
 *   d^3/dXdYdZ F = 1/r,   F = XY ln(Z+r) + YZ ln(X+r) + ZX ln(Y+r) - X^2/2 atan(YZ/(X r)) - Y^2/2 atan(ZX/(Y r)) - Z^2/2 atan(XY/(Z r))
 *   d^2/dYdZ  G = 1/r,   G(X; Y, Z) = Y ln(Z+r) + Z ln(Y+r) - X atan(YZ/(X r))
 * (MacMillan 1930; Waldvogel 1976).  Terms whose prefactor vanishes are dropped (their limit is 0), and ln(Z + r) for
 * Z < 0 is taken as ln((X^2 + Y^2)/(r - Z)) so that it does not cancel. */
static double log_zr(double z, double r, double rho2)
{
    /* ln(z + r), r = sqrt(rho2 + z^2); only called with rho2 > 0 */
    return z >= 0.0 ? log(z + r) : log(rho2 / (r - z));
}

static double corner_F(double X, double Y, double Z)
{
    double r = sqrt(X * X + Y * Y + Z * Z), f = 0.0;
    if (X != 0.0 && Y != 0.0) f += X * Y * log_zr(Z, r, X * X + Y * Y);
    if (Y != 0.0 && Z != 0.0) f += Y * Z * log_zr(X, r, Y * Y + Z * Z);
    if (Z != 0.0 && X != 0.0) f += Z * X * log_zr(Y, r, Z * Z + X * X);
    if (X != 0.0) f -= 0.5 * X * X * atan(Y * Z / (X * r));
    if (Y != 0.0) f -= 0.5 * Y * Y * atan(Z * X / (Y * r));
    if (Z != 0.0) f -= 0.5 * Z * Z * atan(X * Y / (Z * r));
    return f;
}

static double corner_G(double X, double Y, double Z)
{
    double r = sqrt(X * X + Y * Y + Z * Z), g = 0.0;
    if (Y != 0.0) g += Y * log_zr(Z, r, X * X + Y * Y);
    if (Z != 0.0) g += Z * log_zr(Y, r, X * X + Z * Z);
    if (X != 0.0) g -= X * atan(Y * Z / (X * r));
    return g;
}

/* Homogeneous cuboid [lo, hi] of unit density seen from x:
 *   *I = int d^3y / |y - x|                (its potential is -rho I)
 *   g  = int (y - x)/|y - x|^3 d^3y        (the attractive field of unit positive density; = grad_x I)
 * from the eight corners, (X, Y, Z) = corner - x, sign + for an even number of lower corners.
 * Valid inside, outside and on the surface. */
void orc_cuboid_field(const double lo[3], const double hi[3], const double x[3], double *I, double g[3])
{
    double sI = 0.0, sg[3] = {0, 0, 0};
    for (int i = 0; i < 2; i++)
        for (int j = 0; j < 2; j++)
            for (int k = 0; k < 2; k++) {
                double X = (i ? hi[0] : lo[0]) - x[0], Y = (j ? hi[1] : lo[1]) - x[1], Z = (k ? hi[2] : lo[2]) - x[2];
                double sg3 = ((i + j + k) & 1) ? 1.0 : -1.0;          /* product of (+ upper limit, - lower limit) */
                sI += sg3 * corner_F(X, Y, Z);
                /* g_x = int (Y-range)(Z-range) [ -1/r ] from X_lo to X_hi  = - sum sign G(X; Y, Z) */
                sg[0] -= sg3 * corner_G(X, Y, Z);
                sg[1] -= sg3 * corner_G(Y, Z, X);
                sg[2] -= sg3 * corner_G(Z, X, Y);
            }
    if (I) *I = sI;
    if (g) { g[0] = sg[0]; g[1] = sg[1]; g[2] = sg[2]; }
}

/* Moments of the homogeneous unit-density cube of side s centred at ctr about the point z:
 *   C_n = int_cube (y - z)^n d^3y = prod_i [ (s/2 - o_i)^(n_i+1) - (-s/2 - o_i)^(n_i+1) ] / (n_i + 1),   o = z - ctr,
 * for every multi-index |n| <= p in the interface order. */
void orc_cube_moments(double s, const double ctr[3], const double z[3], int p, double *C)
{
    double one[3][ORC_PMAX + 1];
    for (int d = 0; d < 3; d++) {
        double o = z[d] - ctr[d], a = 0.5 * s - o, b = -0.5 * s - o, pa = a, pb = b;
        for (int e = 0; e <= p; e++) {
            one[d][e] = (pa - pb) / (e + 1);
            pa *= a; pb *= b;
        }
    }
    for (int l = 0; l <= p; l++)
        for (int a = l; a >= 0; a--)
            for (int b = l - a; b >= 0; b--) {
                int c = l - a - b;
                C[orc_midx(a, b, c)] = one[0][a] * one[1][b] * one[2][c];
            }
}

/* background level l_b for N particles: the level at which a uniform box holds ~64..512 particles per cell,
 * l_b = max(2, floor((floor(log2 N) - 6) / 3)); and the window half-width in level-l_b cells for opening angle theta,
 * k = min(ceil(1/theta), ws 2^l_b) (the window must stay inside the image block).  A level-l_b cell just outside the
 * window is accepted unless its centre of mass sits within s/theta + delta of the group, i.e. off-centre towards it: rare,
 * and then its cube is one of those summed by itself.  (ceil(1/theta) + 1 would exclude that case, but it opens every
 * coarser cell that touches the larger window: 10 - 60 % longer lists at theta 0.5 - 1 against 0 - 10 %, measured.) */
int orc_bg_level(int64_t n)
{
    int lg = 0;
    while ((n >> (lg + 1)) > 0) lg++;
    int l = (lg - 6) / 3;
    if (lg < 6) l = 0;
    return l < 2 ? 2 : l;
}
int orc_bg_halfwidth(double theta, int ws, int lb)
{
    int k = (int)ceil(1.0 / theta), kmax = ws << lb;
    return k < kmax ? k : kmax;
}
