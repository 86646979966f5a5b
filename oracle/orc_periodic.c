/* orc_periodic.c — ORACLE (test infrastructure): periodic direct summation D-per (Ewald) and the
 * order-8 far-field local expansion of SURVEY.md §8(c) O7.
 * PAPER.md:63 "periodic boundary conditions using a high-order (p=8) multipole local expansion
 * (Challacombe et al. 1997; Metchnik 2009)"; BASELINE.json configs[2] "nearest replicas plus Ewald
 * correction" (reading A11: the (2 WS+1)^3 nearest images are summed explicitly, everything else —
 * the remaining images and the neutralising background — is the smooth field Phi_far).
 * Shares nothing with the CUDA path.  G = 1, unit point mass unless stated.
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846
#define SQRTPI 1.77245385090551602730

static void ewald_cutoffs(double L, double alpha, int *nmax, int *hmax, double *rcut, double *h2cut)
{
    double rc = 6.2 / alpha;                       /* erfc(6.2) ~ 2e-18                          */
    double h2 = 41.0 * alpha * alpha * L * L / (PI * PI);   /* exp(-41) ~ 1.6e-18                 */
    if (rcut) *rcut = rc;
    if (h2cut) *h2cut = h2;
    if (nmax && *nmax < 0) *nmax = (int)ceil(rc / L) + 1;
    if (hmax && *hmax < 0) *hmax = (int)ceil(sqrt(h2));
}

/* Ewald sums for the fully periodic unit point mass with neutralising background (D-per):
 *  psi(x) = pi/(alpha^2 L^3) - sum_n erfc(alpha r_n)/r_n
 *           - 1/(pi L) sum_{h!=0} |h|^-2 exp(-pi^2 |h|^2/(alpha^2 L^2)) cos(2 pi h.x/L)
 *  a(x)   = - sum_n (x-nL) r_n^-3 [erfc(alpha r_n) + (2 alpha r_n/sqrt(pi)) exp(-alpha^2 r_n^2)]
 *           - (2/L^2) sum_{h!=0} (h/|h|^2) exp(-pi^2 |h|^2/(alpha^2 L^2)) sin(2 pi h.x/L)
 * r_n = |x - nL|, |n|_inf <= nmax, |h|_inf <= hmax (pass < 0 for automatic ~1e-17 cutoffs). */
void orc_ewald_pair(const double x[3], double L, double alpha, int nmax, int hmax, double *psi,
                    double a[3])
{
    ewald_cutoffs(L, alpha, &nmax, &hmax, NULL, NULL);
    double ps = PI / (alpha * alpha * L * L * L), ax = 0, ay = 0, az = 0;
    for (int i = -nmax; i <= nmax; i++)
        for (int j = -nmax; j <= nmax; j++)
            for (int k = -nmax; k <= nmax; k++) {
                double dx = x[0] - i * L, dy = x[1] - j * L, dz = x[2] - k * L;
                double r = sqrt(dx * dx + dy * dy + dz * dz);
                double ec = erfc(alpha * r);
                double f = (ec + 2.0 * alpha * r / SQRTPI * exp(-alpha * alpha * r * r)) / (r * r * r);
                ps -= ec / r;
                ax -= dx * f; ay -= dy * f; az -= dz * f;
            }
    for (int i = -hmax; i <= hmax; i++)
        for (int j = -hmax; j <= hmax; j++)
            for (int k = -hmax; k <= hmax; k++) {
                int h2 = i * i + j * j + k * k;
                if (h2 == 0) continue;
                double c = exp(-PI * PI * h2 / (alpha * alpha * L * L)) / h2;
                double ph = 2.0 * PI * (i * x[0] + j * x[1] + k * x[2]) / L;
                ps -= c * cos(ph) / (PI * L);
                double s = 2.0 / (L * L) * c * sin(ph);
                ax -= i * s; ay -= j * s; az -= k * s;
            }
    if (psi) *psi = ps;
    if (a) { a[0] = ax; a[1] = ay; a[2] = az; }
}

/* lim_{x->0} [psi(x) + 1/|x|]: the n = 0 real-space term -erfc(alpha r)/r + 1/r = erf(alpha r)/r
 * tends to 2 alpha/sqrt(pi); everything else is evaluated at x = 0. */
double orc_ewald_self(double L, double alpha, int nmax, int hmax)
{
    ewald_cutoffs(L, alpha, &nmax, &hmax, NULL, NULL);
    double ps = PI / (alpha * alpha * L * L * L) + 2.0 * alpha / SQRTPI;
    for (int i = -nmax; i <= nmax; i++)
        for (int j = -nmax; j <= nmax; j++)
            for (int k = -nmax; k <= nmax; k++) {
                if (!i && !j && !k) continue;
                double r = L * sqrt((double)(i * i + j * j + k * k));
                ps -= erfc(alpha * r) / r;
            }
    for (int i = -hmax; i <= hmax; i++)
        for (int j = -hmax; j <= hmax; j++)
            for (int k = -hmax; k <= hmax; k++) {
                int h2 = i * i + j * j + k * k;
                if (h2 == 0) continue;
                ps -= exp(-PI * PI * h2 / (alpha * alpha * L * L)) / h2 / (PI * L);
            }
    return ps;
}

/* Plummer minus Newton pair terms of the explicit image block, for displacement d (sink - source):
 * adds a_Pl(d) - a_N(d) and phi_Pl(d) - phi_N(d).  d = 0 (coincident distinct particles, or a
 * particle and itself) has no Newtonian term to remove here; the caller handles it. */
static void plummer_minus_newton(const double d[3], double e2, double a[3], double *ph)
{
    /* softened minus Newtonian pair term; the softening law is orc_soft_pair's (Plummer unless the K1 kernel is selected) */
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double r = sqrt(r2), fs, phis;
    orc_soft_pair(r2, sqrt(e2), &fs, &phis);
    double fn = 1.0 / (r * r * r);
    for (int k = 0; k < 3; k++) a[k] += -d[k] * fs + d[k] * fn;
    *ph += -phis + 1.0 / r;
}

/* D-per, pair by pair exactly as SURVEY.md §8(c) writes it:
 *  acc_i = sum_j m_j [ a_Ew(d_ij) + sum_{n in block} ( a_Pl(d_ij + nL) - a_N(d_ij + nL) ) ]
 * with the n = 0 term skipped for j = i (its Ewald part is replaced by the regular limit). */
void orc_direct_per_pairwise(int64_t n, const float *pos, const float *mass, double L, double eps,
                             int ws, double alpha, int64_t nsink, const int64_t *sink, double *acc,
                             double *pot)
{
    double e2 = eps * eps, self = orc_ewald_self(L, alpha, -1, -1);
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        double A[3] = {0, 0, 0}, P = 0;
        for (int64_t j = 0; j < n; j++) {
            double d[3], m = (double)mass[j], a[3] = {0, 0, 0}, ph = 0;
            for (int k = 0; k < 3; k++) d[k] = (double)pos[3 * i + k] - (double)pos[3 * j + k];
            int zero = (d[0] == 0.0 && d[1] == 0.0 && d[2] == 0.0);
            if (!zero) {
                orc_ewald_pair(d, L, alpha, -1, -1, &ph, a);
            } else {
                /* regular part of psi at 0; the force's regular part vanishes by symmetry.  For a
                 * coincident *distinct* pair the Plummer term at d = 0 is kept: -1/eps, no force */
                ph = self;
                if (j != i) { double f0, p0; orc_soft_pair(0.0, eps, &f0, &p0); ph += -p0; }
            }
            for (int ix = -ws; ix <= ws; ix++)
                for (int iy = -ws; iy <= ws; iy++)
                    for (int iz = -ws; iz <= ws; iz++) {
                        if (zero && !ix && !iy && !iz) continue;
                        double dn[3] = { d[0] + ix * L, d[1] + iy * L, d[2] + iz * L };
                        plummer_minus_newton(dn, e2, a, &ph);
                    }
            for (int k = 0; k < 3; k++) A[k] += m * a[k];
            P += m * ph;
        }
        for (int k = 0; k < 3; k++) acc[3 * s + k] = A[k];
        if (pot) pot[s] = P;
    }
}

/* D-per for many sources: the same sums with the reciprocal-space part of a_Ew/psi accumulated
 * through the structure factors C_h = sum_j m_j cos(2 pi h.x_j/L), S_h = sum_j m_j sin(...)
 * (sin(t_i - t_j) = sin t_i cos t_j - cos t_i sin t_j), and the real-space part cut at
 * erfc(alpha r) < 1e-17.  A test pins it to orc_direct_per_pairwise. */
void orc_direct_per(int64_t n, const float *pos, const float *mass, double L, double eps, int ws,
                    double alpha, int64_t nsink, const int64_t *sink, double *acc, double *pot)
{
    int nmax = -1, hmax = -1; double rcut, h2cut;
    ewald_cutoffs(L, alpha, &nmax, &hmax, &rcut, &h2cut);
    if (nmax < ws) nmax = ws;
    double e2 = eps * eps;
    /* reciprocal vectors */
    int nh = 0, cap = (2 * hmax + 1) * (2 * hmax + 1) * (2 * hmax + 1);
    int *hv = malloc(sizeof(int) * 3 * cap);
    double *ch = malloc(sizeof(double) * cap);
    for (int i = -hmax; i <= hmax; i++)
        for (int j = -hmax; j <= hmax; j++)
            for (int k = -hmax; k <= hmax; k++) {
                int h2 = i * i + j * j + k * k;
                if (h2 == 0 || h2 > h2cut) continue;
                hv[3 * nh] = i; hv[3 * nh + 1] = j; hv[3 * nh + 2] = k;
                ch[nh] = exp(-PI * PI * h2 / (alpha * alpha * L * L)) / h2;
                nh++;
            }
    double *Ch = calloc(nh, sizeof(double)), *Sh = calloc(nh, sizeof(double));
#pragma omp parallel
    {
        double *c = calloc(nh, sizeof(double)), *s = calloc(nh, sizeof(double));
#pragma omp for schedule(static)
        for (int64_t j = 0; j < n; j++) {
            double x = pos[3 * j], y = pos[3 * j + 1], z = pos[3 * j + 2], m = mass[j];
            for (int q = 0; q < nh; q++) {
                double t = 2.0 * PI * (hv[3 * q] * x + hv[3 * q + 1] * y + hv[3 * q + 2] * z) / L;
                c[q] += m * cos(t); s[q] += m * sin(t);
            }
        }
#pragma omp critical
        for (int q = 0; q < nh; q++) { Ch[q] += c[q]; Sh[q] += s[q]; }
        free(c); free(s);
    }
    double selfreal = 2.0 * alpha / SQRTPI;        /* lim of the n=0 real-space term + 1/r       */
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        double xi[3] = { pos[3 * i], pos[3 * i + 1], pos[3 * i + 2] };
        double A[3] = {0, 0, 0}, P = 0;
        /* reciprocal part + constant */
        for (int q = 0; q < nh; q++) {
            double t = 2.0 * PI * (hv[3 * q] * xi[0] + hv[3 * q + 1] * xi[1] + hv[3 * q + 2] * xi[2]) / L;
            double st = sin(t), ct = cos(t);
            double f = 2.0 / (L * L) * ch[q] * (st * Ch[q] - ct * Sh[q]);
            A[0] -= hv[3 * q] * f; A[1] -= hv[3 * q + 1] * f; A[2] -= hv[3 * q + 2] * f;
            P -= ch[q] * (ct * Ch[q] + st * Sh[q]) / (PI * L);
        }
        double mtot_term = PI / (alpha * alpha * L * L * L);
        /* real-space part + image block */
        for (int64_t j = 0; j < n; j++) {
            double d[3], m = (double)mass[j], a[3] = {0, 0, 0}, ph = mtot_term;
            for (int k = 0; k < 3; k++) d[k] = xi[k] - (double)pos[3 * j + k];
            int zero = (d[0] == 0.0 && d[1] == 0.0 && d[2] == 0.0);
            /* only the images that can contribute are visited: the real-space term needs |d - nL| < rcut, so per axis
             * n lies in [(d - rcut)/L, (d + rcut)/L]; the range is widened to hold the whole image block */
            int lo[3], hi[3];
            for (int k = 0; k < 3; k++) {
                lo[k] = (int)ceil((d[k] - rcut) / L); hi[k] = (int)floor((d[k] + rcut) / L);
                if (lo[k] > -ws) lo[k] = -ws;
                if (hi[k] < ws) hi[k] = ws;
                if (lo[k] < -nmax) lo[k] = -nmax;
                if (hi[k] > nmax) hi[k] = nmax;
            }
            for (int ix = lo[0]; ix <= hi[0]; ix++)
                for (int iy = lo[1]; iy <= hi[1]; iy++)
                    for (int iz = lo[2]; iz <= hi[2]; iz++) {
                        double dn[3] = { d[0] - ix * L, d[1] - iy * L, d[2] - iz * L };
                        int inblock = (abs(ix) <= ws && abs(iy) <= ws && abs(iz) <= ws);
                        if (zero && !ix && !iy && !iz) {
                            ph += selfreal;
                            if (j != i) { double f0, p0; orc_soft_pair(0.0, eps, &f0, &p0); ph += -p0; }
                            continue;
                        }
                        double r2 = dn[0] * dn[0] + dn[1] * dn[1] + dn[2] * dn[2];
                        if (r2 < rcut * rcut) {
                            double r = sqrt(r2), ec = erfc(alpha * r);
                            double f = (ec + 2.0 * alpha * r / SQRTPI * exp(-alpha * alpha * r2)) / (r2 * r);
                            ph -= ec / r;
                            for (int k = 0; k < 3; k++) a[k] -= dn[k] * f;
                        }
                        if (inblock) plummer_minus_newton(dn, e2, a, &ph);
                    }
            for (int k = 0; k < 3; k++) A[k] += m * a[k];
            P += m * ph;
        }
        for (int k = 0; k < 3; k++) acc[3 * s + k] = A[k];
        if (pot) pot[s] = P;
    }
    free(hv); free(ch); free(Ch); free(Sh);
}

/* ---- O7 far field --------------------------------------------------------------------------- */
/* Phi_far(u) = psi(u) + sum_{|n|_inf <= ws} 1/|u - nL| and a_far = -grad Phi_far, straight from
 * the definition (used to pin the Taylor coefficients below; |u| must be > 0). */
double orc_farfield_phi(const double u[3], double L, int ws, double a[3])
{
    double psi, ae[3];
    orc_ewald_pair(u, L, 2.0 / L, -1, -1, &psi, ae);
    for (int i = -ws; i <= ws; i++)
        for (int j = -ws; j <= ws; j++)
            for (int k = -ws; k <= ws; k++) {
                double d[3] = { u[0] - i * L, u[1] - j * L, u[2] - k * L };
                double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                psi += 1.0 / r;
                for (int q = 0; q < 3; q++) ae[q] += d[q] / (r * r * r);
            }
    if (a) for (int q = 0; q < 3; q++) a[q] = ae[q];
    return psi;
}

/* truncated polynomials in (u_x,u_y,u_z), coefficient of u^n stored at orc_midx(n) */
typedef struct { int order, np; int *ea, *eb, *ec; } ptab_t;

static void poly_mul(const ptab_t *pt, const double *A, const double *B, double *C)
{
    for (int i = 0; i < pt->np; i++) C[i] = 0.0;
    for (int i = 0; i < pt->np; i++) {
        if (A[i] == 0.0) continue;
        int li = pt->ea[i] + pt->eb[i] + pt->ec[i];
        for (int j = 0; j < pt->np; j++) {
            int lj = pt->ea[j] + pt->eb[j] + pt->ec[j];
            if (li + lj > pt->order) break;                 /* indices are rank-ascending      */
            C[orc_midx(pt->ea[i] + pt->ea[j], pt->eb[i] + pt->eb[j], pt->ec[i] + pt->ec[j])] += A[i] * B[j];
        }
    }
}

/* T_n, |n| <= order: Taylor coefficients at u = 0 of Phi_far(u), from the Ewald split:
 *   Phi_far = pi/(alpha^2 L^3) + sum_{|n|<=ws} erf(alpha r_n)/r_n - sum_{|n|>ws} erfc(alpha r_n)/r_n
 *             - 1/(pi L) sum_h |h|^-2 exp(-pi^2 h^2/(alpha L)^2) cos(2 pi h.u/L).
 * A radial term F(s), s = |u - a|^2 = s0 + delta(u), delta = -2 a.u + |u|^2, is composed as
 * sum_k F^(k)(s0)/k! delta^k with F^(k) = (-1/2)^k B_k, B_k = (-(1/r) d/dr)^k F:
 *   erfc(alpha r)/r : B_0 = erfc(alpha r)/r, B_k = [(2k-1) B_{k-1} + (2 alpha^2)^k e^{-alpha^2 r^2}/(alpha sqrt(pi))]/r^2
 *   1/r             : A_k = (2k-1)!!/r^(2k+1)          (erf/r = 1/r - erfc/r)
 * and the n = 0 term erf(alpha r)/r = (2 alpha/sqrt(pi)) sum_k (-alpha^2 r^2)^k / (k! (2k+1)). */
void orc_farfield_T(double L, int ws, int order, double *T)
{
    double alpha = 2.0 / L;
    int np = ORC_NP(order);
    int ea[ORC_NP(ORC_PMAX)], eb[ORC_NP(ORC_PMAX)], ec[ORC_NP(ORC_PMAX)];
    orc_mtable(order, ea, eb, ec);
    ptab_t pt = { order, np, ea, eb, ec };
    double *delta = malloc(sizeof(double) * np), *pw = malloc(sizeof(double) * np),
           *tmp = malloc(sizeof(double) * np);
    for (int i = 0; i < np; i++) T[i] = 0.0;
    T[0] = PI / (alpha * alpha * L * L * L);
    /* n = 0 image: even series in r^2 = ux^2 + uy^2 + uz^2 */
    {
        for (int i = 0; i < np; i++) { delta[i] = 0.0; pw[i] = 0.0; }
        if (order >= 2) { delta[orc_midx(2, 0, 0)] = 1.0; delta[orc_midx(0, 2, 0)] = 1.0; delta[orc_midx(0, 0, 2)] = 1.0; }
        pw[0] = 1.0;                                          /* (r^2)^0                         */
        double fact = 1.0, a2k = 1.0;
        for (int k = 0; 2 * k <= order; k++) {
            if (k > 0) { poly_mul(&pt, pw, delta, tmp); memcpy(pw, tmp, sizeof(double) * np); fact *= k; a2k *= -alpha * alpha; }
            double c = 2.0 * alpha / SQRTPI * a2k / (fact * (2 * k + 1));
            for (int i = 0; i < np; i++) T[i] += c * pw[i];
        }
    }
    /* n != 0 images */
    int nmax = -1, hmax = -1; double rcut, h2cut;
    ewald_cutoffs(L, alpha, &nmax, &hmax, &rcut, &h2cut);
    nmax += 1;
    if (nmax < ws) nmax = ws;
    for (int ix = -nmax; ix <= nmax; ix++)
        for (int iy = -nmax; iy <= nmax; iy++)
            for (int iz = -nmax; iz <= nmax; iz++) {
                if (!ix && !iy && !iz) continue;
                int inblock = (abs(ix) <= ws && abs(iy) <= ws && abs(iz) <= ws);
                double a[3] = { ix * L, iy * L, iz * L };
                double s0 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2], r = sqrt(s0);
                if (!inblock && r > rcut + L) continue;
                /* delta(u) = -2 a.u + |u|^2 */
                for (int i = 0; i < np; i++) delta[i] = 0.0;
                if (order >= 1) { delta[orc_midx(1, 0, 0)] = -2 * a[0]; delta[orc_midx(0, 1, 0)] = -2 * a[1]; delta[orc_midx(0, 0, 1)] = -2 * a[2]; }
                if (order >= 2) { delta[orc_midx(2, 0, 0)] = 1.0; delta[orc_midx(0, 2, 0)] = 1.0; delta[orc_midx(0, 0, 2)] = 1.0; }
                for (int i = 0; i < np; i++) pw[i] = 0.0;
                pw[0] = 1.0;
                double Bk = erfc(alpha * r) / r, Ak = 1.0 / r, ex = exp(-alpha * alpha * s0) / (alpha * SQRTPI);
                double half = 1.0, kfact = 1.0, a2 = 1.0;
                for (int k = 0; k <= order; k++) {
                    if (k > 0) {
                        poly_mul(&pt, pw, delta, tmp); memcpy(pw, tmp, sizeof(double) * np);
                        a2 *= 2.0 * alpha * alpha;
                        Bk = ((2 * k - 1) * Bk + a2 * ex) / s0;
                        Ak = (2 * k - 1) * Ak / s0;
                        half *= -0.5; kfact *= k;
                    }
                    /* in-block: + erf/r = +(A_k - B_k);  outside: - erfc/r = -B_k */
                    double Fk = (inblock ? (Ak - Bk) : -Bk) * half / kfact;
                    for (int i = 0; i < np; i++) T[i] += Fk * pw[i];
                }
            }
    /* reciprocal part: cos(w.u) = sum_m (-1)^m (w.u)^(2m)/(2m)!, (w.u)^q = sum_{|n|=q} q!/n! w^n u^n */
    double fac[ORC_PMAX + 1]; fac[0] = 1.0;
    for (int i = 1; i <= ORC_PMAX; i++) fac[i] = fac[i - 1] * i;
    for (int i = -hmax; i <= hmax; i++)
        for (int j = -hmax; j <= hmax; j++)
            for (int k = -hmax; k <= hmax; k++) {
                int h2 = i * i + j * j + k * k;
                if (h2 == 0 || h2 > h2cut) continue;
                double c = -exp(-PI * PI * h2 / (alpha * alpha * L * L)) / h2 / (PI * L);
                double w[3] = { 2 * PI * i / L, 2 * PI * j / L, 2 * PI * k / L };
                for (int q = 0; q < np; q++) {
                    int l = ea[q] + eb[q] + ec[q];
                    if (l & 1) continue;
                    double sg = ((l / 2) & 1) ? -1.0 : 1.0;
                    T[q] += c * sg * pow(w[0], ea[q]) * pow(w[1], eb[q]) * pow(w[2], ec[q]) /
                            (fac[ea[q]] * fac[eb[q]] * fac[ec[q]]);
                }
            }
    free(delta); free(pw); free(tmp);
}

/* Lambda_n = sum_{|k| <= order-|n|} (-1)^|k| C(n+k,k) M_k^c T_{n+k},
 * M_k^c = sum_j m_j (s_j - c)^k about the box centre c = (L/2,L/2,L/2)   (O7 steps 2-3) */
void orc_farfield_local(int64_t n, const float *pos, const float *mass, double L, int ws, int order,
                        int bg, double *Lambda)
{
    int np = ORC_NP(order);
    int ea[ORC_NP(ORC_PMAX)], eb[ORC_NP(ORC_PMAX)], ec[ORC_NP(ORC_PMAX)];
    orc_mtable(order, ea, eb, ec);
    double *T = malloc(sizeof(double) * np), *M = calloc(np, sizeof(double));
    orc_farfield_T(L, ws, order, T);
    for (int64_t j = 0; j < n; j++) {
        double pw[3][ORC_PMAX + 1];
        for (int k = 0; k < 3; k++) {
            double d = (double)pos[3 * j + k] - 0.5 * L;
            pw[k][0] = 1.0;
            for (int e = 1; e <= order; e++) pw[k][e] = pw[k][e - 1] * d;
        }
        for (int i = 0; i < np; i++) M[i] += (double)mass[j] * pw[0][ea[i]] * pw[1][eb[i]] * pw[2][ec[i]];
    }
    /* O4b: with background subtraction the far images come with their backgrounds, i.e. the far-field operator acts
     * on delta rho = particles - rho_bar: M_k -= rho_bar int_box (y - c)^k d^3y  (exact: int_box psi = 0, so
     * int_box rho_bar Phi_far(x - y) d^3y is the potential of the homogeneous image block). */
    if (bg) {
        double cbox[3] = { 0.5 * L, 0.5 * L, 0.5 * L }, Cb[ORC_NP(ORC_PMAX)];
        orc_cube_moments(L, cbox, cbox, order, Cb);
        const double rhobar = M[0] / (L * L * L);
        for (int i = 0; i < np; i++) M[i] -= rhobar * Cb[i];            /* M_0 becomes 0: the box is neutral */
    }
    double binom[2 * ORC_PMAX + 1][2 * ORC_PMAX + 1];
    for (int i = 0; i <= 2 * ORC_PMAX; i++) {
        binom[i][0] = 1.0;
        for (int j = 1; j <= i; j++) binom[i][j] = (j == i) ? 1.0 : binom[i - 1][j - 1] + binom[i - 1][j];
    }
    for (int i = 0; i < np; i++) {
        int li = ea[i] + eb[i] + ec[i];
        double s = 0.0;
        for (int k = 0; k < np; k++) {
            int lk = ea[k] + eb[k] + ec[k];
            if (li + lk > order) break;
            double sg = (lk & 1) ? -1.0 : 1.0;
            s += sg * binom[ea[i] + ea[k]][ea[k]] * binom[eb[i] + eb[k]][eb[k]] * binom[ec[i] + ec[k]][ec[k]] *
                 M[k] * T[orc_midx(ea[i] + ea[k], eb[i] + eb[k], ec[i] + ec[k])];
        }
        Lambda[i] = s;
    }
    free(T); free(M);
}

/* pot_far = sum_n Lambda_n X^n,  acc_far,i = - sum_n n_i Lambda_n X^(n-e_i),  X = x - c  (O7 step 4) */
void orc_farfield_eval(const double *Lambda, int order, double L, int64_t nsink, const float *pos,
                       const int64_t *sink, double *acc, double *pot)
{
    int np = ORC_NP(order);
    int ea[ORC_NP(ORC_PMAX)], eb[ORC_NP(ORC_PMAX)], ec[ORC_NP(ORC_PMAX)];
    orc_mtable(order, ea, eb, ec);
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        double pw[3][ORC_PMAX + 1];
        for (int k = 0; k < 3; k++) {
            double d = (double)pos[3 * i + k] - 0.5 * L;
            pw[k][0] = 1.0;
            for (int e = 1; e <= order; e++) pw[k][e] = pw[k][e - 1] * d;
        }
        double ph = 0, a[3] = {0, 0, 0};
        for (int q = 0; q < np; q++) {
            int A = ea[q], B = eb[q], C = ec[q];
            ph += Lambda[q] * pw[0][A] * pw[1][B] * pw[2][C];
            if (A) a[0] -= A * Lambda[q] * pw[0][A - 1] * pw[1][B] * pw[2][C];
            if (B) a[1] -= B * Lambda[q] * pw[0][A] * pw[1][B - 1] * pw[2][C];
            if (C) a[2] -= C * Lambda[q] * pw[0][A] * pw[1][B] * pw[2][C - 1];
        }
        for (int k = 0; k < 3; k++) acc[3 * s + k] = a[k];
        if (pot) pot[s] = ph;
    }
}

/* ---- O9 comoving KDK factors (reading A13; "symplectic integrator") ---------------
 * Einstein-de Sitter, H0^2 = (8 pi/3) G M_tot / box^3, H(a) = H0 a^(-3/2):
 *   kick  K(a1,a2) = int dt/a   = (2/H0)(sqrt(a2) - sqrt(a1))
 *   drift D(a1,a2) = int dt/a^2 = (2/H0)(a1^(-1/2) - a2^(-1/2))
 * step a -> a+da: v += g K(a, a+da/2); x += v D(a, a+da); wrap; g = force(x); v += g K(a+da/2, a+da).
 * periodic = 0: Newtonian, `a` ignored, da = dt: K1 = K2 = dt/2, D = dt. */
void orc_kdk_factors(int periodic, double mtot, double box, double a, double da, double *k1,
                     double *drift, double *k2)
{
    if (!periodic) { *k1 = 0.5 * da; *drift = da; *k2 = 0.5 * da; return; }
    double H0 = sqrt(8.0 * PI / 3.0 * mtot / (box * box * box));
    double am = a + 0.5 * da, a1 = a + da;
    *k1 = 2.0 / H0 * (sqrt(am) - sqrt(a));
    *k2 = 2.0 / H0 * (sqrt(a1) - sqrt(am));
    *drift = 2.0 / H0 * (1.0 / sqrt(a) - 1.0 / sqrt(a1));
}

/* ---- O9b Friedmann kick/drift factors ("All of these simulations utilize the
 * exact same cosmology with (Omega_m, ..., Omega_Lambda, ...) = (0.295, ..., 0.705, ...)") -------------------------
 * Same state and composition as O9; only H(a) changes:
 *   H(a) = H0 E(a),  E(a)^2 = Omega_m a^-3 + Omega_k a^-2 + Omega_L,  Omega_k = 1 - Omega_m - Omega_L,
 *   H0^2 = (8 pi/3) G rho_crit, and the box holds the MATTER: M_tot/box^3 = Omega_m rho_crit,
 *   kick  K(a1,a2) = int dt/a   = (1/H0) int_{a1}^{a2} da / (a^2 E(a))
 *   drift D(a1,a2) = int dt/a^2 = (1/H0) int_{a1}^{a2} da / (a^3 E(a))
 * (dt = da / (a H)).  Omega_m = 1, Omega_L = 0 is Einstein-de Sitter and must reproduce orc_kdk_factors.
 * Plain composite Simpson rule, 4096 panels per integral. */
static double simpson_friedmann(double a1, double a2, int apow, double om, double ol)
{
    const int n = 4096;
    const double ok = 1.0 - om - ol, h = (a2 - a1) / n;
    double sum = 0.0;
    for (int i = 0; i <= n; i++) {
        const double a = a1 + h * i;
        const double E = sqrt(om / (a * a * a) + ok / (a * a) + ol);
        const double f = 1.0 / (pow(a, (double)apow) * E);
        sum += f * ((i == 0 || i == n) ? 1.0 : ((i & 1) ? 4.0 : 2.0));
    }
    return sum * h / 3.0;
}

void orc_kdk_factors_friedmann(double mtot, double box, double omega_m, double omega_l, double a, double da,
                               double *k1, double *drift, double *k2)
{
    const double H0 = sqrt(8.0 * PI / 3.0 * mtot / (box * box * box) / omega_m);
    const double am = a + 0.5 * da, a1 = a + da;
    *k1 = simpson_friedmann(a, am, 2, omega_m, omega_l) / H0;
    *k2 = simpson_friedmann(am, a1, 2, omega_m, omega_l) / H0;
    *drift = simpson_friedmann(a, a1, 3, omega_m, omega_l) / H0;
}
