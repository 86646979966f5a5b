/* orc_moments.c — ORACLE (test infrastructure): cell multipole moments, SURVEY.md §8(c) O4.
 * PAPER.md:57 "truncated expansion to approximate the contribution of many bodies",
 * PAPER.md:75 "quadrupole and hexadecapole" => order p = highest moment rank kept (reading A9).
 * Full (non-traceless) Cartesian moments about the centre of mass (reading A7):
 *     M_n = sum_j m_j (y_j - z)^n ,  |n| <= p.
 * The oracle's moments are the plain definition (a direct sum over the cell's whole range);
 * orc_moments_m2m is the translation formula, kept only so a test can pin one against the other.
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

void orc_p2m_range(const orc_tree *t, int64_t first, int64_t count, int p, const double z[3],
                   double *mom)
{
    int np = ORC_NP(p);
    int ea[ORC_NP(ORC_PMAX)], eb[ORC_NP(ORC_PMAX)], ec[ORC_NP(ORC_PMAX)];
    orc_mtable(p, ea, eb, ec);
    for (int i = 0; i < np; i++) mom[i] = 0.0;
    for (int64_t r = first; r < first + count; r++) {
        double d[3], pw[3][ORC_PMAX + 1];
        for (int k = 0; k < 3; k++) {
            d[k] = t->spos[3 * r + k] - z[k];
            pw[k][0] = 1.0;
            for (int e = 1; e <= p; e++) pw[k][e] = pw[k][e - 1] * d[k];
        }
        for (int i = 0; i < np; i++) mom[i] += t->smass[r] * pw[0][ea[i]] * pw[1][eb[i]] * pw[2][ec[i]];
    }
}

void orc_moments(orc_tree *t, int p)
{
    int np = ORC_NP(p);
    free(t->cmass); free(t->com); free(t->delta); free(t->mom);
    t->p = p;
    t->cmass = malloc(sizeof(double) * (size_t)t->ncell);
    t->com = malloc(sizeof(double) * 3 * (size_t)t->ncell);
    t->delta = malloc(sizeof(double) * (size_t)t->ncell);
    t->mom = malloc(sizeof(double) * (size_t)np * (size_t)t->ncell);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t c = 0; c < t->ncell; c++) {
        double M = 0.0, z[3] = {0, 0, 0};
        for (int64_t r = t->first[c]; r < t->first[c] + t->count[c]; r++) {
            M += t->smass[r];
            for (int k = 0; k < 3; k++) z[k] += t->smass[r] * t->spos[3 * r + k];
        }
        double side, ctr[3];
        orc_cell_geometry(t, c, &side, ctr);
        if (M > 0.0) for (int k = 0; k < 3; k++) z[k] /= M;
        else for (int k = 0; k < 3; k++) z[k] = ctr[k];                 /* massless cell      */
        t->cmass[c] = M;
        double d2 = 0.0;
        for (int k = 0; k < 3; k++) { t->com[3 * c + k] = z[k]; d2 += (z[k] - ctr[k]) * (z[k] - ctr[k]); }
        t->delta[c] = sqrt(d2);
        orc_p2m_range(t, t->first[c], t->count[c], p, z, t->mom + (size_t)np * c);
    }
    /* O4b: for the cells of level <= l_b, the moments of  particles - rho_bar  over the cell's cube about the same
     * expansion centre (the centre of mass of the particles): M'_n = M_n - rho_bar C_n, C_n = orc_cube_moments. */
    free(t->mom_bg); t->mom_bg = NULL; t->ntop = 0;
    if (t->periodic && t->ncell > 0) {
        t->bg_level = orc_bg_level(t->n);
        t->rhobar = t->cmass[0] / ((double)t->box * t->box * t->box);
        while (t->ntop < t->ncell && t->level[t->ntop] <= t->bg_level) t->ntop++;
        t->mom_bg = malloc(sizeof(double) * (size_t)np * (size_t)t->ntop);
        for (int64_t c = 0; c < t->ntop; c++) {
            double side, ctr[3], C[ORC_NP(ORC_PMAX)];
            orc_cell_geometry(t, c, &side, ctr);
            orc_cube_moments(side, ctr, t->com + 3 * c, p, C);
            for (int i = 0; i < np; i++) t->mom_bg[(size_t)np * c + i] = t->mom[(size_t)np * c + i] - t->rhobar * C[i];
        }
    }
}

void orc_tree_get_moments_bg(const orc_tree *t, int32_t *bg_level, int64_t *ntop, double *rhobar, double *mom_bg)
{
    *bg_level = t->bg_level; *ntop = t->ntop; *rhobar = t->rhobar;
    if (mom_bg && t->mom_bg) memcpy(mom_bg, t->mom_bg, sizeof(double) * (size_t)ORC_NP(t->p) * (size_t)t->ntop);
}

/* M_n^parent = sum_children sum_{k<=n} C(n,k) M_k^child (z_child - z_parent)^(n-k)   (O4) */
void orc_moments_m2m(const orc_tree *t, int p, double *out)
{
    int np = ORC_NP(p);
    int ea[ORC_NP(ORC_PMAX)], eb[ORC_NP(ORC_PMAX)], ec[ORC_NP(ORC_PMAX)];
    orc_mtable(p, ea, eb, ec);
    double binom[ORC_PMAX + 1][ORC_PMAX + 1];
    for (int i = 0; i <= ORC_PMAX; i++) {
        binom[i][0] = 1.0;
        for (int j = 1; j <= i; j++) binom[i][j] = (j == i) ? 1.0 : binom[i - 1][j - 1] + binom[i - 1][j];
    }
    for (int64_t c = t->ncell - 1; c >= 0; c--) {            /* children have larger indices */
        double *Mp = out + (size_t)np * c;
        if (t->nchild[c] == 0) {
            orc_p2m_range(t, t->first[c], t->count[c], p, t->com + 3 * c, Mp);
            continue;
        }
        for (int i = 0; i < np; i++) Mp[i] = 0.0;
        for (int k = 0; k < t->nchild[c]; k++) {
            int64_t ch = t->child0[c] + k;
            const double *Mc = out + (size_t)np * ch;
            double d[3], pw[3][ORC_PMAX + 1];
            for (int q = 0; q < 3; q++) {
                d[q] = t->com[3 * ch + q] - t->com[3 * c + q];
                pw[q][0] = 1.0;
                for (int e = 1; e <= p; e++) pw[q][e] = pw[q][e - 1] * d[q];
            }
            for (int i = 0; i < np; i++)
                for (int a = 0; a <= ea[i]; a++)
                    for (int b = 0; b <= eb[i]; b++)
                        for (int cc = 0; cc <= ec[i]; cc++)
                            Mp[i] += binom[ea[i]][a] * binom[eb[i]][b] * binom[ec[i]][cc] *
                                     Mc[orc_midx(a, b, cc)] * pw[0][ea[i] - a] * pw[1][eb[i] - b] *
                                     pw[2][ec[i] - cc];
        }
    }
}

void orc_tree_get_moments(const orc_tree *t, double *cmass, double *com, double *delta, double *mom)
{
    int np = ORC_NP(t->p);
    memcpy(cmass, t->cmass, sizeof(double) * (size_t)t->ncell);
    memcpy(com, t->com, sizeof(double) * 3 * (size_t)t->ncell);
    memcpy(delta, t->delta, sizeof(double) * (size_t)t->ncell);
    memcpy(mom, t->mom, sizeof(double) * (size_t)np * (size_t)t->ncell);
}
