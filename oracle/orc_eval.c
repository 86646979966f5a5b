/* orc_eval.c — ORACLE (test infrastructure): direct summation D-iso and the serial tree
 * evaluation Tr (group walk under the opening-angle MAC, then P2P + M2P), SURVEY.md §8(c) D, O5, O6.
 * PAPER.md:57 (bodies interacting through a truncated expansion), PAPER.md:61 (traversal),
 * PAPER.md:69-75 (m x n blocks of sources shared by the sinks of one sink cell; direct
 * interactions near the leaves, multipole interactions for the rest).  G = 1.
 * Shares nothing with the CUDA path.
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int orc_get_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---- D-iso: Plummer-softened direct sum (reading A8, A10) -------------------------------------
 * pot_i = - sum_{j != i} m_j (r_ij^2 + eps^2)^(-1/2)
 * acc_i = - sum_{j != i} m_j (x_i - x_j) (r_ij^2 + eps^2)^(-3/2)            j != i BY INDEX   */
void orc_direct_iso(int64_t n, const float *pos, const float *mass, double eps, int64_t nsink,
                    const int64_t *sink, double *acc, double *pot)
{
    double e2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        double ax = 0, ay = 0, az = 0, ph = 0;
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double dx = xi - (double)pos[3 * j], dy = yi - (double)pos[3 * j + 1],
                   dz = zi - (double)pos[3 * j + 2];
            double R2 = dx * dx + dy * dy + dz * dz + e2;
            double rinv = 1.0 / sqrt(R2), m = (double)mass[j];
            double mr3 = m * rinv / R2;
            ax -= mr3 * dx; ay -= mr3 * dy; az -= mr3 * dz; ph -= m * rinv;
        }
        acc[3 * s] = ax; acc[3 * s + 1] = ay; acc[3 * s + 2] = az;
        if (pot) pot[s] = ph;
    }
}

/* ---- O6: Taylor coefficients b_n = d^n g / n!  of  g(r) = (|r|^2 + eps^2)^(-1/2) ---------------
 * b_0 = 1/R,  R^2 = |r|^2 + eps^2 ;  for |n| >= 1
 *   |n| R^2 b_n + (2|n|-1) sum_i r_i b_{n-e_i} + (|n|-1) sum_i b_{n-2e_i} = 0
 * (terms with a negative index are 0).  b must hold ORC_NP(pmax) doubles. */
void orc_bn(int pmax, const double r[3], double eps2, double *b)
{
    double R2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + eps2;
    b[0] = 1.0 / sqrt(R2);
    for (int l = 1; l <= pmax; l++)
        for (int a = l; a >= 0; a--)
            for (int bb = l - a; bb >= 0; bb--) {
                int c = l - a - bb;
                double s1 = 0.0, s2 = 0.0;
                if (a >= 1) s1 += r[0] * b[orc_midx(a - 1, bb, c)];
                if (bb >= 1) s1 += r[1] * b[orc_midx(a, bb - 1, c)];
                if (c >= 1) s1 += r[2] * b[orc_midx(a, bb, c - 1)];
                if (a >= 2) s2 += b[orc_midx(a - 2, bb, c)];
                if (bb >= 2) s2 += b[orc_midx(a, bb - 2, c)];
                if (c >= 2) s2 += b[orc_midx(a, bb, c - 2)];
                b[orc_midx(a, bb, c)] = -((2 * l - 1) * s1 + (l - 1) * s2) / (l * R2);
            }
}

/* pot += - sum_{|n|<=p} (-1)^|n| M_n b_n(r)
 * acc_i += sum_{|n|<=p} (-1)^|n| (n_i + 1) M_n b_{n+e_i}(r)         r = sink - expansion centre */
void orc_m2p(int p, const double *mom, const double r[3], double eps2, double acc[3], double *pot)
{
    double b[ORC_NP(ORC_PMAX)];
    orc_bn(p + 1, r, eps2, b);
    for (int l = 0; l <= p; l++)
        for (int a = l; a >= 0; a--)
            for (int bb = l - a; bb >= 0; bb--) {
                int c = l - a - bb;
                double sg = (l & 1) ? -1.0 : 1.0, M = mom[orc_midx(a, bb, c)];
                if (pot) *pot -= sg * M * b[orc_midx(a, bb, c)];
                acc[0] += sg * (a + 1) * M * b[orc_midx(a + 1, bb, c)];
                acc[1] += sg * (bb + 1) * M * b[orc_midx(a, bb + 1, c)];
                acc[2] += sg * (c + 1) * M * b[orc_midx(a, bb, c + 1)];
            }
}

/* ---- O5: walk of one sink group ------------------------------------------------------------- */
typedef struct {
    int64_t *cell; int32_t *img; int64_t n, cap;
} ilist_t;

static void il_push(ilist_t *l, int64_t c, int32_t im)
{
    if (l->n == l->cap) {
        l->cap = l->cap ? 2 * l->cap : 1024;
        l->cell = realloc(l->cell, sizeof(int64_t) * l->cap);
        l->img = realloc(l->img, sizeof(int32_t) * l->cap);
    }
    l->cell[l->n] = c; l->img[l->n] = im; l->n++;
}

typedef struct {
    const orc_tree *t; const float *bb; double theta; double shift[3]; int32_t im;
    ilist_t *m2p, *p2p;
} walk_t;

static void walk_rec(walk_t *w, int64_t c)
{
    const orc_tree *t = w->t;
    double s = (double)t->box * ldexp(1.0, -t->level[c]);
    /* d = Euclidean distance from the shifted centre of mass to the group's AABB (0 if inside) */
    double d2 = 0.0;
    for (int k = 0; k < 3; k++) {
        double z = t->com[3 * c + k] + w->shift[k];
        double lo = (double)w->bb[k] - z, hi = z - (double)w->bb[3 + k];
        double dk = lo > 0.0 ? lo : (hi > 0.0 ? hi : 0.0);
        d2 += dk * dk;
    }
    double rc = s / w->theta + t->delta[c];
    if (d2 > rc * rc) { il_push(w->m2p, c, w->im); return; }           /* accept (strict)    */
    if (t->nchild[c] == 0) { il_push(w->p2p, c, w->im); return; }      /* leaf -> direct     */
    for (int k = 0; k < t->nchild[c]; k++) walk_rec(w, t->child0[c] + k);
}

static void walk_group(const orc_tree *t, int64_t g, double theta, int ws, ilist_t *m2p, ilist_t *p2p)
{
    walk_t w = { t, t->gbox + 6 * g, theta, {0, 0, 0}, 0, m2p, p2p };
    m2p->n = 0; p2p->n = 0;
    int W = t->periodic ? ws : 0, im = 0;
    for (int ix = -W; ix <= W; ix++)
        for (int iy = -W; iy <= W; iy++)
            for (int iz = -W; iz <= W; iz++, im++) {
                w.shift[0] = ix * (double)t->box; w.shift[1] = iy * (double)t->box;
                w.shift[2] = iz * (double)t->box; w.im = im;
                walk_rec(&w, 0);
            }
}

static void img_shift(const orc_tree *t, int ws, int32_t im, double sh[3])
{
    int W = t->periodic ? ws : 0, side = 2 * W + 1;
    int iz = im % side - W, iy = (im / side) % side - W, ix = im / (side * side) - W;
    sh[0] = ix * (double)t->box; sh[1] = iy * (double)t->box; sh[2] = iz * (double)t->box;
}

void orc_group_list_counts(orc_tree *t, double theta, int ws, int64_t g, int64_t *n_m2p_cells,
                           int64_t *n_p2p_leaves, int64_t *n_p2p_particles)
{
    ilist_t m2p = {0}, p2p = {0};
    walk_group(t, g, theta, ws, &m2p, &p2p);
    *n_m2p_cells = m2p.n; *n_p2p_leaves = p2p.n;
    int64_t np = 0;
    for (int64_t k = 0; k < p2p.n; k++) np += t->count[p2p.cell[k]];
    *n_p2p_particles = np;
    free(m2p.cell); free(m2p.img); free(p2p.cell); free(p2p.img);
}

/* The two lists of group g themselves (for the tests that pin the acceptance rule): cell indices (canonical
 * order) and image ids, in walk order.  Call with cap = 0 to get the lengths, then with buffers of that size. */
void orc_group_lists(orc_tree *t, double theta, int ws, int64_t g, int64_t cap, int64_t *m2p_cell,
                     int32_t *m2p_img, int64_t *n_m2p, int64_t *p2p_cell, int32_t *p2p_img, int64_t *n_p2p)
{
    ilist_t m2p = {0}, p2p = {0};
    walk_group(t, g, theta, ws, &m2p, &p2p);
    *n_m2p = m2p.n; *n_p2p = p2p.n;
    for (int64_t k = 0; k < m2p.n && k < cap; k++) { m2p_cell[k] = m2p.cell[k]; m2p_img[k] = m2p.img[k]; }
    for (int64_t k = 0; k < p2p.n && k < cap; k++) { p2p_cell[k] = p2p.cell[k]; p2p_img[k] = p2p.img[k]; }
    free(m2p.cell); free(m2p.img); free(p2p.cell); free(p2p.img);
}

/* group containing sorted rank r (groups tile [0,n) in Morton order) */
static int64_t group_of_rank(const orc_tree *t, int64_t r)
{
    int64_t lo = 0, hi = t->ngroup - 1;
    while (lo < hi) {
        int64_t mid = (lo + hi + 1) / 2;
        if (t->gfirst[mid] <= r) lo = mid; else hi = mid - 1;
    }
    return lo;
}

typedef struct { int64_t g, s; } gs_t;
static int gs_cmp(const void *a, const void *b)
{
    const gs_t *x = a, *y = b;
    if (x->g != y->g) return x->g < y->g ? -1 : 1;
    return x->s < y->s ? -1 : (x->s > y->s);
}

/* Tr: acc/pot of the requested sinks (caller-order particle indices; NULL = all), for the tree
 * whose moments were filled by orc_moments(t, p).  n_p2p / n_m2p (may be NULL) receive the
 * number of particle-particle and cell-particle interactions evaluated for these sinks.
 * Periodic: only the (2 ws + 1)^3 image block is summed here; O7's far field is added by the
 * caller (orc_farfield_*). */
int orc_tree_accel(orc_tree *t, double eps, double theta, int ws, int64_t nsink,
                   const int64_t *sink, double *acc, double *pot, int64_t *n_p2p, int64_t *n_m2p)
{
    if (t->p < 0) return -3;
    int p = t->p, np = ORC_NP(p);
    double e2 = eps * eps;
    gs_t *gs = malloc(sizeof(gs_t) * (size_t)(nsink > 0 ? nsink : 1));
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        gs[s].g = group_of_rank(t, t->rank_of[i]); gs[s].s = s;
    }
    qsort(gs, (size_t)nsink, sizeof(gs_t), gs_cmp);
    /* runs of equal group */
    int64_t nrun = 0, *run = malloc(sizeof(int64_t) * (size_t)(nsink + 1));
    for (int64_t s = 0; s < nsink; s++) if (s == 0 || gs[s].g != gs[s - 1].g) run[nrun++] = s;
    run[nrun] = nsink;
    int64_t tot_p2p = 0, tot_m2p = 0;
#pragma omp parallel reduction(+ : tot_p2p, tot_m2p)
    {
        ilist_t m2p = {0}, p2p = {0};
#pragma omp for schedule(dynamic, 1)
        for (int64_t q = 0; q < nrun; q++) {
            int64_t g = gs[run[q]].g;
            walk_group(t, g, theta, ws, &m2p, &p2p);
            for (int64_t u = run[q]; u < run[q + 1]; u++) {
                int64_t s = gs[u].s, i = sink ? sink[s] : s, r = t->rank_of[i];
                const double *x = t->spos + 3 * r;
                double a[3] = {0, 0, 0}, ph = 0.0;
                /* P2P over the listed leaves */
                for (int64_t k = 0; k < p2p.n; k++) {
                    int64_t c = p2p.cell[k];
                    double sh[3]; img_shift(t, ws, p2p.img[k], sh);
                    int self_image = (sh[0] == 0.0 && sh[1] == 0.0 && sh[2] == 0.0);
                    for (int64_t j = t->first[c]; j < t->first[c] + t->count[c]; j++) {
                        if (self_image && j == r) continue;
                        double dx = x[0] - (t->spos[3 * j] + sh[0]), dy = x[1] - (t->spos[3 * j + 1] + sh[1]),
                               dz = x[2] - (t->spos[3 * j + 2] + sh[2]);
                        double R2 = dx * dx + dy * dy + dz * dz + e2, rinv = 1.0 / sqrt(R2);
                        double mr3 = t->smass[j] * rinv / R2;
                        a[0] -= mr3 * dx; a[1] -= mr3 * dy; a[2] -= mr3 * dz; ph -= t->smass[j] * rinv;
                        tot_p2p++;
                    }
                }
                /* M2P over the listed cells */
                for (int64_t k = 0; k < m2p.n; k++) {
                    int64_t c = m2p.cell[k];
                    double sh[3], rr[3]; img_shift(t, ws, m2p.img[k], sh);
                    for (int d = 0; d < 3; d++) rr[d] = x[d] - (t->com[3 * c + d] + sh[d]);
                    orc_m2p(p, t->mom + (size_t)np * c, rr, e2, a, &ph);
                    tot_m2p++;
                }
                acc[3 * s] = a[0]; acc[3 * s + 1] = a[1]; acc[3 * s + 2] = a[2];
                if (pot) pot[s] = ph;
            }
        }
        free(m2p.cell); free(m2p.img); free(p2p.cell); free(p2p.img);
    }
    if (n_p2p) *n_p2p = tot_p2p;
    if (n_m2p) *n_m2p = tot_m2p;
    free(gs); free(run);
    return 0;
}
