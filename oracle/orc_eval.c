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
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < nsink; s++) {
        int64_t i = sink ? sink[s] : s;
        double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        double ax = 0, ay = 0, az = 0, ph = 0;
        for (int64_t j = 0; j < n; j++) {
            if (j == i) continue;
            double dx = xi - (double)pos[3 * j], dy = yi - (double)pos[3 * j + 1],
                   dz = zi - (double)pos[3 * j + 2];
            double f, phi, m = (double)mass[j];
            orc_soft_pair(dx * dx + dy * dy + dz * dz, eps, &f, &phi);      /* Plummer: (r^2+eps^2)^(-3/2), (r^2+eps^2)^(-1/2) */
            double mr3 = m * f;
            ax -= mr3 * dx; ay -= mr3 * dy; az -= mr3 * dz; ph -= m * phi;
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
    int64_t *cell; int32_t *img; int8_t *sub; int64_t n, cap;
} ilist_t;

static void il_push(ilist_t *l, int64_t c, int32_t im, int8_t sub)
{
    if (l->n == l->cap) {
        l->cap = l->cap ? 2 * l->cap : 1024;
        l->cell = realloc(l->cell, sizeof(int64_t) * l->cap);
        l->img = realloc(l->img, sizeof(int32_t) * l->cap);
        l->sub = realloc(l->sub, sizeof(int8_t) * l->cap);
    }
    l->cell[l->n] = c; l->img[l->n] = im; l->sub[l->n] = sub; l->n++;
}
static void il_free(ilist_t *l) { free(l->cell); free(l->img); free(l->sub); }

/* cubes whose background is summed one by one: index ranges [lo, hi] (inclusive) in level-l_b cells, unwrapped frame */
typedef struct { int64_t *lohi; int64_t n, cap; } cubes_t;

typedef struct {
    const orc_tree *t; const float *bb; double theta; double shift[3]; int32_t im; int64_t ishift[3];
    ilist_t *m2p, *p2p;
    /* O4b */
    int bg, lb; int64_t wlo[3], whi[3]; cubes_t *left;
} walk_t;

/* O4b: a cube of the image block whose background no accepted cell carries.  Inside the window it is part of the
 * window's cuboid; otherwise it is kept and summed by itself (minus its overlap with the window). */
static void expose(walk_t *w, const int64_t lo[3], const int64_t hi[3])
{
    int inside = 1;
    for (int k = 0; k < 3; k++) if (lo[k] < w->wlo[k] || hi[k] > w->whi[k]) inside = 0;
    if (inside) return;
    cubes_t *q = w->left;
    if (q->n == q->cap) { q->cap = q->cap ? 2 * q->cap : 64; q->lohi = realloc(q->lohi, sizeof(int64_t) * 6 * q->cap); }
    for (int k = 0; k < 3; k++) { q->lohi[6 * q->n + k] = lo[k]; q->lohi[6 * q->n + 3 + k] = hi[k]; }
    q->n++;
}

/* O5b (reading; "We adjust the error tolerance parameter to limit absolute errors ..."): an upper bound on the
 * acceleration error of the order-p expansion of cell c at distance d from its expansion centre z,
 *     E_c(d) = (p + 2) B_{p+1} / (d^(p+1) (d - b)^2),     d > b,
 * b = (sqrt(3)/2) s + delta  the radius of the ball about z that holds the cell's cube, B_{p+1} = sum m |y - z|^(p+1) bounded by
 * Q b^(p-1), Q = sum m |y - z|^2 = M_200 + M_020 + M_002 (an exact moment).  It follows from |grad (P_n(cos g)/r^(n+1))| ~ (n+1)/r^(n+2):
 * sum_{n>p} (n+1) B_n / d^(n+2) <= B_{p+1}/d^(p+3) sum_k (p+2+k)(b/d)^k <= (p+2) B_{p+1}/(d^(p+1)(d-b)^2)   (Salmon & Warren 1994's form).
 * sub: the cell is listed with background-subtracted moments (O4b): the sources are |particles| + |rho_bar cube|,
 * Q' = Q + rho_bar tr C = 2 Q - tr M'. */
double orc_mac_bound(const orc_tree *t, int64_t c, int sub, double d)
{
    const int p = t->p, np = ORC_NP(p);
    const double s = (double)t->box * ldexp(1.0, -t->level[c]), b = 0.5 * sqrt(3.0) * s + t->delta[c];
    const double *M = t->mom + (size_t)np * c;
    double Q = M[orc_midx(2, 0, 0)] + M[orc_midx(0, 2, 0)] + M[orc_midx(0, 0, 2)];
    if (sub) {
        const double *Mb = t->mom_bg + (size_t)np * c;
        Q = 2.0 * Q - (Mb[orc_midx(2, 0, 0)] + Mb[orc_midx(0, 2, 0)] + Mb[orc_midx(0, 0, 2)]);
    }
    if (!(d > b)) return INFINITY;
    return (p + 2) * Q * pow(b, p - 1) / (pow(d, p + 1) * (d - b) * (d - b));
}

void orc_tree_set_mac(orc_tree *t, int kind, double tol) { t->mac_kind = kind; t->mac_tol = tol; }

static void walk_rec(walk_t *w, int64_t c)
{
    const orc_tree *t = w->t;
    const int level = t->level[c];
    double s = (double)t->box * ldexp(1.0, -level);
    /* O4b: cells of level <= l_b know where they lie relative to the group's window (integer test on level-l_b cells) */
    const int top = w->bg && level <= w->lb;
    int inside = 0, inter = 0;
    int64_t lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, q[3] = {0, 0, 0};
    if (top) {
        orc_cell_coords(t, c, q);
        inside = inter = 1;
        for (int k = 0; k < 3; k++) {
            lo[k] = (q[k] << (w->lb - level)) + (w->ishift[k] << w->lb);
            hi[k] = lo[k] + ((int64_t)1 << (w->lb - level)) - 1;
            if (lo[k] < w->wlo[k] || hi[k] > w->whi[k]) inside = 0;
            if (lo[k] > w->whi[k] || hi[k] < w->wlo[k]) inter = 0;
        }
    }
    /* d = Euclidean distance from the shifted centre of mass to the group's AABB (0 if inside) */
    double d2 = 0.0;
    for (int k = 0; k < 3; k++) {
        double z = t->com[3 * c + k] + w->shift[k];
        double l0 = (double)w->bb[k] - z, h0 = z - (double)w->bb[3 + k];
        double dk = l0 > 0.0 ? l0 : (h0 > 0.0 ? h0 : 0.0);
        d2 += dk * dk;
    }
    double rc = s / w->theta + t->delta[c];
    /* a cell that sticks out of the window (partly in, partly out) is never accepted: its cube's background would be
     * counted twice inside the window */
    const int straddles = top && inter && !inside;
    int ok;
    /* O6b: with the compact K1 kernel a cell is expanded (Newtonian) only if every source lies outside the kernel's support of every
     * sink: d - b > h, b = sqrt(3)/2 s + delta the radius of the ball about the expansion centre that holds the cell */
    const int k1_near = orc_get_softening() == 1 && !(sqrt(d2) - (0.5 * sqrt(3.0) * s + t->delta[c]) > t->soft_len);
    if (t->mac_kind == 0) ok = d2 > rc * rc;                            /* opening angle (strict) */
    else {                                                              /* O5b: theta = 1 for validity, then the error bound */
        double r1 = s + t->delta[c];
        ok = d2 > r1 * r1 && orc_mac_bound(t, c, top && !inter, sqrt(d2)) <= t->mac_tol;
    }
    if (!straddles && !k1_near && ok) {                                 /* accept             */
        il_push(w->m2p, c, w->im, (int8_t)(top && !inter));              /* outside the window: background subtracted */
        return;
    }
    if (t->nchild[c] == 0) {                                            /* leaf -> direct     */
        il_push(w->p2p, c, w->im, 0);
        if (top) expose(w, lo, hi);
        return;
    }
    if (top && level == w->lb) expose(w, lo, hi);                       /* below l_b nothing carries a background */
    int present = 0;
    for (int k = 0; k < t->nchild[c]; k++) {
        present |= 1 << (int)(t->hotkey[t->child0[c] + k] & 7u);
        walk_rec(w, t->child0[c] + k);
    }
    if (top && level < w->lb)                                           /* empty octants hold background only */
        for (int o = 0; o < 8; o++) {
            if (present & (1 << o)) continue;
            int64_t lo2[3], hi2[3];
            const int bit[3] = { (o >> 2) & 1, (o >> 1) & 1, o & 1 };
            for (int k = 0; k < 3; k++) {
                lo2[k] = ((2 * q[k] + bit[k]) << (w->lb - level - 1)) + (w->ishift[k] << w->lb);
                hi2[k] = lo2[k] + ((int64_t)1 << (w->lb - level - 1)) - 1;
            }
            expose(w, lo2, hi2);
        }
}

/* lists of group g; bg != 0 (periodic only): reading O4b, `left` receives the cubes to be summed one by one and
 * window[6] the window's index range (lo xyz, hi xyz; level-l_b cells) */
static void walk_group(const orc_tree *t, int64_t g, double theta, int ws, int bg, ilist_t *m2p, ilist_t *p2p,
                       cubes_t *left, int64_t window[6])
{
    walk_t w;
    memset(&w, 0, sizeof(w));
    w.t = t; w.bb = t->gbox + 6 * g; w.theta = theta; w.m2p = m2p; w.p2p = p2p;
    w.bg = bg && t->periodic; w.left = left;
    m2p->n = 0; p2p->n = 0;
    if (left) left->n = 0;
    if (w.bg) {
        w.lb = t->bg_level;
        const int k = orc_bg_halfwidth(theta, ws, w.lb);
        const int64_t cg = t->gcell[g];
        const int lg = t->level[cg];
        int64_t qg[3];
        orc_cell_coords(t, cg, qg);
        for (int d = 0; d < 3; d++) {
            int64_t flo, fhi;                 /* footprint of the group's cell in level-l_b cells */
            if (lg >= w.lb) flo = fhi = qg[d] >> (lg - w.lb);
            else { flo = qg[d] << (w.lb - lg); fhi = flo + ((int64_t)1 << (w.lb - lg)) - 1; }
            w.wlo[d] = flo - k; w.whi[d] = fhi + k;
            if (window) { window[d] = w.wlo[d]; window[3 + d] = w.whi[d]; }
        }
    }
    int W = t->periodic ? ws : 0, im = 0;
    for (int ix = -W; ix <= W; ix++)
        for (int iy = -W; iy <= W; iy++)
            for (int iz = -W; iz <= W; iz++, im++) {
                w.shift[0] = ix * (double)t->box; w.shift[1] = iy * (double)t->box;
                w.shift[2] = iz * (double)t->box; w.im = im;
                w.ishift[0] = ix; w.ishift[1] = iy; w.ishift[2] = iz;
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
    walk_group(t, g, theta, ws, 0, &m2p, &p2p, NULL, NULL);
    *n_m2p_cells = m2p.n; *n_p2p_leaves = p2p.n;
    int64_t np = 0;
    for (int64_t k = 0; k < p2p.n; k++) np += t->count[p2p.cell[k]];
    *n_p2p_particles = np;
    il_free(&m2p); il_free(&p2p);
}

/* The lists of group g themselves (for the tests that pin the acceptance rule): cell indices (canonical order), image
 * ids and, with bg, whether the entry carries the background-subtracted moments; the cubes summed one by one
 * (left_lohi: 6 int64 each) and the window.  Call with cap = 0 to get the lengths, then with buffers of that size. */
void orc_group_lists(orc_tree *t, double theta, int ws, int bg, int64_t g, int64_t cap, int64_t *m2p_cell,
                     int32_t *m2p_img, int8_t *m2p_sub, int64_t *n_m2p, int64_t *p2p_cell, int32_t *p2p_img,
                     int64_t *n_p2p, int64_t *left_lohi, int64_t *n_left, int64_t window[6])
{
    ilist_t m2p = {0}, p2p = {0};
    cubes_t left = {0};
    int64_t win[6] = {0, 0, 0, 0, 0, 0};
    walk_group(t, g, theta, ws, bg, &m2p, &p2p, &left, win);
    *n_m2p = m2p.n; *n_p2p = p2p.n;
    if (n_left) *n_left = left.n;
    if (window) for (int k = 0; k < 6; k++) window[k] = win[k];
    for (int64_t k = 0; k < m2p.n && k < cap; k++) { m2p_cell[k] = m2p.cell[k]; m2p_img[k] = m2p.img[k]; if (m2p_sub) m2p_sub[k] = m2p.sub[k]; }
    for (int64_t k = 0; k < p2p.n && k < cap; k++) { p2p_cell[k] = p2p.cell[k]; p2p_img[k] = p2p.img[k]; }
    if (left_lohi) for (int64_t k = 0; k < left.n && k < cap; k++) memcpy(left_lohi + 6 * k, left.lohi + 6 * k, sizeof(int64_t) * 6);
    il_free(&m2p); il_free(&p2p); free(left.lohi);
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
int orc_tree_accel(orc_tree *t, double eps, double theta, int ws, int bg, int64_t nsink,
                   const int64_t *sink, double *acc, double *pot, int64_t *n_p2p, int64_t *n_m2p)
{
    if (t->p < 0) return -3;
    int p = t->p, np = ORC_NP(p);
    /* the far cells are expanded with the softened Green's function of reading A8 (Plummer), or, for the compact K1 kernel,
     * with the Newtonian one: the walk then accepts a cell only if all its sources are farther than h from the group (O6b) */
    double e2 = orc_get_softening() == 0 ? eps * eps : 0.0;
    t->soft_len = eps;
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
        cubes_t left = {0};
        int64_t win[6];
        const int use_bg = bg && t->periodic;
        const double sb = use_bg ? (double)t->box * ldexp(1.0, -t->bg_level) : 0.0;     /* side of a level-l_b cell */
#pragma omp for schedule(dynamic, 1)
        for (int64_t q = 0; q < nrun; q++) {
            int64_t g = gs[run[q]].g;
            walk_group(t, g, theta, ws, bg, &m2p, &p2p, &left, win);
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
                        double f, phi;
                        orc_soft_pair(dx * dx + dy * dy + dz * dz, eps, &f, &phi);
                        double mr3 = t->smass[j] * f;
                        a[0] -= mr3 * dx; a[1] -= mr3 * dy; a[2] -= mr3 * dz; ph -= t->smass[j] * phi;
                        tot_p2p++;
                    }
                }
                /* M2P over the listed cells */
                for (int64_t k = 0; k < m2p.n; k++) {
                    int64_t c = m2p.cell[k];
                    double sh[3], rr[3]; img_shift(t, ws, m2p.img[k], sh);
                    for (int d = 0; d < 3; d++) rr[d] = x[d] - (t->com[3 * c + d] + sh[d]);
                    orc_m2p(p, (m2p.sub[k] ? t->mom_bg : t->mom) + (size_t)np * c, rr, e2, a, &ph);
                    tot_m2p++;
                }
                /* O4b: the background (density -rho_bar) that no accepted cell carries, summed exactly: the window's
                 * cuboid, and every kept cube minus its part inside the window.  Newtonian closed form. */
                if (use_bg) {
                    double lo[3], hi[3], I, gg[3];
                    for (int d = 0; d < 3; d++) { lo[d] = win[d] * sb; hi[d] = (win[3 + d] + 1) * sb; }
                    orc_cuboid_field(lo, hi, x, &I, gg);
                    ph += t->rhobar * I;
                    for (int d = 0; d < 3; d++) a[d] -= t->rhobar * gg[d];
                    for (int64_t k = 0; k < left.n; k++) {
                        const int64_t *c6 = left.lohi + 6 * k;
                        int overlap = 1;
                        double olo[3], ohi[3];
                        for (int d = 0; d < 3; d++) {
                            lo[d] = c6[d] * sb; hi[d] = (c6[3 + d] + 1) * sb;
                            int64_t ol = c6[d] > win[d] ? c6[d] : win[d], oh = c6[3 + d] < win[3 + d] ? c6[3 + d] : win[3 + d];
                            if (ol > oh) overlap = 0;
                            olo[d] = ol * sb; ohi[d] = (oh + 1) * sb;
                        }
                        orc_cuboid_field(lo, hi, x, &I, gg);
                        ph += t->rhobar * I;
                        for (int d = 0; d < 3; d++) a[d] -= t->rhobar * gg[d];
                        if (overlap) {
                            orc_cuboid_field(olo, ohi, x, &I, gg);
                            ph -= t->rhobar * I;
                            for (int d = 0; d < 3; d++) a[d] += t->rhobar * gg[d];
                        }
                    }
                }
                acc[3 * s] = a[0]; acc[3 * s + 1] = a[1]; acc[3 * s + 2] = a[2];
                if (pot) pot[s] = ph;
            }
        }
        il_free(&m2p); il_free(&p2p); free(left.lohi);
    }
    if (n_p2p) *n_p2p = tot_p2p;
    if (n_m2p) *n_m2p = tot_m2p;
    free(gs); free(run);
    return 0;
}
