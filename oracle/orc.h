/* orc.h — fp64 CPU ORACLE for the 2HOT tree-force path (arxiv 1407.2600).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, headers,
 * tables or helpers with the CUDA path under paper_1407_2600_b200/csrc/.
 *
 * Everything here is plain, slow and written to be checked by eye against SURVEY.md §8(c)
 * (readings O1..O9 of the paper's prose).  fp64 throughout, except the
 * single fp32 multiply that turns a position into a key (reading O1/A3) and the fp32 periodic
 * wrap, both of which are *defined* in fp32.
 *
 * Multi-index convention (shared with include/dsk.h as an interface fact, not as code):
 * n = (a,b,c), rank l = a+b+c, index(n) = l(l+1)(l+2)/6 + (b+c)(b+c+1)/2 + c,
 * i.e. ranks ascending; within a rank a descending, then b descending.
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>
#include <stddef.h>

#define ORC_KEY_LEVELS 21
#define ORC_PMAX 10               /* highest rank any table here is built for           */
#define ORC_NP(p) (((p) + 1) * ((p) + 2) * ((p) + 3) / 6)

typedef struct orc_tree {
    int64_t n;
    float box;
    int periodic, nleaf, ncrit;
    float *pos;            /* [n,3] caller order, wrapped to [0,box) when periodic (fp32)  */
    float *mass;           /* [n]                                                           */
    uint64_t *key;         /* [n] caller order                                              */
    uint64_t *skey;        /* [n] sorted                                                    */
    uint32_t *order;       /* [n] skey[r] = key[order[r]]                                   */
    int64_t *rank_of;      /* [n] inverse permutation                                       */
    double *spos;          /* [n,3] sorted, exact fp64 copies of the fp32 positions         */
    double *smass;         /* [n]                                                           */
    /* O3 cells, canonical (ascending hotkey) order */
    int64_t ncell;
    uint64_t *hotkey;
    int64_t *first, *count, *child0;
    int32_t *nchild, *level;
    /* O5 groups, Morton order */
    int64_t ngroup;
    int64_t *gcell, *gfirst, *gcount;
    float *gbox;           /* [ngroup,6] = min xyz, max xyz (exact fp32 min/max)            */
    /* O4 moments (filled by orc_moments) */
    int p;
    double *cmass;         /* [ncell]                                                       */
    double *com;           /* [ncell,3]                                                     */
    double *delta;         /* [ncell]  |com - centre|                                       */
    double *mom;           /* [ncell, NP(p)] raw moments about com                          */
    /* O4b background subtraction (periodic only; filled by orc_moments) */
    int bg_level;          /* l_b                                                           */
    int64_t ntop;          /* cells of level <= l_b: the first ntop cells (level-major)     */
    double rhobar;         /* M_tot / box^3                                                 */
    double *mom_bg;        /* [ntop, NP(p)] moments of particles - rho_bar over the cube    */
    /* O5b acceptance rule in use (orc_tree_set_mac): 0 opening angle, 1 absolute error bound   */
    int mac_kind;
    double mac_tol;
    double soft_len;       /* softening length of the walk in progress (K1: the MAC needs h)  */
} orc_tree;

/* multi-index helpers (orc_tree.c) */
int orc_midx(int a, int b, int c);
void orc_mtable(int pmax, int *ea, int *eb, int *ec);     /* exponents of every index      */

/* O1-O3, O5 (orc_tree.c) */
int orc_keys(int64_t n, const float *pos, float box, int periodic, uint64_t *key, float *wrapped);
void orc_sort(int64_t n, const uint64_t *key, uint64_t *skey, uint32_t *order);
orc_tree *orc_tree_build(int64_t n, const float *pos, const float *mass, float box, int periodic,
                         int nleaf, int ncrit, int *err);
void orc_tree_free(orc_tree *t);
void orc_cell_geometry(const orc_tree *t, int64_t c, double *side, double centre[3]);

/* O4 (orc_moments.c) */
void orc_p2m_range(const orc_tree *t, int64_t first, int64_t count, int p, const double z[3],
                   double *mom);
void orc_moments(orc_tree *t, int p);
void orc_moments_m2m(const orc_tree *t, int p, double *mom_out);

/* O6 + D-iso (orc_eval.c) */
void orc_bn(int pmax, const double r[3], double eps2, double *b);
void orc_m2p(int p, const double *mom, const double r[3], double eps2, double acc[3], double *pot);
void orc_direct_iso(int64_t n, const float *pos, const float *mass, double eps, int64_t nsink,
                    const int64_t *sink, double *acc, double *pot);
int orc_tree_accel(orc_tree *t, double eps, double theta, int ws, int bg, int64_t nsink,
                   const int64_t *sink, double *acc, double *pot, int64_t *n_p2p, int64_t *n_m2p);
void orc_group_list_counts(orc_tree *t, double theta, int ws, int64_t g, int64_t *n_m2p_cells,
                           int64_t *n_p2p_leaves, int64_t *n_p2p_particles);

void orc_group_lists(orc_tree *t, double theta, int ws, int bg, int64_t g, int64_t cap, int64_t *m2p_cell,
                     int32_t *m2p_img, int8_t *m2p_sub, int64_t *n_m2p, int64_t *p2p_cell, int32_t *p2p_img,
                     int64_t *n_p2p, int64_t *left_lohi, int64_t *n_left, int64_t window[6]);
void orc_cell_coords(const orc_tree *t, int64_t c, int64_t q[3]);
void orc_tree_set_mac(orc_tree *t, int kind, double tol);
double orc_mac_bound(const orc_tree *t, int64_t c, int sub, double d);

/* softening law: 0 Plummer, 1 Dehnen K1 (orc_soft.c); a setting of the whole oracle library */
void orc_set_softening(int kind);
int orc_get_softening(void);
void orc_soft_pair(double r2, double len, double *f, double *phi);

/* background subtraction, reading O4b (orc_bg.c) */
void orc_cuboid_field(const double lo[3], const double hi[3], const double x[3], double *I, double g[3]);
void orc_cube_moments(double s, const double ctr[3], const double z[3], int p, double *C);
int orc_bg_level(int64_t n);
int orc_bg_halfwidth(double theta, int ws, int lb);

/* D-per, O7 (orc_periodic.c) */
void orc_ewald_pair(const double x[3], double L, double alpha, int nmax, int hmax, double *psi,
                    double a[3]);
double orc_ewald_self(double L, double alpha, int nmax, int hmax);
void orc_direct_per(int64_t n, const float *pos, const float *mass, double L, double eps, int ws,
                    double alpha, int64_t nsink, const int64_t *sink, double *acc, double *pot);
void orc_direct_per_pairwise(int64_t n, const float *pos, const float *mass, double L, double eps,
                             int ws, double alpha, int64_t nsink, const int64_t *sink, double *acc,
                             double *pot);
void orc_farfield_T(double L, int ws, int order, double *T);
double orc_farfield_phi(const double u[3], double L, int ws, double a[3]);
void orc_farfield_local(int64_t n, const float *pos, const float *mass, double L, int ws,
                        int order, int bg, double *Lambda);
void orc_farfield_eval(const double *Lambda, int order, double L, int64_t nsink, const float *pos,
                       const int64_t *sink, double *acc, double *pot);

/* O9 (orc_kdk.c) */
void orc_kdk_factors(int periodic, double mtot, double box, double a, double da, double *k1,
                     double *drift, double *k2);
void orc_kdk_factors_friedmann(double mtot, double box, double omega_m, double omega_l, double a,
                               double da, double *k1, double *drift, double *k2);
#endif
