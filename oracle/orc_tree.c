/* orc_tree.c — ORACLE (test infrastructure): Morton keys, stable sort, canonical octree, sink groups.
 * Follows SURVEY.md §8(c) O1, O2, O3, O5 (readings of PAPER.md:61 "assign a Key to each particle,
 * based on Morton ordering ... implicitly defines the topology of the tree", PAPER.md:69-73 grouping).
 * Shares nothing with the CUDA path.  Compile with -ffp-contract=off (the fp32 steps are exact IEEE).
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---- multi-index helpers ---------------------------------------------------------------- */
int orc_midx(int a, int b, int c)
{
    int l = a + b + c, k = b + c;
    return l * (l + 1) * (l + 2) / 6 + k * (k + 1) / 2 + c;
}

void orc_mtable(int pmax, int *ea, int *eb, int *ec)
{
    for (int l = 0; l <= pmax; l++)
        for (int a = l; a >= 0; a--)
            for (int b = l - a; b >= 0; b--) {
                int c = l - a - b, i = orc_midx(a, b, c);
                ea[i] = a; eb[i] = b; ec[i] = c;
            }
}

/* ---- O1 keys ---------------------------------------------------------------------------- */
/* returns 0 ok, -4 out of box (isolated), -5 non-finite.  `wrapped` (may be NULL) receives the
 * positions actually keyed: the input when isolated, the fp32-wrapped ones when periodic. */
int orc_keys(int64_t n, const float *pos, float box, int periodic, uint64_t *key, float *wrapped)
{
    volatile float scale = 2097152.0f / box;        /* 2^21 / box, one fp32 division           */
    for (int64_t i = 0; i < n; i++) {
        uint32_t q[3];
        for (int d = 0; d < 3; d++) {
            volatile float x = pos[3 * i + d];
            if (!isfinite(x)) return -5;
            if (periodic) {
                volatile float t = x / box;         /* fp32 division                           */
                volatile float f = floorf(t);
                volatile float prod = box * f;      /* fp32 multiply, then a separate subtract */
                volatile float w = x - prod;
                if (!(w >= 0.0f && w < box)) w = 0.0f;
                x = w;
            } else if (!(x >= 0.0f && x < box)) return -4;
            if (wrapped) wrapped[3 * i + d] = x;
            volatile float xs = x * scale;          /* THE fp32 multiply of reading A3         */
            float fl = floorf(xs);
            uint32_t qi = (uint32_t)fl;
            if (qi > 2097151u) qi = 2097151u;
            q[d] = qi;
        }
        uint64_t k = 0;
        for (int b = 0; b < ORC_KEY_LEVELS; b++) {  /* x is the most significant bit of a triple */
            k |= (uint64_t)((q[0] >> b) & 1u) << (3 * b + 2);
            k |= (uint64_t)((q[1] >> b) & 1u) << (3 * b + 1);
            k |= (uint64_t)((q[2] >> b) & 1u) << (3 * b + 0);
        }
        key[i] = k | (1ull << 63);                  /* HOT placeholder bit                     */
    }
    return 0;
}

/* ---- O2 stable sort --------------------------------------------------------------------- */
typedef struct { uint64_t k; uint32_t i; } kv_t;
static int kv_cmp(const void *a, const void *b)
{
    const kv_t *x = a, *y = b;
    if (x->k != y->k) return x->k < y->k ? -1 : 1;
    return x->i < y->i ? -1 : (x->i > y->i);       /* ties: original index ascending (A4)     */
}

void orc_sort(int64_t n, const uint64_t *key, uint64_t *skey, uint32_t *order)
{
    kv_t *kv = malloc(sizeof(kv_t) * (size_t)(n > 0 ? n : 1));
    for (int64_t i = 0; i < n; i++) { kv[i].k = key[i]; kv[i].i = (uint32_t)i; }
    qsort(kv, (size_t)n, sizeof(kv_t), kv_cmp);
    for (int64_t i = 0; i < n; i++) { skey[i] = kv[i].k; order[i] = kv[i].i; }
    free(kv);
}

/* ---- O3 canonical octree ---------------------------------------------------------------- */
static void cells_reserve(orc_tree *t, int64_t *cap, int64_t need)
{
    if (need <= *cap) return;
    int64_t c = *cap * 2; if (c < need) c = need;
    t->hotkey = realloc(t->hotkey, sizeof(uint64_t) * c);
    t->first = realloc(t->first, sizeof(int64_t) * c);
    t->count = realloc(t->count, sizeof(int64_t) * c);
    t->child0 = realloc(t->child0, sizeof(int64_t) * c);
    t->nchild = realloc(t->nchild, sizeof(int32_t) * c);
    t->level = realloc(t->level, sizeof(int32_t) * c);
    *cap = c;
}

/* geometry from the hotkey alone (O3): side = box 2^-l, centre = corner + side/2 */
void orc_cell_geometry(const orc_tree *t, int64_t c, double *side, double centre[3])
{
    int l = t->level[c];
    uint64_t prefix = t->hotkey[c] & ~(1ull << (3 * l));
    uint32_t q[3] = {0, 0, 0};
    for (int b = 0; b < l; b++) {
        q[0] |= (uint32_t)((prefix >> (3 * b + 2)) & 1u) << b;
        q[1] |= (uint32_t)((prefix >> (3 * b + 1)) & 1u) << b;
        q[2] |= (uint32_t)((prefix >> (3 * b + 0)) & 1u) << b;
    }
    double s = (double)t->box * ldexp(1.0, -l);
    *side = s;
    for (int d = 0; d < 3; d++) centre[d] = s * (double)q[d] + 0.5 * s;
}

/* integer coordinates of cell c at its own level (de-interleaved hotkey prefix) */
void orc_cell_coords(const orc_tree *t, int64_t c, int64_t q[3])
{
    int l = t->level[c];
    uint64_t prefix = t->hotkey[c] & ~(1ull << (3 * l));
    q[0] = q[1] = q[2] = 0;
    for (int b = 0; b < l; b++) {
        q[0] |= (int64_t)((prefix >> (3 * b + 2)) & 1u) << b;
        q[1] |= (int64_t)((prefix >> (3 * b + 1)) & 1u) << b;
        q[2] |= (int64_t)((prefix >> (3 * b + 0)) & 1u) << b;
    }
}

static void build_groups_rec(orc_tree *t, int64_t c, int64_t *cap)
{
    if (t->count[c] <= t->ncrit || t->nchild[c] == 0) {
        /* first cell from the root with count <= NCRIT; an over-full level-21 leaf is cut into
         * consecutive chunks of NCRIT (O5) */
        int64_t f = t->first[c], left = t->count[c];
        while (left > 0) {
            int64_t m = left < t->ncrit ? left : t->ncrit;
            if (t->ngroup == *cap) {
                *cap *= 2;
                t->gcell = realloc(t->gcell, sizeof(int64_t) * *cap);
                t->gfirst = realloc(t->gfirst, sizeof(int64_t) * *cap);
                t->gcount = realloc(t->gcount, sizeof(int64_t) * *cap);
                t->gbox = realloc(t->gbox, sizeof(float) * 6 * *cap);
            }
            int64_t g = t->ngroup++;
            t->gcell[g] = c; t->gfirst[g] = f; t->gcount[g] = m;
            float *bb = t->gbox + 6 * g;
            for (int d = 0; d < 3; d++) { bb[d] = INFINITY; bb[3 + d] = -INFINITY; }
            for (int64_t r = f; r < f + m; r++)
                for (int d = 0; d < 3; d++) {
                    float x = t->pos[3 * (int64_t)t->order[r] + d];
                    if (x < bb[d]) bb[d] = x;
                    if (x > bb[3 + d]) bb[3 + d] = x;
                }
            f += m; left -= m;
        }
        return;
    }
    for (int k = 0; k < t->nchild[c]; k++) build_groups_rec(t, t->child0[c] + k, cap);
}

orc_tree *orc_tree_build(int64_t n, const float *pos, const float *mass, float box, int periodic,
                         int nleaf, int ncrit, int *err)
{
    orc_tree *t = calloc(1, sizeof(orc_tree));
    t->n = n; t->box = box; t->periodic = periodic; t->nleaf = nleaf; t->ncrit = ncrit; t->p = -1;
    size_t m = (size_t)(n > 0 ? n : 1);
    t->pos = malloc(sizeof(float) * 3 * m);
    t->mass = malloc(sizeof(float) * m);
    t->key = malloc(sizeof(uint64_t) * m);
    t->skey = malloc(sizeof(uint64_t) * m);
    t->order = malloc(sizeof(uint32_t) * m);
    t->rank_of = malloc(sizeof(int64_t) * m);
    t->spos = malloc(sizeof(double) * 3 * m);
    t->smass = malloc(sizeof(double) * m);
    memcpy(t->mass, mass, sizeof(float) * (size_t)n);
    int e = orc_keys(n, pos, box, periodic, t->key, t->pos);
    if (err) *err = e;
    if (e) { orc_tree_free(t); return NULL; }
    orc_sort(n, t->key, t->skey, t->order);
    for (int64_t r = 0; r < n; r++) {
        int64_t i = t->order[r];
        t->rank_of[i] = r;
        for (int d = 0; d < 3; d++) t->spos[3 * r + d] = (double)t->pos[3 * i + d];
        t->smass[r] = (double)t->mass[i];
    }
    /* breadth-first build: the queue order is level-major, then parent order, then octant,
     * which is ascending hotkey (the placeholder bit encodes the level) */
    int64_t cap = 0;
    cells_reserve(t, &cap, 1024);
    t->ncell = 1;
    t->hotkey[0] = 1; t->first[0] = 0; t->count[0] = n; t->level[0] = 0; t->nchild[0] = 0; t->child0[0] = -1;
    for (int64_t c = 0; c < t->ncell; c++) {
        int l = t->level[c];
        t->nchild[c] = 0; t->child0[c] = -1;
        if (!(t->count[c] > nleaf && l < ORC_KEY_LEVELS)) continue;       /* leaf */
        int shift = 3 * (ORC_KEY_LEVELS - (l + 1));
        int64_t r = t->first[c], end = t->first[c] + t->count[c];
        while (r < end) {
            uint64_t hk = t->skey[r] >> shift;                            /* child hotkey     */
            int64_t r2 = r;
            while (r2 < end && (t->skey[r2] >> shift) == hk) r2++;
            cells_reserve(t, &cap, t->ncell + 1);
            int64_t ch = t->ncell++;
            if (t->nchild[c] == 0) t->child0[c] = ch;
            t->nchild[c]++;
            t->hotkey[ch] = hk; t->first[ch] = r; t->count[ch] = r2 - r; t->level[ch] = l + 1;
            t->nchild[ch] = 0; t->child0[ch] = -1;
            r = r2;
        }
    }
    /* groups */
    int64_t gcap = 1024;
    t->gcell = malloc(sizeof(int64_t) * gcap);
    t->gfirst = malloc(sizeof(int64_t) * gcap);
    t->gcount = malloc(sizeof(int64_t) * gcap);
    t->gbox = malloc(sizeof(float) * 6 * gcap);
    t->ngroup = 0;
    if (n > 0) build_groups_rec(t, 0, &gcap);
    return t;
}

void orc_tree_free(orc_tree *t)
{
    if (!t) return;
    free(t->pos); free(t->mass); free(t->key); free(t->skey); free(t->order); free(t->rank_of);
    free(t->spos); free(t->smass);
    free(t->hotkey); free(t->first); free(t->count); free(t->child0); free(t->nchild); free(t->level);
    free(t->gcell); free(t->gfirst); free(t->gcount); free(t->gbox);
    free(t->cmass); free(t->com); free(t->delta); free(t->mom); free(t->mom_bg);
    free(t);
}

/* ---- flat accessors for ctypes ---------------------------------------------------------- */
int64_t orc_tree_ncell(const orc_tree *t) { return t->ncell; }
int64_t orc_tree_ngroup(const orc_tree *t) { return t->ngroup; }
void orc_tree_get_sorted(const orc_tree *t, uint64_t *skey, uint32_t *order)
{
    memcpy(skey, t->skey, sizeof(uint64_t) * (size_t)t->n);
    memcpy(order, t->order, sizeof(uint32_t) * (size_t)t->n);
}
void orc_tree_get_cells(const orc_tree *t, uint64_t *hotkey, int64_t *first, int64_t *count,
                        int32_t *nchild, int64_t *child0, int32_t *level)
{
    for (int64_t c = 0; c < t->ncell; c++) {
        hotkey[c] = t->hotkey[c]; first[c] = t->first[c]; count[c] = t->count[c];
        nchild[c] = t->nchild[c]; child0[c] = t->child0[c]; level[c] = t->level[c];
    }
}
void orc_tree_get_groups(const orc_tree *t, int64_t *gcell, int64_t *gfirst, int64_t *gcount,
                         float *gbox)
{
    for (int64_t g = 0; g < t->ngroup; g++) {
        gcell[g] = t->gcell[g]; gfirst[g] = t->gfirst[g]; gcount[g] = t->gcount[g];
        for (int d = 0; d < 6; d++) gbox[6 * g + d] = t->gbox[6 * g + d];
    }
}
void orc_tree_get_wrapped(const orc_tree *t, float *pos)
{
    memcpy(pos, t->pos, sizeof(float) * 3 * (size_t)t->n);
}
