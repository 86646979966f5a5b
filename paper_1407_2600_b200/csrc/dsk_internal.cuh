// dsk_internal.cuh — context, workspace layout and small device helpers shared by the CUDA sources of
// libdsk (sm_100a).  Nothing here is shared with the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/dsk.h"

#define DSK_KEY_LEVELS 21
#ifndef DSK_NLEAF
#define DSK_NLEAF 112        // leaf bucket: a cell is split iff count > NLEAF (the oracle's NLEAF must match; sweep)
#endif
#ifndef DSK_NCRIT
#define DSK_NCRIT 192        // sink group: first cell from the root with count <= NCRIT (at most 4 tasks of 32 lanes x 2 sinks)
#endif
#define DSK_RETRY_WALK 1000            // internal: a predicted list slot overflowed (force.cu -> dsk_api.cu): evaluate again with COUNT + FILL
#define DSK_SORT_TILE 2048               // keys per block and pass of the radix sort (keysort.cu)
#define DSK_SORT_ONESWEEP_NMAX (1 << 22) // up to here the sort takes its one-kernel-per-pass form (keysort.cu): sizes its status words
#define DSK_WS 2              // LARGEST image block half-width, and the one image ids are encoded for: id = ((ix+2) 5 + iy+2) 5 + iz+2.
                              // The block actually summed is the context's ws (1 or 2, dsk_set_image_block): ids with |i| <= ws.
#define DSK_WS_DEFAULT 1      // with background subtraction WS = 1 costs 1e-4 of the rms force on a near-lattice box and saves 11-18 %
#define DSK_FAR_ORDER 8
#define DSK_NFAR 165          // C(8+3,3)
#define DSK_PMAX 8
#define DSK_RMAX 8            // deepest rung of the block time steps: 256 substeps per block step
#define DSK_IMG_BITS 7        // list entry = image << 25 | cell ... see below
#define DSK_CELL_BITS 25
#define DSK_FRTAB_BEG 320     // >= fr_nc(8) + 1 = 293
#define DSK_FRTAB_ENT 768     // >= 739 map entries at p = 8
// A list entry packs (image id, cell id).  With WS = 2 there are 125 images (7 bits) which leaves
// 25 bits = 33.5 M cells per tree; larger trees use WS-image ids only in periodic mode, so isolated
// runs could use all 32 bits — kept uniform for simplicity (N <= ~1.3e8 at ~0.25 cells/particle).

__host__ __device__ constexpr int dsk_np(int p) { return (p + 1) * (p + 2) * (p + 3) / 6; }
__host__ __device__ constexpr int dsk_midx(int a, int b, int c)
{
    return (a + b + c) * (a + b + c + 1) * (a + b + c + 2) / 6 + (b + c) * (b + c + 1) / 2 + c;
}
// moment row (floats): [ctr.x ctr.y ctr.z 1/s | off.x off.y off.z delta | Mhat_0 .. Mhat_{Np-1} | pad]
// ctr = geometric cell centre (exact), off = com - ctr, Mhat_n = (-1)^|n| M_n / (n! s^|n|)
__host__ __device__ constexpr int dsk_rowlen(int p) { return ((8 + dsk_np(p)) + 3) / 4 * 4; }

// Force tasks (force_task.cuh): two sinks per lane, so a group of n <= NCRIT sinks is L = ceil(n/2) sink lanes wide.
// A task (warp) takes w <= 32 of them and runs S = 32 / w sub-groups over alternate list entries; per list
// entry it costs one body pass per S entries plus a fixed share of the tile staging.  The group is cut into at
// most 4 tasks of widths w_1 + .. + w_k = L that minimise  sum_i (1/S_i + c)  (exact, by dynamic programming at
// compile time; c = 40/960 from the measured ~240 staging instructions per 32-entry tile against 185 per body
// pass).  Unequal widths matter: L = 33 is (1, 32), 33/32 of a pass per entry, where four equal parts cost 4/3.
#define DSK_LMAX ((DSK_NCRIT + 1) / 2)
#ifndef DSK_PART_COST
#define DSK_PART_COST 40       // c in units of 1/960 of a body pass
#endif
static_assert(DSK_LMAX <= 128, "a group must fit 4 tasks of 32 sink lanes");
struct dsk_parts_tab { uint32_t w[DSK_LMAX + 1]; };      // widths of the parts of L sink lanes, one byte each
constexpr dsk_parts_tab dsk_make_parts_tab()
{
    dsk_parts_tab t{};
    const int INF = 1 << 28;
    int best[5][DSK_LMAX + 1] = {}, pick[5][DSK_LMAX + 1] = {};
    for (int L = 0; L <= DSK_LMAX; L++) best[0][L] = L ? INF : 0;
    for (int k = 1; k <= 4; k++)
        for (int L = 0; L <= DSK_LMAX; L++) {
            best[k][L] = best[k - 1][L];                 // pick 0: fewer parts do as well
            pick[k][L] = 0;
            for (int w = 1; w <= 32 && w <= L; w++) {
                const int v = 960 / (32 / w) + DSK_PART_COST + best[k - 1][L - w];
                if (v < best[k][L]) { best[k][L] = v; pick[k][L] = w; }
            }
        }
    for (int L = 0; L <= DSK_LMAX; L++) {
        uint32_t word = 0;
        int k = 4, rem = L, n = 0;
        while (rem > 0) {
            const int w = pick[k][rem];
            k--;
            if (w == 0) continue;
            word |= (uint32_t)w << (8 * n);
            n++;
            rem -= w;
        }
        t.w[L] = word;
    }
    return t;
}
static __device__ const dsk_parts_tab dsk_parts_dev = dsk_make_parts_tab();
// number of tasks of a group of n sinks, and the sink range [off, off + ns) of part `part`
__device__ __forceinline__ uint32_t dsk_task_parts(uint32_t n)
{
    const uint32_t word = dsk_parts_dev.w[(n + 1u) >> 1];
    return (word != 0u) + ((word >> 8) != 0u) + ((word >> 16) != 0u) + ((word >> 24) != 0u);
}
__device__ __forceinline__ void dsk_task_range(uint32_t n, uint32_t part, uint32_t &off, uint32_t &ns)
{
    const uint32_t word = dsk_parts_dev.w[(n + 1u) >> 1];
    const uint32_t before = word & ((1u << (8u * part)) - 1u);            // widths of the parts before this one
    const uint32_t lanes = (before & 255u) + ((before >> 8) & 255u) + ((before >> 16) & 255u);
    off = 2u * lanes;
    ns = min(2u * ((word >> (8u * part)) & 255u), n - off);
}

struct dsk_cellrec {          // 16 B, one LDG.128 in the walk
    uint32_t first, count, child0, meta;   // meta = nchild | level << 8
};

struct dsk_devstate {         // small device block read back at the end of API calls
    uint32_t status;          // bit flags: 1 out-of-box, 2 non-finite, 4 cell overflow, 8 stack overflow,
                              //            16 list overflow
    uint32_t ncell, ngroup, nlevel;
    uint32_t ntask;           // warp tasks = sum over groups of dsk_task_parts(count)
    uint32_t lvl_start[DSK_KEY_LEVELS + 3];
    uint32_t nleaf_cells;
    unsigned long long tot_m2p_list, tot_p2p_list, tot_p2p_src;   // over all groups
    unsigned long long n_p2p, n_m2p;                               // useful interactions
    unsigned long long scratch[4];
    unsigned long long tot_left_list;                              // cubes kept outside the windows (background.cu), all groups
};

enum { ST_OUTOFBOX = 1, ST_NONFINITE = 2, ST_CELLOVF = 4, ST_STACKOVF = 8, ST_LISTOVF = 16 };

struct dsk_ctx {
    int64_t N;
    float box;
    int periodic;
    float eps, theta;
    int p;
    cudaStream_t stream;
    // workspace
    char *ws;
    size_t ws_bytes;
    // carved arrays
    uint64_t *key_a, *key_b;
    uint32_t *idx_a, *idx_b;
    uint32_t *sort_hist;      // [ntile * 256] per-pass tile histograms (digit-major); small N: histograms, tickets and look-back status words (keysort.cu)
    uint32_t *scan_tmp;       // block sums for the generic scan
    float4 *spos;             // sorted (x,y,z,m); periodic: wrapped
    float4 *sacc;             // sorted (ax,ay,az,pot), high part of the compensated sum
    float4 *sacc_lo;          // low part (two-float accumulators across tiles, kernels and the far field)
    uint64_t *hotkey;
    dsk_cellrec *cell;
    uint32_t *parent;
    uint32_t *nchild_tmp;
    uint32_t *cbounds;        // [8 * ncell_cap] first rank of each octant of a cell being split (tree.cu)
    float4 *whdr;             // walk header per cell: com.xyz, delta
    float4 *wmac;             // what the MAC reads: com.xyz, s/theta + delta (walk.cu, per theta)
    float *rows;              // [ncell_cap * rowlen(p_cap)] moment rows (upward.cu)
    float *frows;             // [ncell_cap * frow_len(p_cap)] force rows read by M2P (m2p.cu)
    uint32_t *frtab_beg;      // [DSK_FRTAB_BEG] moment row -> force row map of the current p
    void *frtab_ent;          // [DSK_FRTAB_ENT] {src, weight}
    uint32_t *gmark;          // [N] group start markers (cell id + 1)
    uint32_t *gscan;          // [N]
    uint32_t *gfirst, *gcount, *gcell;     // [ngroup_cap]
    float4 *gbox;             // [2 * ngroup_cap]: min.xyz,_ ; max.xyz,_
    uint32_t *g_m2p_len, *g_p2p_len, *g_p2p_src;   // [ngroup_cap]
    uint32_t *g_taskoff;      // [ngroup_cap + 1] exclusive scan of dsk_task_parts(count)
    uint32_t *g_task;         // [4 * ngroup_cap] task -> group << 2 | part
    uint8_t *gact;            // [ngroup_cap] group holds an active sink (dsk_accel_active)
    const uint8_t *gact_cur;  // gact during an active-subset evaluation, else nullptr
    uint32_t *g_task_sorted;  // [4 * ngroup_cap] the tasks of the current batch, longest first (m2p.cu)
    uint32_t *task_hist;      // [1024] counting-sort bins
    uint64_t *g_m2p_off, *g_p2p_off;               // [ngroup_cap + 1] exclusive offsets into lists
    uint32_t *list_m2p, *list_p2p;
    size_t list_m2p_cap, list_p2p_cap;             // entries
    // background subtraction (background.cu; periodic contexts only)
    int img_ws;               // image block half-width in use, 1 or 2 (dsk_set_image_block)
    int bg;                   // on / off (dsk_set_background)
    int bg_level;             // l_b
    uint32_t ntop;            // cells of level <= l_b of the current tree
    int64_t ntop_cap;
    int4 *topgeo;             // [ntop_cap] integer coordinates, level | child octant mask << 8
    double *mass64;           // [ntop_cap] fp64 masses
    float *kbg;               // [ntop_cap] error-bound constants of the subtracted copies (absolute-error MAC, walk.cu)
    float *rows_bg;           // [ntop_cap * rowlen(p_cap)] subtracted moment rows (their force rows are frows[ncell ..])
    uint32_t *g_left_len;     // [ngroup_cap] cubes kept outside the window, per group (the walk's third list)
    uint64_t *g_left_off;     // [ngroup_cap + 1]
    uint4 *list_left;         // records: lo | hi << 16 per axis (int16 each), level-l_b cells
    size_t list_left_cap;
    float *kdk_acc;           // [N,3] cached force, caller order
    uint8_t *kdk_active;      // [N] particles whose step ends at the current substep (dsk_kdk_block_step)
    double *far_partial;      // [nblk * 165]
    double *far_M;            // [165]
    double *far_lambda;       // [165]
    double *far_T_dev;        // [165]
    dsk_devstate *dstate;     // device
    dsk_devstate *hstate;     // pinned host
    // sizes
    int64_t ncell_cap, ngroup_cap;
    int ntile;
    // state
    int have_tree, moments_p, lists_valid, kdk_have_acc;
    double omega_m, omega_l;  // background cosmology of dsk_kdk_step (default 1, 0)
    int p_cap;                // order the workspace was sized for (dsk_create's p); set_params may lower p
    int frow_tab_p;           // order of the uploaded force-row map
    int frow_tab_dip;         // and whether it has the dipole block
    int frow_dip;             // layout of the force rows in memory: dipole block present (periodic with subtraction)
    uint32_t m2m_tab_mask;    // orders whose M2M pair table this context has uploaded (bit p - 2)
    int soft_kind;            // 0 Plummer (eps), 1 Dehnen K1 (eps holds the support h) (dsk_set_softening)
    int mac_kind;             // 0 opening angle, 1 absolute error bound (dsk_set_mac)
    float mac_tol;
    float lists_theta;
    int walk_two_pass_only;   // dsk_set_walk_mode(1)
    int bg_closed;            // dsk_set_background(2): the windows' background by the closed form everywhere (diagnostic)
    uint64_t *pg_key;         // [ngroup_cap] previous evaluation's groups: start of the Morton-key interval of the group's cell (walk.cu)
    uint32_t *pg_m2p, *pg_p2p, *pg_left;      // ... and their list lengths
    uint32_t pg_n;
    int pg_valid;             // the remembered lengths belong to this context's current parameters
    int64_t pg_retries;       // evaluations that started over because a predicted slot overflowed (dsk_get_walk_info)
    int pg_backoff, pg_wait;  // after an overflow: evaluations to sit out before predicting again (1, 3, 7, 15; 0 after a success)
    int walk_predicted;       // the offsets of the current evaluation are scanned PREDICTED capacities: fill with MODE 3, check the overflow flag
    int walk_share;           // dsk_set_walk_sharing: groups per shared walk (0 = automatic)
    int walk_onepass;         // the lists of the current evaluation were written by the one-pass walk
    float onepass_bad_theta;  // theta at which a list overflowed its fixed capacity (skip the one-pass attempt)
    double far_T[DSK_NFAR];
    dsk_stats stats;
    int pending_build_ms, pending_force_ms;   // event times not read yet: 1 = the stream has to be synchronised first (dsk_get_stats, end of dsk_accel)
    cudaEvent_t ev[20];
    int nsm;
};

#define DSK_COUNT(c, k) ((c)->stats.n_launch += (k))
// Constant tables and function attributes are per device: a "done once" flag is kept per device ordinal (a process
// normally drives one GPU, but two contexts on two devices must both get their tables).
#define DSK_MAXDEV 64
static inline bool *dsk_device_flag(bool *flags)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= DSK_MAXDEV) dev = 0;
    return flags + dev;
}
#define DSK_CUDA(x)                                 \
    do {                                            \
        cudaError_t e__ = (x);                      \
        if (e__ != cudaSuccess) return DSK_ECUDA;   \
    } while (0)

// ---- internal entry points (one per source file) -------------------------------------------------
int dsk_run_keysort(dsk_ctx *c, const float *pos, const float *mass);         // keysort.cu: K, S, gather
int dsk_run_scatter(dsk_ctx *c, float *acc, float *pot, const uint8_t *active, uint32_t r_lo, uint32_t r_hi);   // keysort.cu: X
int dsk_run_group_active(dsk_ctx *c, const uint8_t *active);                  // keysort.cu
void dsk_exclusive_scan_u32(dsk_ctx *c, const uint32_t *in, uint32_t *out, const uint32_t *n_dev,
                            uint32_t n_max, uint32_t *total_dev);             // keysort.cu
int dsk_run_build(dsk_ctx *c);                                                // tree.cu: T, G
int dsk_run_upward(dsk_ctx *c);                                               // upward.cu: U
int dsk_run_get_moments(dsk_ctx *c, float *com_mass, float *moments, int scaled);         // upward.cu
int dsk_walk_remember(dsk_ctx *c);                                           // walk.cu: list lengths for the next evaluation
int dsk_run_walk(dsk_ctx *c);                                                 // walk.cu: W
int dsk_run_shard(dsk_ctx *c, int rank, int nranks, uint32_t flop_m2p, uint32_t flop_p2p, uint32_t *cut_host);   // walk.cu
int dsk_run_force(dsk_ctx *c, int want_pot);                                  // force.cu: F1 + orchestration
int dsk_frow_len(int p, int dip);                                             // m2p.cu
int dsk_run_frows(dsk_ctx *c);                                                // m2p.cu: moment rows -> force rows
int dsk_run_frows_bg(dsk_ctx *c, uint32_t ntop);                              // m2p.cu: subtracted rows -> force rows [ncell ..]
int dsk_bg_level(int64_t n);                                                  // background.cu
int dsk_bg_halfwidth(float theta, int lb, int ws);                            // background.cu
int dsk_run_bg_rows(dsk_ctx *c);                                              // background.cu: after the upward pass
int dsk_run_bg_window(dsk_ctx *c, int want_pot);                              // background.cu: after all batches
int dsk_run_bg_left(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t base, int want_pot);   // background.cu: per batch
int dsk_run_get_bg_moments(dsk_ctx *c, float *moments);                       // background.cu
int dsk_order_tasks(dsk_ctx *c, uint32_t t0, uint32_t t1, const uint32_t *len, int shift);   // m2p.cu
int dsk_launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot);   // m2p.cu: F2
int dsk_run_farfield(dsk_ctx *c);                                             // farfield.cu: F3
void dsk_lattice_tensors(double L, int ws, double *T);                        // farfield.cu (host)
int dsk_run_kick(dsk_ctx *c, float *vel, const float *acc, float k);          // kdk.cu
int dsk_run_drift(dsk_ctx *c, float *pos, const float *vel, float d);         // kdk.cu
int dsk_run_kick_rung(dsk_ctx *c, float *vel, const float *acc, const uint8_t *rung, uint32_t s, uint32_t nsub,
                      int rmax, const float *k);                              // kdk.cu
int dsk_run_rung_active(dsk_ctx *c, const uint8_t *rung, uint32_t t, uint32_t nsub, int rmax, uint8_t *active);   // kdk.cu
int dsk_run_rung_update(dsk_ctx *c, const float *acc, const uint8_t *active, uint8_t *rung, uint32_t t, uint32_t nsub,
                        int rmax, float da, float eta);                       // kdk.cu

// ---- packed f32x2 arithmetic (sm_100a: FFMA2 / FADD2 / FMUL2) ----------------------------------
// One 64-bit register pair carries two independent fp32 lanes.  Measured on B200: scalar FFMA with
// three distinct source registers tops out at ~46 TFLOP/s (register-bank limited), FFMA2 reaches the
// 74 TFLOP/s nominal peak — so the force kernels run two sources per thread in packed form.
#ifdef __CUDACC__
struct f2 {
    unsigned long long v;
};
__device__ __forceinline__ f2 f2_make(float lo, float hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 f2_dup(float x) { return f2_make(x, x); }
__device__ __forceinline__ float f2_lo(f2 a) { return __uint_as_float((unsigned int)(a.v & 0xffffffffull)); }
__device__ __forceinline__ float f2_hi(f2 a) { return __uint_as_float((unsigned int)(a.v >> 32)); }
__device__ __forceinline__ f2 f2_fma(f2 a, f2 b, f2 c)
{
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ f2 f2_mul(f2 a, f2 b)
{
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 f2_add(f2 a, f2 b)
{
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 f2_sub(f2 a, f2 b)
{
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 f2_rsqrt(f2 a)
{
    return f2_make(rsqrtf(f2_lo(a)), rsqrtf(f2_hi(a)));
}
#endif

#ifdef __CUDACC__
// two-float accumulation: (hi, lo) += t without losing the rounding error of the addition (TwoSum)
__device__ __forceinline__ void dsk_fold(float &hi, float &lo, float t)
{
    const float s = hi + t;
    const float bb = s - hi;
    lo += (hi - (s - bb)) + (t - bb);
    hi = s;
}
#endif
