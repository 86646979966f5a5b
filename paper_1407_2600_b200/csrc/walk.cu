// walk.cu — step W: warp-cooperative group tree walk under the opening-angle MAC.
// DESIGN.md O5 ("this tree is traversed": the sinks of one sink cell share
// the list of source cells; near the leaves the rest is done with direct interactions).
//   accept cell c (image shift nL) for group g  iff  d^2 > (s_c/theta + delta_c)^2   (strict)
//   d = distance from com_c + nL to the AABB of g's members.
// accepted -> M2P list; rejected leaf -> P2P list; rejected internal -> children are visited.
// One warp per group, 64 cells tested per trip (two stack entries per lane) from a LIFO stack in shared memory (depth-first order
// keeps it short); list entries are compacted with ballots and written as contiguous runs.
// Run once into a fixed capacity per group when every list fits (the usual case), else twice: COUNT (list
// lengths, for the offsets) and FILL.
#include "dsk_internal.cuh"
#include <string.h>
#include <stdio.h>

// one warp per block: walks differ in length, and a block ends with its longest
#define WRESERVE 160         // stack entries kept free for the depth-first tail (7 per level, 21 levels)
#ifndef WEPL
#define WEPL 2               // stack entries per lane and trip
#endif
#ifndef WSTACK
#define WSTACK 2048          // stack entries per warp
#endif

// Image ids (the 5^3 encoding of the list entries) -> integer offsets: a 125-word table in shared memory, filled by each warp at
// the start of its kernel.  (Dividing the id by 5 and 25 for every tested cell, once for the shift and once for the window test,
// was 15 % of the walk's instructions: ncu, profiles/r02b_walk_ncu_full.md.)
#define WK_NIMG ((2 * DSK_WS + 1) * (2 * DSK_WS + 1) * (2 * DSK_WS + 1))
__device__ __forceinline__ void wk_img_table(uint32_t *tab, int lane)
{
    const int side = 2 * DSK_WS + 1;
    for (int i = lane; i < WK_NIMG; i += 32)
        tab[i] = (uint32_t)(i / (side * side)) | (uint32_t)((i / side) % side) << 8 | (uint32_t)(i % side) << 16;      // ix, iy, iz + DSK_WS
    __syncwarp();
}
__device__ __forceinline__ void wk_image(const uint32_t *tab, int img, int periodic, float box, float sh[3], int ish[3])
{
    if (!periodic) { sh[0] = sh[1] = sh[2] = 0.0f; ish[0] = ish[1] = ish[2] = 0; return; }
    const uint32_t w = tab[img];
    ish[0] = (int)(w & 255u) - DSK_WS; ish[1] = (int)((w >> 8) & 255u) - DSK_WS; ish[2] = (int)(w >> 16) - DSK_WS;
    sh[0] = ish[0] * box; sh[1] = ish[1] * box; sh[2] = ish[2] * box;
}

// Background subtraction (reading O4b of DESIGN.md, background.cu).  lb < 0: off.  The cells of level <= lb are the first
// ntop cells (canonical order is level-major); topgeo holds their integer coordinates, level and child-octant mask.
struct walk_bg {
    int lb, k;
    uint32_t ntop, ncell;
    const int4 *topgeo;
    const uint32_t *gcell;
    const uint64_t *hotkey;
    uint32_t *left_len;            // [ngroup] cubes kept outside the window (third list)
    const uint64_t *left_off;      // FILL: scanned offsets
    uint64_t left_base;
    uint4 *list_left;
    uint32_t cap_l;                // ONE pass: fixed capacity per group
    uint64_t *left_off_out;
    const float *kbg;              // [ntop] error-bound constant of the subtracted copies (absolute-error MAC)
};

__device__ __forceinline__ uint32_t wk_compact3(uint64_t x)
{
    x &= 0x1249249249249249ull;
    x = (x | x >> 2) & 0x10c30c30c30c30c3ull;
    x = (x | x >> 4) & 0x100f00f00f00f00full;
    x = (x | x >> 8) & 0x1f0000ff0000ffull;
    x = (x | x >> 16) & 0x1f00000000ffffull;
    x = (x | x >> 32) & 0x1fffffull;
    return (uint32_t)x;
}

// The cubes a rejected cell of level <= lb exposes (cubes of the image block whose background no accepted cell carries): the
// cell's own cube if it is a leaf or sits at level lb (below lb nothing carries a background), else its empty octants.  Those
// inside the window are part of the window's cuboid; the others are kept: returns their number and, with out != nullptr, writes
// their records (lo | hi << 16 per axis, int16 index ranges in level-lb cells).
__device__ __forceinline__ uint32_t wk_exposed(bool whole, int lvl, int lb, const int4 geo, const int ish[3], const int wlo[3],
                                               const int whi[3], uint4 *out)
{
    uint32_t n = 0;
    const int q[3] = {geo.x, geo.y, geo.z};
    if (whole) {
        int lo[3], hi[3];
        bool inside = true;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            lo[d] = (q[d] << (lb - lvl)) + (ish[d] << lb); hi[d] = lo[d] + (1 << (lb - lvl)) - 1;
            inside = inside && lo[d] >= wlo[d] && hi[d] <= whi[d];
        }
        if (!inside) {
            if (out) out[0] = make_uint4((uint32_t)(lo[0] & 0xffff) | (uint32_t)hi[0] << 16, (uint32_t)(lo[1] & 0xffff) | (uint32_t)hi[1] << 16,
                                         (uint32_t)(lo[2] & 0xffff) | (uint32_t)hi[2] << 16, 0u);
            n = 1;
        }
        return n;
    }
    const int mask = (geo.w >> 8) & 255, sh = lb - lvl - 1;
    for (int o = 0; o < 8; o++) {
        if (mask & (1 << o)) continue;
        const int bit[3] = {(o >> 2) & 1, (o >> 1) & 1, o & 1};
        int lo[3], hi[3];
        bool inside = true;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            lo[d] = ((2 * q[d] + bit[d]) << sh) + (ish[d] << lb); hi[d] = lo[d] + (1 << sh) - 1;
            inside = inside && lo[d] >= wlo[d] && hi[d] <= whi[d];
        }
        if (inside) continue;
        if (out) out[n] = make_uint4((uint32_t)(lo[0] & 0xffff) | (uint32_t)hi[0] << 16, (uint32_t)(lo[1] & 0xffff) | (uint32_t)hi[1] << 16,
                                     (uint32_t)(lo[2] & 0xffff) | (uint32_t)hi[2] << 16, 0u);
        n++;
    }
    return n;
}

// ABS: the absolute-error acceptance rule (reading O5b of DESIGN.md) instead of the opening angle: accept iff
//   d^2 > (s + delta)^2   (theta = 1: the expansion converges)   and   (d/b)^(p+1) (d - b)^2 >= kappa_c,
// b = sqrt(3)/2 s + delta, kappa_c = (p + 2) Q_c / (tol b^2), i.e. E_c(d) = (p+2) Q b^(p-1) / (d^(p+1) (d-b)^2) <= tol.
// The MAC record then holds s + delta in .w and kappa_c in the slot of `first` (which the walk does not use).
// Every step below is monotone in d2 under IEEE rounding (the shared walk relies on it: what the union of several groups'
// boxes accepts, each of them accepts).
template <bool ABS>
__device__ __forceinline__ bool wk_ok(float d2, float crit, uint32_t meta, float kappa, float box, int pow1, float k1_h)
{
    bool ok = d2 > crit * crit;
    if (ABS && ok) {
        const float s = box * exp2f(-(float)((meta >> 8) & 255u));
        const float b = crit - 0.1339746f * s, d = sqrtf(d2), x = d / b;
        float xp = x;
        for (int k = 1; k < pow1; k++) xp *= x;
        ok = xp * (d - b) * (d - b) >= kappa && d > b + k1_h;      // k1_h = 0 unless K1 softening (O6b)
    }
    return ok;
}
__device__ __forceinline__ float wk_d2(float zx, float zy, float zz, const float lo[3], const float hi[3])
{
    const float dx = fmaxf(fmaxf(lo[0] - zx, zx - hi[0]), 0.0f);
    const float dy = fmaxf(fmaxf(lo[1] - zy, zy - hi[1]), 0.0f);
    const float dz = fmaxf(fmaxf(lo[2] - zz, zz - hi[2]), 0.0f);
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// THE LONE WALK: one warp per group.
#define WW 1                 // warps (groups) per block: walks differ in length, a block ends with its longest
template <int MODE, bool ABS>          // MODE 0 COUNT, 1 FILL at the scanned offsets, 2 ONE pass into a fixed capacity per group,
                                       // 3 ONE pass into PREDICTED capacities: the offsets are scanned capacities (dsk_run_walk), lengths are written
__global__ void __launch_bounds__(WW * 32) k_walk(uint32_t g0, uint32_t g1, int periodic, float box, int pow1, float k1_h,
                                                  const dsk_cellrec *__restrict__ cell,
                                                  const float4 *__restrict__ wmac,
                                                  const float4 *__restrict__ gbox,
                                                  const uint32_t *__restrict__ gcount,
                                                  uint32_t *__restrict__ m2p_len, uint32_t *__restrict__ p2p_len,
                                                  uint32_t *__restrict__ p2p_src,
                                                  const uint64_t *__restrict__ m2p_off,
                                                  const uint64_t *__restrict__ p2p_off, uint64_t m2p_base,
                                                  uint64_t p2p_base, uint32_t *__restrict__ list_m2p,
                                                  uint32_t *__restrict__ list_p2p, const uint8_t *__restrict__ gact,
                                                  uint32_t cap_m, uint32_t cap_p, uint64_t *__restrict__ m2p_off_out,
                                                  uint64_t *__restrict__ p2p_off_out, const walk_bg bg, dsk_devstate *st)
{
    constexpr bool FILL = MODE != 0;
    constexpr uint32_t CELL_MASK = (1u << DSK_CELL_BITS) - 1u;
    __shared__ uint32_t stack[WW][WSTACK];
    __shared__ uint32_t imgtabs[WW][WK_NIMG];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *imgtab = imgtabs[warp];
    const uint32_t g = g0 + blockIdx.x * WW + warp;
    if (g >= g1) return;
    const bool BG = bg.lb >= 0;
    if (gact && !gact[g]) {                          // no active sink in this group (dsk_accel_active): empty lists
        if (MODE != 1 && lane == 0) {
            m2p_len[g] = 0; p2p_len[g] = 0; p2p_src[g] = 0;
            if (BG) bg.left_len[g] = 0;
            if (MODE == 2) {
                m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p;
                if (BG) bg.left_off_out[g] = (uint64_t)g * bg.cap_l;
            }
        }
        return;
    }
    const float4 blo = gbox[2 * (size_t)g], bhi = gbox[2 * (size_t)g + 1];
    const float blo3[3] = {blo.x, blo.y, blo.z}, bhi3[3] = {bhi.x, bhi.y, bhi.z};
    // the group's window: the level-lb cells within k of the footprint of its cell (integer index range, unwrapped frame)
    int wlo[3] = {0, 0, 0}, whi[3] = {0, 0, 0};
    if (BG) {
        const uint32_t cg = bg.gcell[g];
        const int lg = (int)(cell[cg].meta >> 8);
        const uint64_t prefix = bg.hotkey[cg] & ~(1ull << (3 * lg));
        const int q[3] = {(int)wk_compact3(prefix >> 2), (int)wk_compact3(prefix >> 1), (int)wk_compact3(prefix)};
#pragma unroll
        for (int d = 0; d < 3; d++) {
            int flo, fhi;
            if (lg >= bg.lb) flo = fhi = q[d] >> (lg - bg.lb);
            else { flo = q[d] << (bg.lb - lg); fhi = flo + (1 << (bg.lb - lg)) - 1; }
            wlo[d] = flo - bg.k; whi[d] = fhi + bg.k;
        }
    }
    uint32_t *stk = stack[warp];
    if (periodic) wk_img_table(imgtab, lane);
    // root of every image of the block in use: periodic = the block's half-width ws (0 isolated); ids are those of the 5^3 encoding
    int sp = 0;
    {
        const int side = 2 * DSK_WS + 1, nid = periodic ? side * side * side : 1;
        for (int i0 = 0; i0 < nid; i0 += 32) {
            const int i = i0 + lane;
            bool in = i < nid;
            if (periodic && in) {
                const int iz = i % side - DSK_WS, iy = (i / side) % side - DSK_WS, ix = i / (side * side) - DSK_WS;
                in = abs(ix) <= periodic && abs(iy) <= periodic && abs(iz) <= periodic;
            }
            const uint32_t m = __ballot_sync(0xffffffffu, in);
            if (in) stk[sp + __popc(m & ((1u << lane) - 1u))] = (uint32_t)(periodic ? i : 0) << DSK_CELL_BITS;
            sp += __popc(m);
        }
    }
    __syncwarp();
    uint32_t nm = 0, np = 0, nsrc = 0, nl = 0;
    uint64_t mo = 0, po = 0, lo_ = 0;
    uint32_t lim_m = 0xffffffffu, lim_p = 0xffffffffu, lim_l = 0xffffffffu;          // what the group's list slots hold
    if (MODE == 1 || MODE == 3) { mo = m2p_off[g] - m2p_base; po = p2p_off[g] - p2p_base; if (BG) lo_ = bg.left_off[g] - bg.left_base; }
    if (MODE == 2) { mo = (uint64_t)g * cap_m; po = (uint64_t)g * cap_p; if (BG) lo_ = (uint64_t)g * bg.cap_l; lim_m = cap_m; lim_p = cap_p; lim_l = bg.cap_l; }
    if (MODE == 3) {
        lim_m = (uint32_t)(m2p_off[g + 1] - m2p_off[g]); lim_p = (uint32_t)(p2p_off[g + 1] - p2p_off[g]);
        if (BG) lim_l = (uint32_t)(bg.left_off[g + 1] - bg.left_off[g]);
    }
    const uint32_t lt = (1u << lane) - 1u;
    // WEPL stack entries per lane and trip: their loads are independent, so a trip exposes one L2 round trip for
    // 32 * WEPL cells
    while (sp > 0) {
        // A popped cell pushes at most 8 children (net +7), so a trip of `take` cells needs 7 * take free entries.  Trips
        // shrink as the stack fills and end as a plain depth-first walk (take = 1), whose height above its starting
        // point is at most 7 per level = 147 < WRESERVE: the stack cannot overflow on any tree of <= 21 levels.
        const int room = (WSTACK - WRESERVE - sp) / 7;
        int take = sp < 32 * WEPL ? sp : 32 * WEPL;
        take = min(take, max(room, 1));
        uint32_t e[WEPL], nchild[WEPL], child0[WEPL];
        bool act[WEPL], accept[WEPL], leaf[WEPL];
        float4 h[WEPL], rr[WEPL];
        int4 geo[WEPL];
#pragma unroll
        for (int q = 0; q < WEPL; q++) {
            act[q] = lane + 32 * q < take;
            e[q] = act[q] ? stk[sp - 1 - lane - 32 * q] : 0u;
        }
        sp -= take;
        __syncwarp();
#pragma unroll
        for (int q = 0; q < WEPL; q++)
            if (act[q]) {
                const uint32_t c = e[q] & CELL_MASK;
                h[q] = wmac[2 * (size_t)c];            // com.xyz, critical radius s/theta + delta
                rr[q] = wmac[2 * (size_t)c + 1];       // the cell record (same sector)
                if (BG && c < bg.ntop) geo[q] = bg.topgeo[c];
            }
        uint32_t push[WEPL], ptot = 0;
#pragma unroll
        for (int q = 0; q < WEPL; q++) {
            accept[q] = false; leaf[q] = false; nchild[q] = 0; child0[q] = 0;
            uint32_t cnt = 0, nexp = 0, entry = e[q];
            const uint32_t c = e[q] & CELL_MASK;
            const bool top = BG && act[q] && c < bg.ntop;
            int ish[3] = {0, 0, 0};
            bool whole = false, winside = false, winter = false;
            if (act[q]) {
                float sh[3];
                const int img = (int)(e[q] >> DSK_CELL_BITS);
                wk_image(imgtab, img, periodic, box, sh, ish);
                const float zx = h[q].x + sh[0], zy = h[q].y + sh[1], zz = h[q].z + sh[2];
                const float d2 = wk_d2(zx, zy, zz, blo3, bhi3);
                bool straddles = false;
                if (top) {
                    // where the cell's cube lies relative to the window (integers: both sides decide alike)
                    const int lvl = geo[q].w & 255;
                    const int qq[3] = {geo[q].x, geo[q].y, geo[q].z};
                    winside = true; winter = true;
#pragma unroll
                    for (int d = 0; d < 3; d++) {
                        const int lo = (qq[d] << (bg.lb - lvl)) + (ish[d] << bg.lb), hi = lo + (1 << (bg.lb - lvl)) - 1;
                        winside = winside && lo >= wlo[d] && hi <= whi[d];
                        winter = winter && lo <= whi[d] && hi >= wlo[d];
                    }
                    straddles = winter && !winside;      // partly inside the window: never accepted (its background would count twice)
                    if (!winter) entry = (e[q] & ~CELL_MASK) | (bg.ncell + c);      // outside: the background-subtracted copy
                }
                float kappa = 0.0f;
                if (ABS) kappa = (top && entry != e[q]) ? bg.kbg[c] : rr[q].x;      // the subtracted copy has its own bound
                const bool ok = wk_ok<ABS>(d2, h[q].w, __float_as_uint(rr[q].w), kappa, box, pow1, k1_h);
                accept[q] = !straddles && ok;
                if (!accept[q]) {
                    nchild[q] = __float_as_uint(rr[q].w) & 255u; child0[q] = __float_as_uint(rr[q].z); cnt = __float_as_uint(rr[q].y);
                    leaf[q] = nchild[q] == 0;
                    if (top) {
                        whole = leaf[q] || (geo[q].w & 255) == bg.lb;
                        // cubes this cell exposes outside the window: none if it lies inside; itself; all its empty octants if it lies outside;
                        // octant by octant only when it straddles the window's edge
                        nexp = winside ? 0u : whole ? 1u : !winter ? 8u - (uint32_t)__popc((geo[q].w >> 8) & 255)
                                                                   : wk_exposed(false, geo[q].w & 255, bg.lb, geo[q], ish, wlo, whi, nullptr);
                    }
                }
            }
            const uint32_t bm = __ballot_sync(0xffffffffu, accept[q]);
            const uint32_t bl = __ballot_sync(0xffffffffu, leaf[q]);
            if (FILL) {
                const uint32_t im = nm + __popc(bm & lt), ip = np + __popc(bl & lt);
                if (accept[q] && (MODE == 1 || im < lim_m)) list_m2p[mo + im] = entry;
                if (leaf[q] && (MODE == 1 || ip < lim_p)) list_p2p[po + ip] = e[q];
            }
            nm += __popc(bm); np += __popc(bl);
            if (leaf[q]) nsrc += cnt;
            if (BG && __any_sync(0xffffffffu, nexp != 0u)) {           // rare: cubes kept outside the window
                uint32_t x = nexp;
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                const uint32_t tot = __shfl_sync(0xffffffffu, x, 31), at = nl + x - nexp;
                if (FILL && nexp && (MODE == 1 || at + nexp <= lim_l))
                    wk_exposed(whole, geo[q].w & 255, bg.lb, geo[q], ish, wlo, whi, bg.list_left + lo_ + at);
                nl += tot;
            }
            push[q] = (act[q] && !accept[q]) ? nchild[q] : 0u;      // children of rejected internal cells
            ptot += push[q];
        }
        uint32_t x = ptot;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        const uint32_t tot = __shfl_sync(0xffffffffu, x, 31);
        if (sp + (int)tot > WSTACK) {
            if (lane == 0) atomicOr(&st->status, ST_STACKOVF);
            break;
        }
        uint32_t at = sp + x - ptot;
#pragma unroll
        for (int q = 0; q < WEPL; q++) {
            const uint32_t img = e[q] & ~CELL_MASK;
#pragma unroll
            for (uint32_t k = 0; k < 8; k++)
                if (k < push[q]) stk[at + k] = img | (child0[q] + k);
            at += push[q];
        }
        sp += (int)tot;
        __syncwarp();
    }
    for (int o = 16; o; o >>= 1) nsrc += __shfl_xor_sync(0xffffffffu, nsrc, o);
    if (lane == 0) {
        if (MODE != 1) {
            m2p_len[g] = nm; p2p_len[g] = np; p2p_src[g] = nsrc;
            if (BG) bg.left_len[g] = nl;
        }
        if (MODE == 2) {
            m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p;
            if (BG) bg.left_off_out[g] = (uint64_t)g * bg.cap_l;
        }
        if (MODE >= 2 && (nm > lim_m || np > lim_p || (BG && nl > lim_l)))      // a list did not fit: the host falls back to two passes
            atomicOr(&st->scratch[0], (nm > lim_m ? 1ull : 0ull) | (np > lim_p ? 2ull : 0ull) | (BG && nl > lim_l ? 4ull : 0ull));
        if (FILL) {
            const unsigned long long ns = gcount[g];
            atomicAdd(&st->n_m2p, ns * nm);
            atomicAdd(&st->n_p2p, ns * nsrc);
            atomicAdd(&st->tot_m2p_list, (unsigned long long)nm);
            atomicAdd(&st->tot_p2p_list, (unsigned long long)np);
            atomicAdd(&st->tot_p2p_src, (unsigned long long)nsrc);
            if (BG && nl) atomicAdd(&st->tot_left_list, (unsigned long long)nl);
        }
    }
}

// SHARED WALK ("bundle a set of m source cells which have interactions in common with a set of n sink particles";
// SURVEY.md 8(f) NEXT-4, second half: a walk that shares lists between neighbouring groups).  One warp walks a RUN of up to
// `sgn` (<= WSG) consecutive groups - groups [j sgn, (j+1) sgn), neighbours along the Morton curve - in two kinds of phases:
//   common  : against the UNION of the run's boxes.  A cell the union accepts is accepted by every member (its distance to a
//             member's box is no smaller) and goes to every member's list; a cell that every member rejects (it fails even at
//             the union's farthest point, or fails box by box) is opened once for all; a cell on which the members disagree is
//             set aside together with its image id (the "residual" list, kept at the top of the stack array);
//   member  : each member in turn walks the residual cells against its own box, exactly as a lone group would.
// A group's lists hold the same entries as those of a walk of its own (an ancestor of an accepted cell was rejected by that
// group either way), in another order; sgn = 1 is the lone walk.  The run's composition depends on the group indices and, with
// background subtraction, on the windows (only groups with the same window share: the window decides which copy of a cell is
// listed and which cubes are exposed) - not on g0, g1 or the active flags, which only select the members whose lists are written:
// a sharded, batched or active-subset evaluation lists every group's entries in the same order as a full one.
#define WSG 8
#ifdef DSK_DEBUG_BOUNDS
#define WK_CHECK(cond) do { if (!(cond)) { printf("walk bounds: %s line %d block %d lane %d\n", #cond, __LINE__, blockIdx.x, threadIdx.x); __trap(); } } while (0)
#else
#define WK_CHECK(cond) do { } while (0)
#endif
template <int MODE, bool ABS>          // MODE 0 COUNT, 1 FILL at the scanned offsets, 2 ONE pass into a fixed capacity per group
__global__ void __launch_bounds__(32) k_walk_sh(uint32_t g0, uint32_t g1, uint32_t ngroup, int sgn, int periodic, float box, int pow1, float k1_h,
                                             const dsk_cellrec *__restrict__ cell,
                                             const float4 *__restrict__ wmac,
                                             const float4 *__restrict__ gbox,
                                             const uint32_t *__restrict__ gcount,
                                             uint32_t *__restrict__ m2p_len, uint32_t *__restrict__ p2p_len,
                                             uint32_t *__restrict__ p2p_src,
                                             const uint64_t *__restrict__ m2p_off,
                                             const uint64_t *__restrict__ p2p_off, uint64_t m2p_base,
                                             uint64_t p2p_base, uint32_t *__restrict__ list_m2p,
                                             uint32_t *__restrict__ list_p2p, const uint8_t *__restrict__ gact,
                                             uint32_t cap_m, uint32_t cap_p, uint64_t *__restrict__ m2p_off_out,
                                             uint64_t *__restrict__ p2p_off_out, const walk_bg bg, dsk_devstate *st)
{
    constexpr bool FILL = MODE != 0;
    constexpr uint32_t CELL_MASK = (1u << DSK_CELL_BITS) - 1u;
    constexpr int TRIP = 32 * WEPL;
    __shared__ uint32_t stk[WSTACK];
    __shared__ uint32_t imgtab[WK_NIMG];
    __shared__ float4 mbox[WSG][2];
    __shared__ uint64_t moff[WSG], poff[WSG], loff[WSG];
    const int lane = threadIdx.x;
    const uint32_t lt = (1u << lane) - 1u;
    // the runs that hold a group of [g0, g1)
    const uint32_t gs = (g0 / (uint32_t)sgn + blockIdx.x) * (uint32_t)sgn;
    if (gs >= g1) return;
    const int nrun = (int)min((uint32_t)sgn, ngroup - gs);
    const bool BG = bg.lb >= 0;
    if (periodic) wk_img_table(imgtab, lane);
    // lane i < nrun holds group gs + i: its box, its window, whether its lists are wanted
    int wl[3] = {0, 0, 0}, wh[3] = {0, 0, 0};
    bool want = false;
    if (lane < nrun) {
        const uint32_t g = gs + lane;
        mbox[lane][0] = gbox[2 * (size_t)g]; mbox[lane][1] = gbox[2 * (size_t)g + 1];
        const bool inr = g >= g0 && g < g1;
        want = inr && !(gact && !gact[g]);
        if (inr && !want && MODE != 1) {              // no active sink in this group (dsk_accel_active): empty lists
            m2p_len[g] = 0; p2p_len[g] = 0; p2p_src[g] = 0;
            if (BG) bg.left_len[g] = 0;
            if (MODE == 2) {
                m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p;
                if (BG) bg.left_off_out[g] = (uint64_t)g * bg.cap_l;
            }
        }
        if (want) {
            if (MODE == 1) { moff[lane] = m2p_off[g] - m2p_base; poff[lane] = p2p_off[g] - p2p_base; loff[lane] = BG ? bg.left_off[g] - bg.left_base : 0; }
            if (MODE == 2) { moff[lane] = (uint64_t)g * cap_m; poff[lane] = (uint64_t)g * cap_p; loff[lane] = BG ? (uint64_t)g * bg.cap_l : 0; }
        }
        if (BG) {
            // the group's window: the level-lb cells within k of the footprint of its cell (integer index range, unwrapped frame)
            const uint32_t cg = bg.gcell[g];
            const int lg = (int)(cell[cg].meta >> 8);
            const uint64_t prefix = bg.hotkey[cg] & ~(1ull << (3 * lg));
            const int q[3] = {(int)wk_compact3(prefix >> 2), (int)wk_compact3(prefix >> 1), (int)wk_compact3(prefix)};
#pragma unroll
            for (int d = 0; d < 3; d++) {
                int flo, fhi;
                if (lg >= bg.lb) flo = fhi = q[d] >> (lg - bg.lb);
                else { flo = q[d] << (bg.lb - lg); fhi = flo + (1 << (bg.lb - lg)) - 1; }
                wl[d] = flo - bg.k; wh[d] = fhi + bg.k;
            }
        }
    }
    __syncwarp();
    uint32_t todo = __ballot_sync(0xffffffffu, lane < nrun);
    while (todo) {
        // the next set of members: the first group not yet walked and those of the run with its window
        const int a = __ffs(todo) - 1;
        int wlo[3], whi[3];
        bool same = (todo >> lane) & 1u;
#pragma unroll
        for (int d = 0; d < 3; d++) {
            wlo[d] = __shfl_sync(0xffffffffu, wl[d], a); whi[d] = __shfl_sync(0xffffffffu, wh[d], a);
            same = same && wl[d] == wlo[d] && wh[d] == whi[d];
        }
        const uint32_t mset = __ballot_sync(0xffffffffu, same);
        const uint32_t wantset = __ballot_sync(0xffffffffu, same && want);
        todo &= ~mset;
        if (!wantset) continue;
        const int m = __popc(mset);
        float ulo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, uhi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        for (uint32_t t = mset; t; t &= t - 1u) {
            const int i = __ffs(t) - 1;
            const float4 lo = mbox[i][0], hi = mbox[i][1];
            ulo[0] = fminf(ulo[0], lo.x); ulo[1] = fminf(ulo[1], lo.y); ulo[2] = fminf(ulo[2], lo.z);
            uhi[0] = fmaxf(uhi[0], hi.x); uhi[1] = fmaxf(uhi[1], hi.y); uhi[2] = fmaxf(uhi[2], hi.z);
        }
        // root of every image of the block in use: periodic = the block's half-width ws (0 isolated); ids are those of the 5^3
        // encoding.  A lone group starts its member phase from them; a set starts its common phase from them.
        int sp = 0, rtop = WSTACK;
        auto seed_roots = [&](bool top_end) {
            const int side = 2 * DSK_WS + 1, nid = periodic ? side * side * side : 1;
            for (int i0 = 0; i0 < nid; i0 += 32) {
                const int i = i0 + lane;
                bool in = i < nid;
                if (periodic && in) {
                    const int iz = i % side - DSK_WS, iy = (i / side) % side - DSK_WS, ix = i / (side * side) - DSK_WS;
                    in = abs(ix) <= periodic && abs(iy) <= periodic && abs(iz) <= periodic;
                }
                const uint32_t mk = __ballot_sync(0xffffffffu, in);
                const uint32_t v = (uint32_t)(periodic ? i : 0) << DSK_CELL_BITS;
                if (top_end) { rtop -= __popc(mk); if (in) stk[rtop + __popc(mk & lt)] = v; }
                else { if (in) stk[sp + __popc(mk & lt)] = v; sp += __popc(mk); }
            }
            __syncwarp();
        };
        seed_roots(m == 1);
        uint32_t cnm = 0, cnp = 0, cnsrc = 0, cnl = 0;            // what the common phase listed (for every member)
        uint32_t rest = wantset;
        for (int ph = (m > 1 ? 0 : 1); rest != 0u; ph++) {
            const bool common = ph == 0;
            float blo[3], bhi[3];
            uint32_t wset = wantset;
            int gi = -1;
            uint32_t nm = 0, np = 0, nsrc = 0, nl = 0;
            if (common) {
#pragma unroll
                for (int d = 0; d < 3; d++) { blo[d] = ulo[d]; bhi[d] = uhi[d]; }
            } else {
                gi = __ffs(rest) - 1; rest &= rest - 1u; wset = 1u << gi;
                const float4 lo = mbox[gi][0], hi = mbox[gi][1];
                blo[0] = lo.x; blo[1] = lo.y; blo[2] = lo.z; bhi[0] = hi.x; bhi[1] = hi.y; bhi[2] = hi.z;
                nm = cnm; np = cnp; nsrc = cnsrc; nl = cnl;
                sp = 0;
            }
            int rp = rtop;                            // member phase: the residual cells not yet taken
            bool ovf = false;
            // WEPL stack entries per lane and trip: their loads are independent, so a trip exposes one L2 round trip for 32 * WEPL cells
            while (sp > 0 || (!common && rp < WSTACK)) {
                uint32_t e[WEPL], nchild[WEPL], child0[WEPL];
                bool act[WEPL], accept[WEPL], leaf[WEPL];
                float4 h[WEPL], rr[WEPL];
                int4 geo[WEPL];
                if (sp > 0) {
                    // A popped cell pushes at most 8 children (net +7), so a trip of `take` cells needs 7 * take free entries (the
                    // common phase also up to `take` residual entries at the other end).  Trips shrink as the stack fills and end
                    // as a plain depth-first walk (take = 1), whose height above its starting point is at most 7 per level = 147 <
                    // WRESERVE: a member phase cannot overflow on any tree of <= 21 levels while the residual list leaves it
                    // WRESERVE + 8 entries, which the common phase guarantees (it gives up sharing before that).
                    const int room = ((common ? rtop - TRIP : rtop) - WRESERVE - sp) / 7;
                    if (common && (room < 1 || rtop < WSTACK / 4)) { ovf = true; break; }
                    int take = sp < TRIP ? sp : TRIP;
                    take = min(take, max(room, 1));
#pragma unroll
                    for (int q = 0; q < WEPL; q++) {
                        act[q] = lane + 32 * q < take;
                        e[q] = act[q] ? stk[sp - 1 - lane - 32 * q] : 0u;
                    }
                    sp -= take;
                } else {
                    const int take = min(min(TRIP, WSTACK - rp), max((rtop - WRESERVE) / 7, 1));      // the stack is empty: room as above
#pragma unroll
                    for (int q = 0; q < WEPL; q++) {
                        act[q] = lane + 32 * q < take;
                        WK_CHECK(!act[q] || (rp + lane + 32 * q >= rtop && rp + lane + 32 * q < WSTACK));
                        e[q] = act[q] ? stk[rp + lane + 32 * q] : 0u;
                    }
                    rp += take;
                }
                __syncwarp();
#pragma unroll
                for (int q = 0; q < WEPL; q++)
                    if (act[q]) {
                        const uint32_t c = e[q] & CELL_MASK;
                        h[q] = wmac[2 * (size_t)c];            // com.xyz, critical radius s/theta + delta
                        rr[q] = wmac[2 * (size_t)c + 1];       // the cell record (same sector)
                        if (BG && c < bg.ntop) geo[q] = bg.topgeo[c];
                    }
                uint32_t push[WEPL], ptot = 0;
#pragma unroll
                for (int q = 0; q < WEPL; q++) {
                    accept[q] = false; leaf[q] = false; nchild[q] = 0; child0[q] = 0;
                    uint32_t cnt = 0, nexp = 0, entry = e[q];
                    const uint32_t c = e[q] & CELL_MASK;
                    const bool top = BG && act[q] && c < bg.ntop;
                    int ish[3] = {0, 0, 0};
                    bool whole = false, mixed = false, winside = false, winter = false;
                    if (act[q]) {
                        float sh[3];
                        const int img = (int)(e[q] >> DSK_CELL_BITS);
                        wk_image(imgtab, img, periodic, box, sh, ish);
                        const float zx = h[q].x + sh[0], zy = h[q].y + sh[1], zz = h[q].z + sh[2];
                        const float d2 = wk_d2(zx, zy, zz, blo, bhi);
                        bool straddles = false;
                        if (top) {
                            // where the cell's cube lies relative to the window (integers: both sides decide alike)
                            const int lvl = geo[q].w & 255;
                            const int qq[3] = {geo[q].x, geo[q].y, geo[q].z};
                            winside = true; winter = true;
#pragma unroll
                            for (int d = 0; d < 3; d++) {
                                const int lo = (qq[d] << (bg.lb - lvl)) + (ish[d] << bg.lb), hi = lo + (1 << (bg.lb - lvl)) - 1;
                                winside = winside && lo >= wlo[d] && hi <= whi[d];
                                winter = winter && lo <= whi[d] && hi >= wlo[d];
                            }
                            straddles = winter && !winside;      // partly inside the window: never accepted (its background would count twice)
                            if (!winter) entry = (e[q] & ~CELL_MASK) | (bg.ncell + c);      // outside: the background-subtracted copy
                        }
                        const uint32_t meta = __float_as_uint(rr[q].w);
                        float kappa = 0.0f;
                        if (ABS) kappa = (top && entry != e[q]) ? bg.kbg[c] : rr[q].x;      // the subtracted copy has its own bound
                        const float crit = h[q].w;
                        const bool ok = wk_ok<ABS>(d2, crit, meta, kappa, box, pow1, k1_h);
                        accept[q] = !straddles && ok;
                        if (common && !straddles && !ok) {
                            // rejected by the union: by every member?  Not if it passes at the union's farthest point and at a member's box.
                            const float fx = fmaxf(fabsf(zx - blo[0]), fabsf(zx - bhi[0])), fy = fmaxf(fabsf(zy - blo[1]), fabsf(zy - bhi[1])),
                                        fz = fmaxf(fabsf(zz - blo[2]), fabsf(zz - bhi[2]));
                            if (wk_ok<ABS>(__fmaf_rn(fz, fz, __fmaf_rn(fy, fy, __fmul_rn(fx, fx))), crit, meta, kappa, box, pow1, k1_h))
                                for (uint32_t t = mset; t && !mixed; t &= t - 1u) {
                                    const int i = __ffs(t) - 1;
                                    const float4 lo4 = mbox[i][0], hi4 = mbox[i][1];
                                    const float lo[3] = {lo4.x, lo4.y, lo4.z}, hi[3] = {hi4.x, hi4.y, hi4.z};
                                    mixed = wk_ok<ABS>(wk_d2(zx, zy, zz, lo, hi), crit, meta, kappa, box, pow1, k1_h);
                                }
                        }
                        if (!accept[q] && !mixed) {
                            nchild[q] = meta & 255u; child0[q] = __float_as_uint(rr[q].z); cnt = __float_as_uint(rr[q].y);
                            leaf[q] = nchild[q] == 0;
                            if (top) {
                                whole = leaf[q] || (geo[q].w & 255) == bg.lb;
                                // cubes this cell exposes outside the window: none if it lies inside; itself; all its empty octants if it lies outside;
                        // octant by octant only when it straddles the window's edge
                        nexp = winside ? 0u : whole ? 1u : !winter ? 8u - (uint32_t)__popc((geo[q].w >> 8) & 255)
                                                                   : wk_exposed(false, geo[q].w & 255, bg.lb, geo[q], ish, wlo, whi, nullptr);
                            }
                        }
                    }
                    const uint32_t bm = __ballot_sync(0xffffffffu, accept[q]);
                    const uint32_t bl = __ballot_sync(0xffffffffu, leaf[q]);
                    if (FILL) {
                        const uint32_t im = nm + __popc(bm & lt), ip = np + __popc(bl & lt);
                        const bool wm = accept[q] && (MODE == 1 || im < cap_m), wp = leaf[q] && (MODE == 1 || ip < cap_p);
                        if (wm || wp)
                            for (uint32_t t = wset; t; t &= t - 1u) {
                                const int i = __ffs(t) - 1;
                                WK_CHECK(i < nrun && ((wantset >> i) & 1u));
                                if (wm) list_m2p[moff[i] + im] = entry;
                                if (wp) list_p2p[poff[i] + ip] = e[q];
                            }
                    }
                    nm += __popc(bm); np += __popc(bl);
                    if (leaf[q]) nsrc += cnt;
                    if (common) {                                           // cells the members disagree on: to the residual list
                        const uint32_t bx = __ballot_sync(0xffffffffu, mixed);
                        rtop -= __popc(bx);
                        WK_CHECK(rtop >= sp && rtop + __popc(bx) <= WSTACK);
                        if (mixed) stk[rtop + __popc(bx & lt)] = e[q];
                    }
                    if (BG && __any_sync(0xffffffffu, nexp != 0u)) {           // rare: cubes kept outside the window
                        uint32_t x = nexp;
                        for (int o = 1; o < 32; o <<= 1) {
                            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
                            if (lane >= o) x += y;
                        }
                        const uint32_t tot = __shfl_sync(0xffffffffu, x, 31), at = nl + x - nexp;
                        if (FILL && nexp && (MODE == 1 || at + nexp <= bg.cap_l))
                            for (uint32_t t = wset; t; t &= t - 1u)
                                wk_exposed(whole, geo[q].w & 255, bg.lb, geo[q], ish, wlo, whi, bg.list_left + loff[__ffs(t) - 1] + at);
                        nl += tot;
                    }
                    push[q] = (act[q] && !accept[q] && !mixed) ? nchild[q] : 0u;      // children of rejected internal cells
                    ptot += push[q];
                }
                uint32_t x = ptot;
                for (int o = 1; o < 32; o <<= 1) {
                    uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
                    if (lane >= o) x += y;
                }
                const uint32_t tot = __shfl_sync(0xffffffffu, x, 31);
                if (sp + (int)tot > rtop) {
                    if (lane == 0) atomicOr(&st->status, ST_STACKOVF);
                    sp = 0; rp = WSTACK;
                    break;
                }
                uint32_t at = sp + x - ptot;
#pragma unroll
                for (int q = 0; q < WEPL; q++) {
                    const uint32_t img = e[q] & ~CELL_MASK;
                    WK_CHECK(at + push[q] <= (uint32_t)rtop);
#pragma unroll
                    for (uint32_t k = 0; k < 8; k++)
                        if (k < push[q]) stk[at + k] = img | (child0[q] + k);
                    at += push[q];
                }
                sp += (int)tot;
                __syncwarp();
            }
            __syncwarp();
            if (common) {
                if (ovf) {           // the residual list and the stack met: no sharing for this set, every member walks from the roots
                    rtop = WSTACK; sp = 0;
                    seed_roots(true);
                } else { cnm = nm; cnp = np; cnsrc = nsrc; cnl = nl; }
                continue;
            }
            for (int o = 16; o; o >>= 1) nsrc += __shfl_xor_sync(0xffffffffu, nsrc, o);      // per-lane partial sums (cnsrc too)
            if (lane == 0) {
                const uint32_t g = gs + (uint32_t)gi;
                if (MODE != 1) {
                    m2p_len[g] = nm; p2p_len[g] = np; p2p_src[g] = nsrc;
                    if (BG) bg.left_len[g] = nl;
                }
                if (MODE == 2) {
                    m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p;
                    if (BG) bg.left_off_out[g] = (uint64_t)g * bg.cap_l;
                    if (nm > cap_m || np > cap_p || (BG && nl > bg.cap_l)) st->scratch[0] = 1ull;      // a list did not fit: the host falls back to two passes
                }
                if (FILL) {
                    const unsigned long long ns = gcount[g];
                    atomicAdd(&st->n_m2p, ns * nm);
                    atomicAdd(&st->n_p2p, ns * nsrc);
                    atomicAdd(&st->tot_m2p_list, (unsigned long long)nm);
                    atomicAdd(&st->tot_p2p_list, (unsigned long long)np);
                    atomicAdd(&st->tot_p2p_src, (unsigned long long)nsrc);
                    if (BG && nl) atomicAdd(&st->tot_left_list, (unsigned long long)nl);
                }
            }
        }
        __syncwarp();
    }
}

// u32 lengths -> u64 exclusive offsets, off[n] = total.  Two launches over a fixed grid: per-block sums, then
// each block adds the sums of the blocks before it to the scan of its own contiguous chunk.
#define S64_THREADS 256
__global__ void __launch_bounds__(S64_THREADS) k_scan64_reduce(const uint32_t *__restrict__ len, uint32_t n,
                                                              uint64_t *__restrict__ bsum)
{
    __shared__ uint64_t sh[S64_THREADS / 32];
    const uint32_t chunk = ((n + gridDim.x - 1) / gridDim.x + S64_THREADS - 1) / S64_THREADS * S64_THREADS;
    const uint64_t lo = (uint64_t)blockIdx.x * chunk, hi = min((uint64_t)n, lo + chunk);
    uint64_t s = 0;
    for (uint64_t i = lo + threadIdx.x; i < hi; i += S64_THREADS) s += len[i];
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint64_t t = 0;
        for (int w = 0; w < S64_THREADS / 32; w++) t += sh[w];
        bsum[blockIdx.x] = t;
    }
}
__global__ void __launch_bounds__(S64_THREADS) k_scan64_apply(const uint32_t *__restrict__ len, uint32_t n,
                                                             const uint64_t *__restrict__ bsum,
                                                             uint64_t *__restrict__ off)
{
    __shared__ uint64_t wsum[S64_THREADS / 32];
    __shared__ uint64_t s_pre, s_all;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) {
        uint64_t pre = 0, all = 0;
        for (uint32_t b = lane; b < gridDim.x; b += 32) {
            const uint64_t v = bsum[b];
            all += v;
            if (b < blockIdx.x) pre += v;
        }
        for (int o = 16; o; o >>= 1) { pre += __shfl_xor_sync(0xffffffffu, pre, o); all += __shfl_xor_sync(0xffffffffu, all, o); }
        if (lane == 0) { s_pre = pre; s_all = all; }
    }
    __syncthreads();
    if (blockIdx.x == 0 && threadIdx.x == 0) off[n] = s_all;
    const uint32_t chunk = ((n + gridDim.x - 1) / gridDim.x + S64_THREADS - 1) / S64_THREADS * S64_THREADS;
    const uint64_t lo = (uint64_t)blockIdx.x * chunk, hi = min((uint64_t)n, lo + chunk);
    uint64_t carry = s_pre;
    for (uint64_t i0 = lo; i0 < hi; i0 += S64_THREADS) {
        const uint64_t i = i0 + threadIdx.x;
        const uint64_t v = i < hi ? len[i] : 0;
        uint64_t x = v;
        for (int o = 1; o < 32; o <<= 1) {
            const uint64_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        uint64_t wpre = 0, tot = 0;
        for (int w = 0; w < S64_THREADS / 32; w++) { const uint64_t t = wsum[w]; if (w < warp) wpre += t; tot += t; }
        if (i < hi) off[i] = carry + wpre + x - v;
        carry += tot;
        __syncthreads();
    }
}
static void scan64(dsk_ctx *c, const uint32_t *len, uint32_t n, uint64_t *off)
{
    int grid = c->nsm * 2;
    if ((uint64_t)grid * S64_THREADS > (uint64_t)n) grid = (int)((n + S64_THREADS - 1) / S64_THREADS);
    if (grid < 1) grid = 1;
    uint64_t *bsum = reinterpret_cast<uint64_t *>(c->scan_tmp);        // 4096 u32 = 2048 u64 >= grid
    k_scan64_reduce<<<grid, S64_THREADS, 0, c->stream>>>(len, n, bsum);
    k_scan64_apply<<<grid, S64_THREADS, 0, c->stream>>>(len, n, bsum, off);
    DSK_COUNT(c, 2);
}

// the 32 bytes the walk reads per tested cell: centre of mass and critical radius s/theta + delta | the cell record.
// abs_tol > 0 (absolute-error MAC): critical radius s + delta, and kappa_c = (p + 2) Q_c / (tol b_c^2) in the slot of `first`;
// kbg[c] = the same for the background-subtracted copy of a top cell, Q' = Q + rho_bar tr C = 2 Q - tr M'.
// k1_h > 0 (K1 softening, O6b): the critical radius is at least b + h, b = sqrt(3)/2 s + delta: a cell is expanded only if all its
// sources lie outside the kernel's support of every sink of the group.
__global__ void __launch_bounds__(256) k_walk_mac(uint32_t ncell, float box, float inv_theta, float abs_tol, float k1_h, int p, int rowlen,
                                                  const float *__restrict__ rows, uint32_t ntop, const float *__restrict__ rows_bg,
                                                  const dsk_cellrec *__restrict__ cell, const float4 *__restrict__ whdr,
                                                  float4 *__restrict__ wmac, float *__restrict__ kbg)
{
    const uint32_t c = blockIdx.x * 256 + threadIdx.x;
    if (c >= ncell) return;
    float4 h = whdr[c];
    const int level = (int)(cell[c].meta >> 8);
    const float s = box * exp2f((float)-level), delta = h.w;
    h.w = s * inv_theta + delta;
    if (k1_h > 0.0f && !(abs_tol > 0.0f)) h.w = fmaxf(h.w, 0.8660254f * s + delta + k1_h);     // (the absolute-error walk tests d > b + h itself)
    wmac[2 * (size_t)c] = h;
    // the cell record rides in the same 32-byte sector: a rejected cell needs it, and a second, dependent load would
    // double the latency of every walk iteration
    const dsk_cellrec r = cell[c];
    float4 rec = make_float4(__uint_as_float(r.first), __uint_as_float(r.count), __uint_as_float(r.child0), __uint_as_float(r.meta));
    if (abs_tol > 0.0f) {
        const float *row = rows + (size_t)c * rowlen;
        const float tr = row[8 + dsk_midx(2, 0, 0)] + row[8 + dsk_midx(0, 2, 0)] + row[8 + dsk_midx(0, 0, 2)];   // sum Mhat_2 = Q / (2 s^2)
        const float bs = 0.8660254f + delta / s;                                                         // b / s
        rec.x = (float)(p + 2) * 2.0f * tr / (abs_tol * bs * bs);
        if (c < ntop && kbg) {
            const float *rb = rows_bg + (size_t)c * rowlen;
            const float trb = rb[8 + dsk_midx(2, 0, 0)] + rb[8 + dsk_midx(0, 2, 0)] + rb[8 + dsk_midx(0, 0, 2)];
            kbg[c] = (float)(p + 2) * 2.0f * (2.0f * tr - trb) / (abs_tol * bs * bs);
        }
    }
    wmac[2 * (size_t)c + 1] = rec;
}

// groups per shared walk: the context's setting (dsk_set_walk_sharing); 0 = the library's choice = 1, the lone walk (measured faster
// on every config of BASELINE.json: the walk is latency-bound and wants warps)
static int walk_sgn(const dsk_ctx *c)
{
    if (c->walk_share > 0) return c->walk_share < WSG ? c->walk_share : WSG;
    return 1;
}
static unsigned walk_grid(uint32_t g0, uint32_t g1, int sgn) { return g1 > g0 ? (g1 - 1) / (uint32_t)sgn - g0 / (uint32_t)sgn + 1 : 0u; }

static walk_bg make_walk_bg(dsk_ctx *c, uint64_t left_base, uint32_t cap_l)
{
    walk_bg b;
    memset(&b, 0, sizeof(b));
    b.lb = -1;
    if (c->periodic && c->bg) {
        b.lb = c->bg_level; b.k = dsk_bg_halfwidth(c->theta, c->bg_level, c->img_ws);
        b.ntop = c->ntop; b.ncell = c->hstate->ncell;
        b.topgeo = c->topgeo; b.gcell = c->gcell; b.hotkey = c->hotkey;
        b.left_len = c->g_left_len; b.left_off = c->g_left_off; b.left_base = left_base;
        b.list_left = c->list_left; b.cap_l = cap_l; b.left_off_out = c->g_left_off;
        b.kbg = c->kbg;
    }
    return b;
}

// one launch of the walk over the groups [g0, g1): the lone kernel, or the shared one when groups share (walk_sgn > 1)
template <int MODE>
static void launch_walk(dsk_ctx *c, uint32_t g0, uint32_t g1, const uint64_t *m2p_off, const uint64_t *p2p_off, uint64_t m2p_base,
                        uint64_t p2p_base, uint32_t *list_m2p, uint32_t *list_p2p, const uint8_t *gact, uint32_t cap_m, uint32_t cap_p,
                        uint64_t *m2p_off_out, uint64_t *p2p_off_out, const walk_bg &bg)
{
    if (g1 <= g0) return;
    const bool ABS = c->mac_kind == 1;
    const int sgn = walk_sgn(c), per = c->periodic ? c->img_ws : 0, pow1 = c->p + 1;
    const float k1_h = c->soft_kind == 1 ? c->eps : 0.0f;
    if constexpr (MODE != 3) {          // (predicted capacities are a lone-walk form: dsk_run_walk does not predict when groups share)
        if (sgn > 1) {
            (ABS ? k_walk_sh<MODE, true> : k_walk_sh<MODE, false>)<<<walk_grid(g0, g1, sgn), 32, 0, c->stream>>>(
                g0, g1, c->hstate->ngroup, sgn, per, c->box, pow1, k1_h, c->cell, c->wmac, c->gbox, c->gcount, c->g_m2p_len, c->g_p2p_len, c->g_p2p_src,
                m2p_off, p2p_off, m2p_base, p2p_base, list_m2p, list_p2p, gact, cap_m, cap_p, m2p_off_out, p2p_off_out, bg, c->dstate);
            return;
        }
    }
    {
        (ABS ? k_walk<MODE, true> : k_walk<MODE, false>)<<<(g1 - g0 + WW - 1) / WW, WW * 32, 0, c->stream>>>(
            g0, g1, per, c->box, pow1, k1_h, c->cell, c->wmac, c->gbox, c->gcount, c->g_m2p_len, c->g_p2p_len, c->g_p2p_src,
            m2p_off, p2p_off, m2p_base, p2p_base, list_m2p, list_p2p, gact, cap_m, cap_p, m2p_off_out, p2p_off_out, bg, c->dstate);
    }
}

// ---- list lengths predicted from the previous evaluation ---------------------------------------------------------------------------
// When the lists do not fit a fixed capacity per group (512^3: 3.4 M groups, lists of 1500 cells on average and 2800 at most against a
// 12 GiB buffer), the walk runs twice, COUNT and FILL: 2 x 28 ms of a dsk_kdk_step.  From one step to the next the tree hardly changes, so
// the second evaluation onwards sizes every group's slots from the lengths the groups of the SAME REGION had last time: a group is a tree
// cell, i.e. an interval of Morton keys; the old groups' interval starts are kept sorted (they are in Morton order), a new group takes the
// largest old length among the old groups its interval meets, plus a half and 128 entries (cells; twice + 64 for the leaves).  One walk
// (MODE 3) fills the slots and writes the true lengths; a list that outgrew its slot sets the overflow flag and the evaluation starts
// over with COUNT + FILL, and the context then sits out 1, 3, 7, 15 evaluations before it predicts again.  Measured on C5 (a synthetic
// box far from equilibrium: the number of groups falls 3.47 -> 3.07 -> 2.67 -> 2.60 M over the first steps): no overflow from the
// second step on, 1351 -> 1319 ms per step; with margins of a quarter + 96 / 32 a slot overflowed in every step (then 1382 ms).
__device__ __forceinline__ uint64_t pg_interval(uint32_t cg, const dsk_cellrec *__restrict__ cell, const uint64_t *__restrict__ hotkey, uint64_t *hi)
{
    const int l = (int)(cell[cg].meta >> 8), sh = 3 * (DSK_KEY_LEVELS - l);
    const uint64_t prefix = hotkey[cg] & ~(1ull << (3 * l));
    const uint64_t lo = prefix << sh;
    *hi = lo + (1ull << sh);
    return lo;
}
__global__ void __launch_bounds__(256) k_pg_store(uint32_t ng, const uint32_t *__restrict__ gcell, const dsk_cellrec *__restrict__ cell,
                                                  const uint64_t *__restrict__ hotkey, const uint32_t *__restrict__ m2p_len,
                                                  const uint32_t *__restrict__ p2p_len, const uint32_t *__restrict__ left_len,
                                                  uint64_t *__restrict__ pg_key, uint32_t *__restrict__ pg_m2p, uint32_t *__restrict__ pg_p2p,
                                                  uint32_t *__restrict__ pg_left)
{
    const uint32_t g = blockIdx.x * 256 + threadIdx.x;
    if (g >= ng) return;
    uint64_t hi;
    pg_key[g] = pg_interval(gcell[g], cell, hotkey, &hi);
    pg_m2p[g] = m2p_len[g]; pg_p2p[g] = p2p_len[g]; pg_left[g] = left_len ? left_len[g] : 0u;
}
__global__ void __launch_bounds__(256) k_pg_predict(uint32_t ng, const uint32_t *__restrict__ gcell, const dsk_cellrec *__restrict__ cell,
                                                    const uint64_t *__restrict__ hotkey, uint32_t pg_n, const uint64_t *__restrict__ pg_key,
                                                    const uint32_t *__restrict__ pg_m2p, const uint32_t *__restrict__ pg_p2p,
                                                    const uint32_t *__restrict__ pg_left, uint32_t *__restrict__ cap_m,
                                                    uint32_t *__restrict__ cap_p, uint32_t *__restrict__ cap_l)
{
    const uint32_t g = blockIdx.x * 256 + threadIdx.x;
    if (g >= ng) return;
    uint64_t hi;
    const uint64_t lo = pg_interval(gcell[g], cell, hotkey, &hi);
    uint32_t a = 0, b = pg_n;                        // last old group whose interval starts at or before lo (or the first)
    while (b - a > 1) {
        const uint32_t mid = a + ((b - a) >> 1);
        if (pg_key[mid] <= lo) a = mid; else b = mid;
    }
    uint32_t m = 0, p = 0, l = 0;
    for (uint32_t j = a, k = 0; j < pg_n && k < 64 && (k < 2 || pg_key[j] < hi); j++, k++) {       // it, its successor, and all that start inside
        m = max(m, pg_m2p[j]); p = max(p, pg_p2p[j]); l = max(l, pg_left[j]);
    }
    cap_m[g] = m + (m >> 1) + 128u; cap_p[g] = 2u * p + 64u;
    if (cap_l) cap_l[g] = 2u * l + 16u;
}

// W.  First choice: ONE pass into a fixed capacity per group (list buffer / number of groups), which saves the COUNT
// pass and the scans whenever every list fits — checked with one flag read; a context that saw an overflow at this
// theta goes straight to the general form: COUNT pass + offsets here, FILL per batch from dsk_walk_fill (force.cu).
int dsk_run_walk(dsk_ctx *c)
{
    const uint32_t ng = c->hstate->ngroup;
    cudaStream_t s = c->stream;
    const float inv_theta = 1.0f / c->theta;
    cudaEventRecord(c->ev[7], s);
    const uint32_t nc = c->hstate->ncell;
    const bool ABS = c->mac_kind == 1;
    k_walk_mac<<<(nc + 255) / 256, 256, 0, s>>>(nc, c->box, ABS ? 1.0f : inv_theta, ABS ? c->mac_tol : 0.0f, c->soft_kind == 1 ? c->eps : 0.0f, c->p, dsk_rowlen(c->p), c->rows,
                                                c->periodic && c->bg ? c->ntop : 0u, c->rows_bg, c->cell, c->whdr, c->wmac, c->kbg);
    DSK_COUNT(c, 1);
    c->walk_onepass = 0;
    const bool BG = c->periodic && c->bg;
    const uint64_t cap_m = ng ? c->list_m2p_cap / ng : 0, cap_p = ng ? c->list_p2p_cap / ng : 0, cap_l = ng && BG ? c->list_left_cap / ng : 0;
    const bool tiny = c->walk_two_pass_only == 2;          // diagnostic: capacities that overflow, to exercise the fallback
    if (cap_m >= 4096 && cap_p >= 512 && (c->onepass_bad_theta != c->theta || tiny) && c->walk_two_pass_only != 1 &&
        c->walk_two_pass_only < 3) {
        DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_m2p_list, 0, sizeof(unsigned long long) * 5, s));
        DSK_CUDA(cudaMemsetAsync(&c->dstate->scratch[0], 0, sizeof(unsigned long long), s));
        DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_left_list, 0, sizeof(unsigned long long), s));
        const uint32_t cm = tiny ? 64u : (uint32_t)(cap_m > 0xffffff00ull ? 0xffffff00ull : cap_m),
                       cp = tiny ? 8u : (uint32_t)(cap_p > 0xffffff00ull ? 0xffffff00ull : cap_p),
                       cl = (uint32_t)(cap_l > 0xffffff00ull ? 0xffffff00ull : cap_l);
        launch_walk<2>(c, 0, ng, nullptr, nullptr, 0, 0, c->list_m2p, c->list_p2p, c->gact_cur, cm, cp, c->g_m2p_off, c->g_p2p_off, make_walk_bg(c, 0, cl));
        DSK_COUNT(c, 1);
        unsigned long long ovf = 0;
        DSK_CUDA(cudaMemcpyAsync(&ovf, &c->dstate->scratch[0], sizeof(ovf), cudaMemcpyDeviceToHost, s));
        DSK_CUDA(cudaStreamSynchronize(s));
        if (!ovf) { c->walk_onepass = 1; return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA; }
        c->onepass_bad_theta = c->theta;
    }
    c->walk_predicted = 0;
    if (c->pg_valid && c->pg_n > 0 && !c->gact_cur && walk_sgn(c) == 1 && c->walk_two_pass_only != 1 && ng > 0) {
        // no COUNT pass: slots sized from the previous evaluation's lengths (above); dsk_run_force fills them with MODE 3
        k_pg_predict<<<(ng + 255) / 256, 256, 0, s>>>(ng, c->gcell, c->cell, c->hotkey, c->pg_n, c->pg_key, c->pg_m2p, c->pg_p2p, c->pg_left,
                                                      c->g_m2p_len, c->g_p2p_len, BG ? c->g_left_len : nullptr);
        c->walk_predicted = 1;
    } else {
        launch_walk<0>(c, 0, ng, nullptr, nullptr, 0, 0, nullptr, nullptr, c->gact_cur, 0, 0, nullptr, nullptr, make_walk_bg(c, 0, 0));
    }
    scan64(c, c->g_m2p_len, ng, c->g_m2p_off);
    scan64(c, c->g_p2p_len, ng, c->g_p2p_off);
    if (BG) scan64(c, c->g_left_len, ng, c->g_left_off);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// after an evaluation in the two-pass regime: remember every group's key interval and list lengths for the next one
int dsk_walk_remember(dsk_ctx *c)
{
    const uint32_t ng = c->hstate->ngroup;
    c->pg_valid = 0;
    if (!ng || (int64_t)ng > c->ngroup_cap) return DSK_OK;
    const bool BG = c->periodic && c->bg;
    k_pg_store<<<(ng + 255) / 256, 256, 0, c->stream>>>(ng, c->gcell, c->cell, c->hotkey, c->g_m2p_len, c->g_p2p_len, BG ? c->g_left_len : nullptr,
                                                        c->pg_key, c->pg_m2p, c->pg_p2p, c->pg_left);
    DSK_COUNT(c, 1);
    c->pg_n = ng;
    if (c->walk_predicted) c->pg_backoff = 0;        // the prediction held
    if (c->pg_wait > 0) c->pg_wait--;               // sitting out after an overflow (dsk_api.cu)
    else c->pg_valid = 1;
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_walk_fill(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t m2p_base, uint64_t p2p_base, uint64_t left_base)
{
    if (c->walk_predicted)
        launch_walk<3>(c, g0, g1, c->g_m2p_off, c->g_p2p_off, m2p_base, p2p_base, c->list_m2p, c->list_p2p, c->gact_cur, 0, 0, nullptr, nullptr,
                       make_walk_bg(c, left_base, 0));
    else
        launch_walk<1>(c, g0, g1, c->g_m2p_off, c->g_p2p_off, m2p_base, p2p_base, c->list_m2p, c->list_p2p, c->gact_cur, 0, 0, nullptr, nullptr,
                       make_walk_bg(c, left_base, 0));
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// ---- sink-group sharding over ranks ("cut the sorted list into N_p pieces weighted by work") ----------
// Every rank holds the whole tree.  A COUNT walk of all groups gives each group's list lengths, hence its work
//   w_g = n_sinks (len_M2P flop_M2P + src_P2P flop_P2P);
// the groups are in Morton order, and rank r takes the contiguous run whose prefix sums fall in [r, r+1) total / nranks.  All ranks
// compute the same cut from the same tree: no communication is needed to agree on it.
__global__ void __launch_bounds__(256) k_shard_weight(uint32_t ng, const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ m2p_len,
                                                      const uint32_t *__restrict__ p2p_src, uint32_t fm, uint32_t fp, uint32_t *__restrict__ w)
{
    const uint32_t g = blockIdx.x * 256 + threadIdx.x;
    if (g >= ng) return;
    const unsigned long long v = (unsigned long long)gcount[g] * ((unsigned long long)m2p_len[g] * fm + (unsigned long long)p2p_src[g] * fp);
    w[g] = (uint32_t)min(v >> 10, 0xffffffffull) + 1u;          // + 1: an empty list still costs a task
}
__global__ void k_shard_cut(uint32_t ng, const uint64_t *__restrict__ off, int nranks, uint32_t *__restrict__ cut)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k > nranks) return;
    const uint64_t total = off[ng], target = (uint64_t)(((unsigned __int128)total * (unsigned)k) / (unsigned)nranks);
    uint32_t lo = 0, hi = ng;                                    // first g with off[g] >= target
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (off[mid] < target) lo = mid + 1; else hi = mid;
    }
    cut[k] = k == nranks ? ng : lo;
}
__global__ void __launch_bounds__(256) k_shard_mark(uint32_t ng, uint32_t g_lo, uint32_t g_hi, uint8_t *__restrict__ gact)
{
    const uint32_t g = blockIdx.x * 256 + threadIdx.x;
    if (g < ng) gact[g] = (g >= g_lo && g < g_hi) ? 1 : 0;
}

// cut[0..nranks] (host) for the current tree, theta and acceptance rule; marks the groups of `rank` in c->gact
int dsk_run_shard(dsk_ctx *c, int rank, int nranks, uint32_t flop_m2p, uint32_t flop_p2p, uint32_t *cut_host)
{
    const uint32_t ng = c->hstate->ngroup, nc = c->hstate->ncell;
    cudaStream_t s = c->stream;
    const bool ABS = c->mac_kind == 1;
    k_walk_mac<<<(nc + 255) / 256, 256, 0, s>>>(nc, c->box, ABS ? 1.0f : 1.0f / c->theta, ABS ? c->mac_tol : 0.0f, c->soft_kind == 1 ? c->eps : 0.0f, c->p, dsk_rowlen(c->p), c->rows,
                                                c->periodic && c->bg ? c->ntop : 0u, c->rows_bg, c->cell, c->whdr, c->wmac, c->kbg);
    launch_walk<0>(c, 0, ng, nullptr, nullptr, 0, 0, nullptr, nullptr, nullptr, 0, 0, nullptr, nullptr, make_walk_bg(c, 0, 0));
    uint32_t *w = c->gscan;                                      // [N] scratch of the group extraction, free by now
    k_shard_weight<<<(ng + 255) / 256, 256, 0, s>>>(ng, c->gcount, c->g_m2p_len, c->g_p2p_src, flop_m2p, flop_p2p, w);
    scan64(c, w, ng, c->g_m2p_off);                              // the offsets are rewritten by the walk that follows
    uint32_t *cut = c->task_hist;                                // [1024] scratch
    k_shard_cut<<<(nranks + 1 + 63) / 64, 64, 0, s>>>(ng, c->g_m2p_off, nranks, cut);
    DSK_CUDA(cudaMemcpyAsync(cut_host, cut, sizeof(uint32_t) * (size_t)(nranks + 1), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaStreamSynchronize(s));
    k_shard_mark<<<(ng + 255) / 256, 256, 0, s>>>(ng, cut_host[rank], cut_host[rank + 1], c->gact);
    DSK_COUNT(c, 7);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
