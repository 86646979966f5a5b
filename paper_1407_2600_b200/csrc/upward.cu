// upward.cu — step U: multipole upward pass, P2M at the leaves and M2M up the levels.
// DESIGN.md O4 ("truncated expansion to approximate the contribution of many bodies",
// PAPER.md:75 quadrupole / hexadecapole => order p = highest rank kept).
//
// Stored form (fp32 range + precision):
//   ctr  = geometric cell centre from the hotkey (exact for power-of-two boxes), s = box 2^-level
//   off  = com - ctr                      (so the centre of mass keeps ~1e-7 s absolute precision)
//   Mhat_n = (-1)^|n| M_n / (n! s^|n|),   M_n = sum_j m_j (y_j - com)^n   (size-scaled, sign and 1/n!
//            folded in so that M2P needs plain derivatives D_n and no per-term factors)
// In this normalisation M2M is a convolution:  Mhat_n^parent = sum_{k<=n} Mhat_k^child 2^-|k| E_{n-k},
//   E_j = prod_i e_i^{j_i}/j_i!,  e = -(com_child - com_parent)/s_parent.
// One warp per cell, lanes over the multi-indices n; one launch per level, deepest first.
#include "dsk_internal.cuh"
#include <type_traits>

#define UW 4                     // warps (cells) per block
#define UNP dsk_np(DSK_PMAX)     // 165

__constant__ uint8_t c_ea[UNP], c_eb[UNP], c_ec[UNP], c_rank[UNP];
__device__ uint8_t g_ea[UNP], g_eb[UNP], g_ec[UNP], g_rank[UNP];   // the same tables for per-lane (divergent) indexing
// M2M pair tables, one per order p = 2 .. 8 (slot p - 2): for moment n (visited heaviest first through g_m2m_perm) the entries
// k <= n packed as k_index | (n-k).a << 8 | (n-k).b << 12 | (n-k).c << 16
#define M2M_MAXPAIR 3003       // C(14, 6): pairs (k <= n, |n| <= 8)
__device__ uint32_t g_m2m_ent[7][M2M_MAXPAIR];
__device__ uint16_t g_m2m_beg[7][UNP + 1];
__device__ uint8_t g_m2m_perm[7][UNP];
__constant__ float c_sgn_invfact[UNP];   // (-1)^|n| / (a! b! c!)
__constant__ float c_invfact1[DSK_PMAX + 1];

static bool g_tables_done[DSK_MAXDEV];
static int upload_tables()
{
    bool *done = dsk_device_flag(g_tables_done);
    if (*done) return DSK_OK;
    uint8_t ea[UNP], eb[UNP], ec[UNP], rk[UNP];
    float sif[UNP], if1[DSK_PMAX + 1];
    double fact[DSK_PMAX + 1];
    fact[0] = 1.0;
    for (int i = 1; i <= DSK_PMAX; i++) fact[i] = fact[i - 1] * i;
    for (int i = 0; i <= DSK_PMAX; i++) if1[i] = (float)(1.0 / fact[i]);
    for (int l = 0; l <= DSK_PMAX; l++)
        for (int a = l; a >= 0; a--)
            for (int b = l - a; b >= 0; b--) {
                int cc = l - a - b, i = dsk_midx(a, b, cc);
                ea[i] = (uint8_t)a; eb[i] = (uint8_t)b; ec[i] = (uint8_t)cc; rk[i] = (uint8_t)l;
                sif[i] = (float)(((l & 1) ? -1.0 : 1.0) / (fact[a] * fact[b] * fact[cc]));
            }
    DSK_CUDA(cudaMemcpyToSymbol(c_ea, ea, sizeof(ea)));
    DSK_CUDA(cudaMemcpyToSymbol(c_eb, eb, sizeof(eb)));
    DSK_CUDA(cudaMemcpyToSymbol(c_ec, ec, sizeof(ec)));
    DSK_CUDA(cudaMemcpyToSymbol(c_rank, rk, sizeof(rk)));
    DSK_CUDA(cudaMemcpyToSymbol(g_ea, ea, sizeof(ea)));
    DSK_CUDA(cudaMemcpyToSymbol(g_eb, eb, sizeof(eb)));
    DSK_CUDA(cudaMemcpyToSymbol(g_ec, ec, sizeof(ec)));
    DSK_CUDA(cudaMemcpyToSymbol(g_rank, rk, sizeof(rk)));
    DSK_CUDA(cudaMemcpyToSymbol(c_sgn_invfact, sif, sizeof(sif)));
    DSK_CUDA(cudaMemcpyToSymbol(c_invfact1, if1, sizeof(if1)));
    *done = true;
    return DSK_OK;
}


// pair table for order p: each context uploads it the first time it runs that order (the contents depend on p only, so
// a second context writing the same bytes while another reads them is harmless; no state is shared on the host)
static int upload_m2m_table(dsk_ctx *c, int p)
{
    const int slot = p - 2;
    if (c->m2m_tab_mask & (1u << slot)) return DSK_OK;
    const int np = dsk_np(p);
    uint32_t ent[M2M_MAXPAIR];
    uint16_t beg[UNP + 1];
    uint8_t perm[UNP];
    int cnt[UNP], ea[UNP], eb[UNP], ec[UNP];
    for (int l = 0; l <= p; l++)
        for (int a = l; a >= 0; a--)
            for (int b = l - a; b >= 0; b--) {
                const int c = l - a - b, i = dsk_midx(a, b, c);
                ea[i] = a; eb[i] = b; ec[i] = c; cnt[i] = (a + 1) * (b + 1) * (c + 1);
            }
    int ne = 0;
    for (int n = 0; n < np; n++) {
        beg[n] = (uint16_t)ne;
        for (int ka = 0; ka <= ea[n]; ka++)
            for (int kb = 0; kb <= eb[n]; kb++)
                for (int kc = 0; kc <= ec[n]; kc++)
                    ent[ne++] = (uint32_t)dsk_midx(ka, kb, kc) | (uint32_t)(ea[n] - ka) << 8 | (uint32_t)(eb[n] - kb) << 12 |
                                (uint32_t)(ec[n] - kc) << 16;
    }
    beg[np] = (uint16_t)ne;
    for (int i = 0; i < np; i++) perm[i] = (uint8_t)i;
    for (int i = 1; i < np; i++) {            // insertion sort, heaviest moment first: a warp's 32 lanes get similar work
        const uint8_t v = perm[i];
        int j = i;
        while (j > 0 && cnt[perm[j - 1]] < cnt[v]) { perm[j] = perm[j - 1]; j--; }
        perm[j] = v;
    }
    DSK_CUDA(cudaMemcpyToSymbol(g_m2m_ent, ent, sizeof(uint32_t) * ne, sizeof(uint32_t) * M2M_MAXPAIR * slot));
    DSK_CUDA(cudaMemcpyToSymbol(g_m2m_beg, beg, sizeof(uint16_t) * (np + 1), sizeof(uint16_t) * (UNP + 1) * slot));
    DSK_CUDA(cudaMemcpyToSymbol(g_m2m_perm, perm, sizeof(uint8_t) * np, sizeof(uint8_t) * UNP * slot));
    c->m2m_tab_mask |= 1u << slot;
    return DSK_OK;
}

__device__ __forceinline__ uint32_t compact3(uint64_t x)
{   // every third bit -> 21 contiguous bits
    x &= 0x1249249249249249ull;
    x = (x | x >> 2) & 0x10c30c30c30c30c3ull;
    x = (x | x >> 4) & 0x100f00f00f00f00full;
    x = (x | x >> 8) & 0x1f0000ff0000ffull;
    x = (x | x >> 16) & 0x1f00000000ffffull;
    x = (x | x >> 32) & 0x1fffffull;
    return (uint32_t)x;
}

__device__ __forceinline__ void cell_centre(uint64_t hotkey, int level, float box, float &s, float ctr[3])
{
    uint64_t prefix = hotkey & ~(1ull << (3 * level));
    s = box * exp2f((float)-level);
    ctr[0] = ((float)compact3(prefix >> 2) + 0.5f) * s;
    ctr[1] = ((float)compact3(prefix >> 1) + 0.5f) * s;
    ctr[2] = ((float)compact3(prefix) + 0.5f) * s;
}

__device__ __forceinline__ float warp_sum(float v)
{
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// scratch of one warp
template <int P> struct up_smem {
    float crow[8][dsk_np(P) | 1]; // the children's moments, pre-scaled by 2^-|k| (odd stride: children on distinct banks)
    float pw[8][3][12];           // per child: e_d^j / j!
};

// multi-index helpers for compile-time unrolled monomials (same scheme as the M2P body)
struct UMI { int a, b, c; };
__host__ __device__ constexpr UMI up_mi(int i)
{
    int l = 0;
    while ((l + 1) * (l + 2) * (l + 3) / 6 <= i) l++;
    int rem = i - l * (l + 1) * (l + 2) / 6, k = 0;
    while ((k + 1) * (k + 2) / 2 <= rem) k++;
    int c = rem - k * (k + 1) / 2;
    return UMI{l - k, k - c, c};
}
template <int I, int N, typename F>
__device__ __forceinline__ void up_static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        up_static_for<I + 1, N>(f);
    }
}

// One warp computes one cell.  P2M: one particle per lane and round, all N_p monomials in registers, one
// shuffle reduction per moment at the end.  M2M: the (child, moment) pairs are spread over the lanes.
template <int P>
__device__ __forceinline__ void upward_cell(uint32_t c, int level, float box, const dsk_cellrec *__restrict__ cell,
                                            const uint64_t *__restrict__ hotkey, const float4 *__restrict__ spos,
                                            float *__restrict__ rows, float4 *__restrict__ whdr, up_smem<P> &sm)
{
    constexpr int NP = dsk_np(P), ROW = dsk_rowlen(P);
    const int lane = threadIdx.x & 31;
    const dsk_cellrec r = cell[c];
    const int nchild = r.meta & 255;
    float s, ctr[3];
    cell_centre(hotkey[c], level, box, s, ctr);
    const float sinv = 1.0f / s;
    float M, off[3];
    float *row = rows + (size_t)c * ROW;
    if (nchild == 0) {
        // ---- P2M ----
        float m = 0, sx = 0, sy = 0, sz = 0;
        for (uint32_t j = r.first + lane; j < r.first + r.count; j += 32) {
            const float4 q = spos[j];
            m += q.w; sx += q.w * (q.x - ctr[0]); sy += q.w * (q.y - ctr[1]); sz += q.w * (q.z - ctr[2]);
        }
        M = warp_sum(m); sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
        const float minv = M > 0.0f ? 1.0f / M : 0.0f;
        off[0] = sx * minv; off[1] = sy * minv; off[2] = sz * minv;
        float acc[NP];
#pragma unroll
        for (int n = 0; n < NP; n++) acc[n] = 0.0f;
        for (uint32_t j = r.first + lane; j < r.first + r.count; j += 32) {
            const float4 q = spos[j];
            const float u0 = ((q.x - ctr[0]) - off[0]) * sinv, u1 = ((q.y - ctr[1]) - off[1]) * sinv,
                        u2 = ((q.z - ctr[2]) - off[2]) * sinv;
            float mu[NP];
            mu[0] = q.w;
            up_static_for<1, NP>([&](auto I) {
                constexpr int i = decltype(I)::value;
                constexpr UMI n = up_mi(i);
                // multiply the lower monomial along the first non-zero axis
                if constexpr (n.a > 0) mu[i] = mu[dsk_midx(n.a - 1, n.b, n.c)] * u0;
                else if constexpr (n.b > 0) mu[i] = mu[dsk_midx(n.a, n.b - 1, n.c)] * u1;
                else mu[i] = mu[dsk_midx(n.a, n.b, n.c - 1)] * u2;
                acc[i] += mu[i];
            });
        }
        up_static_for<1, NP>([&](auto I) {
            constexpr int i = decltype(I)::value;
            const float v = warp_sum(acc[i]);
            if (lane == (i & 31)) row[8 + i] = v * c_sgn_invfact[i];
        });
        if (lane == 0) row[8] = M;
    } else {
        // ---- M2M ----
        const float sc = 0.5f * s;              // child side
        float m = 0, sx = 0, sy = 0, sz = 0, cx = 0, cy = 0, cz = 0;
        if (lane < nchild) {
            const uint32_t ch = r.child0 + lane;
            const float *cr = rows + (size_t)ch * ROW;
            const int o = (int)(hotkey[ch] & 7ull);
            m = cr[8];
            cx = ((o & 4) ? 0.5f : -0.5f) * sc + cr[4];        // child com - parent centre
            cy = ((o & 2) ? 0.5f : -0.5f) * sc + cr[5];
            cz = ((o & 1) ? 0.5f : -0.5f) * sc + cr[6];
            sx = m * cx; sy = m * cy; sz = m * cz;
        }
        M = warp_sum(m); sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
        const float minv = M > 0.0f ? 1.0f / M : 0.0f;
        off[0] = sx * minv; off[1] = sy * minv; off[2] = sz * minv;
        // powers of e = -(com_child - com_parent)/s_parent, divided by j!
        if (lane < nchild) {
            const float e[3] = {-(cx - off[0]) * sinv, -(cy - off[1]) * sinv, -(cz - off[2]) * sinv};
#pragma unroll
            for (int d = 0; d < 3; d++) {
                float v = 1.0f;
                for (int j = 0; j <= P; j++) { sm.pw[lane][d][j] = v * c_invfact1[j]; v *= e[d]; }
            }
        }
        for (int i = lane; i < nchild * NP; i += 32) {
            const int k = i / NP, n = i - k * NP;
            sm.crow[k][n] = rows[(size_t)(r.child0 + k) * ROW + 8 + n] * exp2f(-(float)g_rank[n]);
        }
        __syncwarp();
        // lane = (moment slot, child): 4 moments per round, heaviest first so the 4 have similar pair counts; the
        // pairs (k <= n) come from the table (no index arithmetic) and the 8 children are summed by 3 shuffles
        {
            const int ch = lane & 7;
            const bool live = ch < nchild;
            const float *cr = sm.crow[live ? ch : 0];
            const float *px = sm.pw[live ? ch : 0][0], *py = sm.pw[live ? ch : 0][1], *pz = sm.pw[live ? ch : 0][2];
            for (int q0 = 0; q0 < NP; q0 += 4) {
                const int q = q0 + (lane >> 3);
                const int n = g_m2m_perm[P - 2][q < NP ? q : NP - 1];
                const int t1 = (q < NP && live) ? g_m2m_beg[P - 2][n + 1] : 0;
                float sum = 0.0f;
                for (int t = g_m2m_beg[P - 2][n]; t < t1; t++) {
                    const uint32_t e = g_m2m_ent[P - 2][t];
                    sum = fmaf(cr[e & 255u], px[(e >> 8) & 15u] * py[(e >> 12) & 15u] * pz[(e >> 16) & 15u], sum);
                }
                sum += __shfl_xor_sync(0xffffffffu, sum, 1);
                sum += __shfl_xor_sync(0xffffffffu, sum, 2);
                sum += __shfl_xor_sync(0xffffffffu, sum, 4);
                if (ch == 0 && q < NP) row[8 + n] = (n == 0) ? M : sum;
            }
        }
        __syncwarp();
    }
    // ---- header + walk header ----
    if (lane == 0) {
        const float delta = sqrtf(off[0] * off[0] + off[1] * off[1] + off[2] * off[2]);
        row[0] = ctr[0]; row[1] = ctr[1]; row[2] = ctr[2]; row[3] = sinv;
        row[4] = off[0]; row[5] = off[1]; row[6] = off[2]; row[7] = delta;
        whdr[c] = make_float4(ctr[0] + off[0], ctr[1] + off[1], ctr[2] + off[2], delta);
    }
    for (int n = 8 + NP + lane; n < ROW; n += 32) row[n] = 0.0f;
}

// one level per launch (deep levels: many cells)
template <int P>
__global__ void __launch_bounds__(UW * 32) k_upward(uint32_t cbeg, uint32_t ncells, int level, float box,
                                                    const dsk_cellrec *__restrict__ cell,
                                                    const uint64_t *__restrict__ hotkey,
                                                    const float4 *__restrict__ spos,
                                                    float *__restrict__ rows, float4 *__restrict__ whdr)
{
    __shared__ up_smem<P> sm[UW];
    const int warp = threadIdx.x >> 5;
    const uint32_t ci = blockIdx.x * UW + warp;
    if (ci >= ncells) return;
    upward_cell<P>(cbeg + ci, level, box, cell, hotkey, spos, rows, whdr, sm[warp]);
}

// the top of the tree in ONE block: levels ltop-1 .. 0, a block barrier between levels (the levels near the
// root hold a handful of cells each; a launch per level costs ~45 us of dependent latency apiece)
#define UTOP_WARPS 8
struct up_levels { uint32_t start[DSK_KEY_LEVELS + 3]; };
template <int P>
__global__ void __launch_bounds__(UTOP_WARPS * 32) k_upward_top(up_levels lv, int ltop, float box,
                                                                const dsk_cellrec *__restrict__ cell,
                                                                const uint64_t *__restrict__ hotkey,
                                                                const float4 *__restrict__ spos,
                                                                float *__restrict__ rows, float4 *__restrict__ whdr)
{
    extern __shared__ __align__(16) unsigned char up_raw[];
    up_smem<P> *sm = reinterpret_cast<up_smem<P> *>(up_raw);
    const int warp = threadIdx.x >> 5;
    for (int l = ltop - 1; l >= 0; l--) {
        for (uint32_t c = lv.start[l] + warp; c < lv.start[l + 1]; c += UTOP_WARPS)
            upward_cell<P>(c, l, box, cell, hotkey, spos, rows, whdr, sm[warp]);
        __threadfence_block();
        __syncthreads();
    }
}

template <int P>
static int launch_upward(dsk_ctx *c, const uint32_t *lvl_start, int nlevel)
{
    // levels [0, ltop) go to the single-block kernel: as many levels from the root as hold <= 24 cells together (the root and its
    // children; with a 64-cell level in it as well a warp works through eight cells in a row: upward ms with a limit of 96 / 24 / 1 / 600
    // cells: C1 0.091 / 0.047 / 0.051 / 0.250, C2 0.195 / 0.171 / 0.178 / 0.270, C3 0.268 / 0.229 / 0.231 / 0.684, C4 4.36 / 4.24 / 4.25 / 5.36)
    int ltop = 0;
    while (ltop < nlevel && lvl_start[ltop + 1] <= 24u) ltop++;
    for (int l = nlevel - 1; l >= ltop; l--) {
        uint32_t beg = lvl_start[l], n = lvl_start[l + 1] - beg;
        if (!n) continue;
        k_upward<P><<<(n + UW - 1) / UW, UW * 32, 0, c->stream>>>(beg, n, l, c->box, c->cell, c->hotkey,
                                                                  c->spos, c->rows, c->whdr);
        DSK_COUNT(c, 1);
    }
    if (ltop > 0) {
        static bool attr_flags[DSK_MAXDEV];
        bool *attr_done = dsk_device_flag(attr_flags);
        const size_t smem = sizeof(up_smem<P>) * UTOP_WARPS;
        if (!*attr_done) {
            DSK_CUDA(cudaFuncSetAttribute(k_upward_top<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            *attr_done = true;
        }
        up_levels lv;
        for (int i = 0; i < DSK_KEY_LEVELS + 3; i++) lv.start[i] = lvl_start[i];
        k_upward_top<P><<<1, UTOP_WARPS * 32, smem, c->stream>>>(lv, ltop, c->box, c->cell, c->hotkey, c->spos, c->rows, c->whdr);
        DSK_COUNT(c, 1);
    }
    return DSK_OK;
}

int dsk_run_upward(dsk_ctx *c)
{
    int e = upload_tables();
    if (e) return e;
    e = upload_m2m_table(c, c->p);
    if (e) return e;
    const uint32_t *ls = c->hstate->lvl_start;
    int nl = (int)c->hstate->nlevel;
    cudaEventRecord(c->ev[5], c->stream);
    switch (c->p) {
    case 2: e = launch_upward<2>(c, ls, nl); break;
    case 3: e = launch_upward<3>(c, ls, nl); break;
    case 4: e = launch_upward<4>(c, ls, nl); break;
    case 5: e = launch_upward<5>(c, ls, nl); break;
    case 6: e = launch_upward<6>(c, ls, nl); break;
    case 8: e = launch_upward<8>(c, ls, nl); break;
    default: return DSK_EINVAL;
    }
    if (e) return e;
    c->frow_dip = c->periodic && c->bg;        // rows of a periodic run with background subtraction carry a dipole block
    e = dsk_run_frows(c);                      // the fixed linear map to the rows M2P reads (m2p.cu)
    if (e) return e;
    c->ntop = 0;
    if (c->frow_dip) {                         // the subtracted copies of the cells of level <= l_b (background.cu)
        e = dsk_run_bg_rows(c);
        if (e) return e;
    }
    cudaEventRecord(c->ev[6], c->stream);
    c->moments_p = c->p;
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// raw moments for parity tests: M_n = Mhat_n (-1)^|n| n! s^|n|
template <int P>
__global__ void k_get_moments(uint32_t ncell, const float *__restrict__ rows, float *__restrict__ com_mass,
                              float *__restrict__ mom, int scaled)
{
    constexpr int NP = dsk_np(P), ROW = dsk_rowlen(P);
    uint32_t c = blockIdx.x;
    if (c >= ncell) return;
    const float *row = rows + (size_t)c * ROW;
    float s = 1.0f / row[3];
    if (threadIdx.x == 0 && com_mass) {
        com_mass[4 * (size_t)c] = row[0] + row[4]; com_mass[4 * (size_t)c + 1] = row[1] + row[5];
        com_mass[4 * (size_t)c + 2] = row[2] + row[6]; com_mass[4 * (size_t)c + 3] = row[8];
    }
    if (mom)
        for (int n = threadIdx.x; n < NP; n += blockDim.x) {
            float sp = 1.0f;
            if (!scaled)
                for (int t = 0; t < c_rank[n]; t++) sp *= s;
            mom[(size_t)c * NP + n] = row[8 + n] / c_sgn_invfact[n] * sp;
        }
}

int dsk_run_get_moments(dsk_ctx *c, float *com_mass, float *moments, int scaled)
{
    uint32_t nc = c->hstate->ncell;
    switch (c->p) {
    case 2: k_get_moments<2><<<nc, 32, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    case 3: k_get_moments<3><<<nc, 32, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    case 4: k_get_moments<4><<<nc, 64, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    case 5: k_get_moments<5><<<nc, 64, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    case 6: k_get_moments<6><<<nc, 96, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    case 8: k_get_moments<8><<<nc, 192, 0, c->stream>>>(nc, c->rows, com_mass, moments, scaled); break;
    default: return DSK_EINVAL;
    }
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
