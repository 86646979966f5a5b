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

#define UW 4                     // warps (cells) per block
#define UNP dsk_np(DSK_PMAX)     // 165

__constant__ uint8_t c_ea[UNP], c_eb[UNP], c_ec[UNP], c_rank[UNP];
__constant__ float c_sgn_invfact[UNP];   // (-1)^|n| / (a! b! c!)
__constant__ float c_invfact1[DSK_PMAX + 1];

static bool g_tables_done = false;
static int upload_tables()
{
    if (g_tables_done) return DSK_OK;
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
    DSK_CUDA(cudaMemcpyToSymbol(c_sgn_invfact, sif, sizeof(sif)));
    DSK_CUDA(cudaMemcpyToSymbol(c_invfact1, if1, sizeof(if1)));
    g_tables_done = true;
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

template <int P>
__global__ void __launch_bounds__(UW * 32) k_upward(uint32_t cbeg, uint32_t ncells, int level, float box,
                                                    const dsk_cellrec *__restrict__ cell,
                                                    const uint64_t *__restrict__ hotkey,
                                                    const float4 *__restrict__ spos,
                                                    float *__restrict__ rows, float4 *__restrict__ whdr)
{
    constexpr int NP = dsk_np(P), ROW = dsk_rowlen(P), NSLOT = (NP + 31) / 32;
    __shared__ float pw[UW][3][12];
    __shared__ float crow[UW][NP];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t ci = blockIdx.x * UW + warp;
    if (ci >= ncells) return;
    const uint32_t c = cbeg + ci;
    const dsk_cellrec r = cell[c];
    const int nchild = r.meta & 255;
    float s, ctr[3];
    cell_centre(hotkey[c], level, box, s, ctr);
    const float sinv = 1.0f / s;
    float acc[NSLOT];
#pragma unroll
    for (int k = 0; k < NSLOT; k++) acc[k] = 0.0f;
    float M, off[3];
    if (nchild == 0) {
        // ---- P2M ----
        float m = 0, sx = 0, sy = 0, sz = 0;
        for (uint32_t j = r.first + lane; j < r.first + r.count; j += 32) {
            float4 q = spos[j];
            m += q.w; sx += q.w * (q.x - ctr[0]); sy += q.w * (q.y - ctr[1]); sz += q.w * (q.z - ctr[2]);
        }
        M = warp_sum(m); sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
        float minv = M > 0.0f ? 1.0f / M : 0.0f;
        off[0] = sx * minv; off[1] = sy * minv; off[2] = sz * minv;
        for (uint32_t j = r.first; j < r.first + r.count; j++) {
            float4 q = spos[j];
            if (lane < 27) {
                int d = lane / 9, e = lane % 9;
                float x = d == 0 ? q.x : (d == 1 ? q.y : q.z);
                float u = ((x - ctr[d]) - off[d]) * sinv, v = 1.0f;
                for (int t = 0; t < e; t++) v *= u;
                pw[warp][d][e] = v;
            }
            __syncwarp();
#pragma unroll
            for (int k = 0; k < NSLOT; k++) {
                int n = lane + 32 * k;
                if (n < NP) acc[k] += q.w * pw[warp][0][c_ea[n]] * pw[warp][1][c_eb[n]] * pw[warp][2][c_ec[n]];
            }
            __syncwarp();
        }
#pragma unroll
        for (int k = 0; k < NSLOT; k++) {
            int n = lane + 32 * k;
            if (n < NP) acc[k] *= c_sgn_invfact[n];
        }
    } else {
        // ---- M2M ----
        const float sc = 0.5f * s;              // child side
        float m = 0, sx = 0, sy = 0, sz = 0;
        if (lane < nchild) {
            uint32_t ch = r.child0 + lane;
            const float *cr = rows + (size_t)ch * ROW;
            int o = (int)(hotkey[ch] & 7ull);
            m = cr[8];
            sx = m * (((o & 4) ? 0.5f : -0.5f) * sc + cr[4]);
            sy = m * (((o & 2) ? 0.5f : -0.5f) * sc + cr[5]);
            sz = m * (((o & 1) ? 0.5f : -0.5f) * sc + cr[6]);
        }
        M = warp_sum(m); sx = warp_sum(sx); sy = warp_sum(sy); sz = warp_sum(sz);
        float minv = M > 0.0f ? 1.0f / M : 0.0f;
        off[0] = sx * minv; off[1] = sy * minv; off[2] = sz * minv;
        for (int k = 0; k < nchild; k++) {
            uint32_t ch = r.child0 + k;
            const float *cr = rows + (size_t)ch * ROW;
            int o = (int)(hotkey[ch] & 7ull);
            // child moments, pre-scaled by 2^-|k|
            for (int n = lane; n < NP; n += 32) crow[warp][n] = cr[8 + n] * exp2f(-(float)c_rank[n]);
            if (lane < 27) {
                int d = lane / 9, e = lane % 9;
                int bit = d == 0 ? 4 : (d == 1 ? 2 : 1);
                float dd = ((o & bit) ? 0.5f : -0.5f) * sc + (cr[4 + d] - off[d]);   // com_child - com_parent
                float u = -dd * sinv, v = 1.0f;
                for (int t = 0; t < e; t++) v *= u;
                pw[warp][d][e] = v * c_invfact1[e];
            }
            __syncwarp();
#pragma unroll
            for (int q = 0; q < NSLOT; q++) {
                int n = lane + 32 * q;
                if (n < NP) {
                    int a = c_ea[n], b = c_eb[n], cc = c_ec[n];
                    float sum = 0.0f;
                    for (int ka = 0; ka <= a; ka++)
                        for (int kb = 0; kb <= b; kb++)
                            for (int kc = 0; kc <= cc; kc++)
                                sum += crow[warp][dsk_midx(ka, kb, kc)] * pw[warp][0][a - ka] * pw[warp][1][b - kb] *
                                       pw[warp][2][cc - kc];
                    acc[q] += sum;
                }
            }
            __syncwarp();
        }
    }
    // ---- store row + walk header ----
    float *row = rows + (size_t)c * ROW;
    if (lane == 0) {
        float delta = sqrtf(off[0] * off[0] + off[1] * off[1] + off[2] * off[2]);
        row[0] = ctr[0]; row[1] = ctr[1]; row[2] = ctr[2]; row[3] = sinv;
        row[4] = off[0]; row[5] = off[1]; row[6] = off[2]; row[7] = delta;
        whdr[c] = make_float4(ctr[0] + off[0], ctr[1] + off[1], ctr[2] + off[2], delta);
    }
#pragma unroll
    for (int k = 0; k < NSLOT; k++) {
        int n = lane + 32 * k;
        if (n < NP) row[8 + n] = (n == 0) ? M : acc[k];
    }
    for (int n = 8 + NP + lane; n < ROW; n += 32) row[n] = 0.0f;
}

template <int P>
static void launch_upward(dsk_ctx *c, const uint32_t *lvl_start, int nlevel)
{
    for (int l = nlevel - 1; l >= 0; l--) {
        uint32_t beg = lvl_start[l], n = lvl_start[l + 1] - beg;
        if (!n) continue;
        k_upward<P><<<(n + UW - 1) / UW, UW * 32, 0, c->stream>>>(beg, n, l, c->box, c->cell, c->hotkey,
                                                                  c->spos, c->rows, c->whdr);
        DSK_COUNT(c, 1);
    }
}

int dsk_run_upward(dsk_ctx *c)
{
    int e = upload_tables();
    if (e) return e;
    const uint32_t *ls = c->hstate->lvl_start;
    int nl = (int)c->hstate->nlevel;
    cudaEventRecord(c->ev[5], c->stream);
    switch (c->p) {
    case 2: launch_upward<2>(c, ls, nl); break;
    case 4: launch_upward<4>(c, ls, nl); break;
    case 6: launch_upward<6>(c, ls, nl); break;
    case 8: launch_upward<8>(c, ls, nl); break;
    default: return DSK_EINVAL;
    }
    e = dsk_run_frows(c);                      // the fixed linear map to the rows M2P reads (m2p.cu)
    if (e) return e;
    cudaEventRecord(c->ev[6], c->stream);
    c->moments_p = c->p;
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// raw moments for parity tests: M_n = Mhat_n (-1)^|n| n! s^|n|
template <int P>
__global__ void k_get_moments(uint32_t ncell, const float *__restrict__ rows, float *__restrict__ com_mass,
                              float *__restrict__ mom)
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
            for (int t = 0; t < c_rank[n]; t++) sp *= s;
            mom[(size_t)c * NP + n] = row[8 + n] / c_sgn_invfact[n] * sp;
        }
}

int dsk_run_get_moments(dsk_ctx *c, float *com_mass, float *moments)
{
    uint32_t nc = c->hstate->ncell;
    switch (c->p) {
    case 2: k_get_moments<2><<<nc, 32, 0, c->stream>>>(nc, c->rows, com_mass, moments); break;
    case 4: k_get_moments<4><<<nc, 64, 0, c->stream>>>(nc, c->rows, com_mass, moments); break;
    case 6: k_get_moments<6><<<nc, 96, 0, c->stream>>>(nc, c->rows, com_mass, moments); break;
    case 8: k_get_moments<8><<<nc, 192, 0, c->stream>>>(nc, c->rows, com_mass, moments); break;
    default: return DSK_EINVAL;
    }
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
