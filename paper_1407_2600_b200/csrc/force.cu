// force.cu — step F1 (P2P) and the orchestration of W(fill) + F1 + F2 over batches of groups.
// DESIGN.md O6 ("bundle a set of m source cells which have interactions in common with a
// set of n sink particles ... perform the full m x n interactions on this block"; PAPER.md:75 direct
// interactions near the leaves).  F2 (M2P) lives in m2p.cu; the task decomposition in force_task.cuh.
//
// One warp per task (force_task.cuh), two sinks per lane in the halves of packed f32x2 registers (FFMA2 is
// the only way to reach the FP32 peak with three distinct operands on sm_100, see dsk_internal.cuh); source
// tiles are staged through per-warp shared memory as (x, y, z, m) and enter as broadcast scalar operands.
// All coordinates are taken relative to the group's cell centre c_g (exact subtraction for nearby
// values), which keeps fp32 differences accurate and absorbs the periodic image shift.
//
// F1: Plummer pair, acc_i += m_j d / (|d|^2+eps^2)^(3/2), pot_i -= m_j / sqrt(...), d = x_j - x_i.
#include "force_task.cuh"

#define FW 4                 // warps (tasks) per block
#define P2P_TILE 512         // sources per warp tile

int dsk_walk_fill(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t m2p_base, uint64_t p2p_base);   // walk.cu

// ---- F1 ----------------------------------------------------------------------------------------------
template <bool POT>
__global__ void __launch_bounds__(FW * 32, 6) k_p2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic, float box, float eps2,
                                                 int rowlen, const float *__restrict__ rows,
                                                 const dsk_cellrec *__restrict__ cell, const float4 *__restrict__ spos,
                                                 const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                 const uint32_t *__restrict__ gcell, const uint32_t *__restrict__ list,
                                                 const uint64_t *__restrict__ off, uint64_t base,
                                                 const uint32_t *__restrict__ len, float4 *__restrict__ sacc,
                                                 float4 *__restrict__ sacc_lo)
{
    __shared__ __align__(16) float4 src_all[FW][P2P_TILE];        // (x, y, z, m) relative to the group centre
    const warp_task t = make_task(t0, t1, FW, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4 *src = src_all[warp];
    const float *grow = rows + (size_t)gcell[t.g] * rowlen;
    const float cgx = grow[0], cgy = grow[1], cgz = grow[2];
    const float4 ma = spos[t.sa], mb = spos[t.sb];
    const f2 X = f2_make(ma.x - cgx, mb.x - cgx), Y = f2_make(ma.y - cgy, mb.y - cgy), Z = f2_make(ma.z - cgz, mb.z - cgz);
    const f2 E2 = f2_dup(eps2);
    const uint32_t n = len[t.g];
    const uint32_t *lst = list + (off[t.g] - base);
    sink_acc A;                                               // two-float running sums (see k_m2p)
    acc_zero(A);
    // evaluate the nt staged sources against the lane's two sinks
    auto eval_tile = [&](uint32_t nt) {
        __syncwarp();
        if (t.active) {
            f2 ax = f2_dup(0.0f), ay = f2_dup(0.0f), az = f2_dup(0.0f), pot = f2_dup(0.0f);
#pragma unroll 4
            for (int k = t.sub; k < (int)nt; k += t.S) {
                const float4 s = src[k];
                const f2 dx = f2_sub(f2_dup(s.x), X), dy = f2_sub(f2_dup(s.y), Y), dz = f2_sub(f2_dup(s.z), Z);
                f2 r2 = f2_fma(dx, dx, E2);
                r2 = f2_fma(dy, dy, r2);
                r2 = f2_fma(dz, dz, r2);
                const f2 ri = f2_rsqrt(r2);
                const f2 ri2 = f2_mul(ri, ri), mri = f2_mul(f2_dup(s.w), ri), mri3 = f2_mul(mri, ri2);
                ax = f2_fma(dx, mri3, ax); ay = f2_fma(dy, mri3, ay); az = f2_fma(dz, mri3, az);
                if (POT) pot = f2_sub(pot, mri);
            }
            acc_fold(A, ax, ay, az, pot, POT);
        }
        __syncwarp();
    };
    // Staging: 32 listed leaves at a time, one per lane.  A leaf is a contiguous run of the sorted particle
    // array; its lane copies it (shifted into the group's frame) to the run's place in the tile, which is the
    // exclusive prefix sum of the run lengths.  Windows of P2P_TILE sources are evaluated in turn, a run that
    // straddles two windows is copied in two parts.
    for (uint32_t b0 = 0; b0 < n; b0 += 32) {
        uint32_t my_first = 0, cnt = 0;
        float shx = 0.0f, shy = 0.0f, shz = 0.0f;
        if (b0 + lane < n) {
            const uint32_t e = lst[b0 + lane];
            const dsk_cellrec r = cell[e & ((1u << DSK_CELL_BITS) - 1u)];
            my_first = r.first; cnt = r.count;
            if (periodic) {
                const int img = (int)(e >> DSK_CELL_BITS), side = 2 * DSK_WS + 1;
                shz = (float)(img % side - DSK_WS) * box;
                shy = (float)((img / side) % side - DSK_WS) * box;
                shx = (float)(img / (side * side) - DSK_WS) * box;
            }
        }
        uint32_t x = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        const uint32_t total = __shfl_sync(0xffffffffu, x, 31), pref = x - cnt;
        for (uint32_t lo = 0; lo < total; lo += P2P_TILE) {
            const uint32_t hi = min(lo + (uint32_t)P2P_TILE, total);
            const uint32_t i0 = max(pref, lo) - pref, i1 = min(pref + cnt, hi) > pref ? min(pref + cnt, hi) - pref : 0u;
            for (uint32_t i = i0; i < i1; i++) {
                const float4 p = spos[my_first + i];
                src[pref + i - lo] = make_float4((p.x - cgx) + shx, (p.y - cgy) + shy, (p.z - cgz) + shz, p.w);
            }
            eval_tile(hi - lo);
        }
    }
    // the sink's own leaf is always in the list: remove its self term -m_i/eps from the potential (once)
    if (POT && t.active && t.sub == 0) {
        dsk_fold(A.hi[0].w, A.lo[0].w, ma.w * rsqrtf(eps2));
        dsk_fold(A.hi[1].w, A.lo[1].w, mb.w * rsqrtf(eps2));
    }
    __syncwarp();
    task_store(t, A, reinterpret_cast<double *>(src), sacc, sacc_lo);
}

static int eval_batch(dsk_ctx *c, uint32_t g0, uint32_t g1, uint32_t t0, uint32_t t1, uint64_t mb, uint64_t pb,
                      int want_pot, bool fill)
{
    cudaStream_t s = c->stream;
    if (fill) {
        int e = dsk_walk_fill(c, g0, g1, mb, pb);
        if (e) return e;
    }
    cudaEventRecord(c->ev[8], s);
    const float e2 = c->eps * c->eps;
    const int rowlen = dsk_frow_len(c->p);
    {
        int e = dsk_order_tasks(c, t0, t1, c->g_p2p_src, 6);      // longest first (m2p.cu)
        if (e) return e;
    }
    if (want_pot)
        k_p2p<true><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, s>>>(t0, t1, c->g_task_sorted, c->periodic, c->box, e2, rowlen, c->frows, c->cell, c->spos, c->gfirst,
                                           c->gcount, c->gcell, c->list_p2p, c->g_p2p_off, pb, c->g_p2p_len, c->sacc, c->sacc_lo);
    else
        k_p2p<false><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, s>>>(t0, t1, c->g_task_sorted, c->periodic, c->box, e2, rowlen, c->frows, c->cell, c->spos, c->gfirst,
                                            c->gcount, c->gcell, c->list_p2p, c->g_p2p_off, pb, c->g_p2p_len, c->sacc, c->sacc_lo);
    cudaEventRecord(c->ev[9], s);
    {
        int e = dsk_launch_m2p(c, t0, t1, mb, want_pot);
        if (e) return e;
    }
    cudaEventRecord(c->ev[10], s);
    DSK_COUNT(c, 2);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

static void add_ms(cudaEvent_t a, cudaEvent_t b, float *acc)
{
    float ms = 0.0f;
    if (cudaEventElapsedTime(&ms, a, b) == cudaSuccess) *acc += ms;
    else cudaGetLastError();      // an event that was never recorded: not an error of the path
}

// W (fill) + F1 + F2 over all groups, in one batch when the lists fit, else in batches of groups.
// Expects dsk_run_walk (COUNT + offsets) to have been enqueued unless the cached lists are valid.
int dsk_run_force(dsk_ctx *c, int want_pot)
{
    cudaStream_t s = c->stream;
    const uint32_t ng = c->hstate->ngroup;
    const bool reuse = c->lists_valid && c->lists_theta == c->theta;
    c->stats.ms_p2p = c->stats.ms_m2p = 0.0f;
    if (reuse) {
        int e = eval_batch(c, 0, ng, 0, c->hstate->ntask, 0, 0, want_pot, false);
        if (e) return e;
        DSK_CUDA(cudaStreamSynchronize(s));
        add_ms(c->ev[8], c->ev[9], &c->stats.ms_p2p);
        add_ms(c->ev[9], c->ev[10], &c->stats.ms_m2p);
        c->stats.ms_walk = 0.0f;
        return DSK_OK;
    }
    c->stats.ms_walk = 0.0f;
    // totals of the COUNT pass
    uint64_t tot[2];
    DSK_CUDA(cudaMemcpyAsync(&tot[0], c->g_m2p_off + ng, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaMemcpyAsync(&tot[1], c->g_p2p_off + ng, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaStreamSynchronize(s));
    // reset the interaction counters (filled by the FILL pass)
    DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_m2p_list, 0, sizeof(unsigned long long) * 5, s));
    if (tot[0] <= c->list_m2p_cap && tot[1] <= c->list_p2p_cap) {
        int e = eval_batch(c, 0, ng, 0, c->hstate->ntask, 0, 0, want_pot, true);
        if (e) return e;
        DSK_CUDA(cudaStreamSynchronize(s));
        add_ms(c->ev[7], c->ev[8], &c->stats.ms_walk);
        add_ms(c->ev[8], c->ev[9], &c->stats.ms_p2p);
        add_ms(c->ev[9], c->ev[10], &c->stats.ms_m2p);
        c->stats.nbatch = 1;
        c->lists_valid = 1; c->lists_theta = c->theta;
        return DSK_OK;
    }
    // batches: cut the group range where either list would overflow
    uint64_t *hm = (uint64_t *)malloc(sizeof(uint64_t) * ((size_t)ng + 1) * 2 + sizeof(uint32_t) * ((size_t)ng + 1));
    if (!hm) return DSK_ECUDA;
    uint64_t *hp = hm + ng + 1;
    uint32_t *ht = (uint32_t *)(hp + ng + 1);
    cudaMemcpyAsync(ht, c->g_taskoff, sizeof(uint32_t) * (size_t)ng, cudaMemcpyDeviceToHost, s);
    ht[ng] = c->hstate->ntask;
    cudaMemcpyAsync(hm, c->g_m2p_off, sizeof(uint64_t) * ((size_t)ng + 1), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(hp, c->g_p2p_off, sizeof(uint64_t) * ((size_t)ng + 1), cudaMemcpyDeviceToHost, s);
    if (cudaStreamSynchronize(s) != cudaSuccess) { free(hm); return DSK_ECUDA; }
    uint32_t g0 = 0;
    int nb = 0, rc = DSK_OK;
    while (g0 < ng) {
        uint32_t g1 = g0;
        while (g1 < ng && hm[g1 + 1] - hm[g0] <= c->list_m2p_cap && hp[g1 + 1] - hp[g0] <= c->list_p2p_cap) g1++;
        if (g1 == g0) { rc = DSK_ELISTOVERFLOW; break; }           // one group alone does not fit
        cudaEventRecord(c->ev[11], s);
        rc = eval_batch(c, g0, g1, ht[g0], ht[g1], hm[g0], hp[g0], want_pot, true);
        if (rc) break;
        if (cudaStreamSynchronize(s) != cudaSuccess) { rc = DSK_ECUDA; break; }
        add_ms(c->ev[11], c->ev[8], &c->stats.ms_walk);
        add_ms(c->ev[8], c->ev[9], &c->stats.ms_p2p);
        add_ms(c->ev[9], c->ev[10], &c->stats.ms_m2p);
        g0 = g1; nb++;
    }
    free(hm);
    c->stats.nbatch = nb;
    c->lists_valid = 0;
    return rc;
}
