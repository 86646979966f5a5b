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

#define FW 1                 // warps (tasks) per block: tasks differ in length, see m2p.cu
#ifndef P2P_MINB
#define P2P_MINB 16          // resident warps per SM the register budget is cut for
#endif
#ifndef P2P_TILE
#define P2P_TILE 384         // sources per window (two windows per warp): 16 warps x 12 KB per SM; measured 256: 1.916 ms, 320: 1.890, 384: 1.872, 416: 1.874, 512: 1.898 (13 warps) on C2
#endif

int dsk_walk_fill(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t m2p_base, uint64_t p2p_base, uint64_t left_base);   // walk.cu

// ---- F1 ----------------------------------------------------------------------------------------------
// Sources are staged as they are stored: a listed leaf is a contiguous run of the sorted (x, y, z, m) array,
// its lane copies it with ONE cp.async.bulk (TMA 1-D copy, completion on the window's mbarrier) to the run's place
// in the window, which is the exclusive prefix sum of the run lengths of the 32 leaves handled at a time.  Windows of P2P_TILE sources are
// double-buffered: the next window travels while the current one is evaluated, and the cell records of the
// next 32 leaves are already in registers, so no global latency is exposed (ncu of the synchronous version:
// 2.6 warps per issue waiting on a long scoreboard).  Differences are taken between raw coordinates (one
// rounding of the exact difference); a periodic image shift is added to the staged copy of a run in place.
__device__ __forceinline__ void cp_async16_p2p(void *smem_dst, const void *gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}

__device__ __forceinline__ uint32_t p2p_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void p2p_mbar_init(uint64_t *bar)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(p2p_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void p2p_mbar_expect(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(p2p_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void p2p_mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(p2p_smem_u32(bar)), "r"(parity) : "memory");
}
// one TMA bulk copy: a leaf's run (or the part of it inside the window), bytes a multiple of 16
__device__ __forceinline__ void p2p_bulk(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(p2p_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(p2p_smem_u32(bar)) : "memory");
}

struct leaf_batch {              // one leaf per lane
    uint32_t first, cnt, pref, total;
    uint32_t mcnt;               // sources of the run that STARTS at my leaf (my leaf + the listed leaves after it that continue it in memory), else 0
    float shx, shy, shz;
};

// K1: Dehnen's K1 compensating kernel of support h instead of Plummer softening (reading O6b of DESIGN.md): for
// u = r^2/h^2 < 1   acc = -m d / h^3 (175/16 - 147/8 u + 135/16 u^2),  pot = -(m/h)(105/32 - 175/32 u + 147/32 u^2 - 135/96 u^3),
// Newtonian beyond (eps2 then carries h^2).  Both branches are evaluated packed and the halves selected: ~27 packed instructions
// per pair instead of 13.
template <bool POT, bool K1>
__global__ void __launch_bounds__(FW * 32, P2P_MINB) k_p2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic, float box, float eps2,
                                                 const dsk_cellrec *__restrict__ cell, const float4 *__restrict__ spos,
                                                 const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                 const uint32_t *__restrict__ list,
                                                 const uint64_t *__restrict__ off, uint64_t base,
                                                 const uint32_t *__restrict__ len, float4 *__restrict__ sacc,
                                                 float4 *__restrict__ sacc_lo)
{
    __shared__ __align__(16) float4 src_all[FW][2][P2P_TILE];     // two windows of raw (x, y, z, m) per warp
    __shared__ __align__(8) uint64_t bar_all[FW][2];              // one mbarrier per window buffer
    const warp_task t = make_task(t0, t1, FW, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float4 ma = spos[t.sa], mb = spos[t.sb];
    const f2 X = f2_make(ma.x, mb.x), Y = f2_make(ma.y, mb.y), Z = f2_make(ma.z, mb.z);
    const f2 E2 = f2_dup(eps2);
    const float hinv = rsqrtf(eps2), hinv2 = hinv * hinv, hinv3 = hinv2 * hinv;       // K1: eps2 = h^2
    const uint32_t n = len[t.g];
    const uint32_t *lst = list + (off[t.g] - base);
    sink_acc A;                                               // two-float running sums (see k_m2p)
    acc_zero(A);
    const uint32_t sinv16 = (65536u + (uint32_t)t.S - 1u) / (uint32_t)t.S;    // n / S == (n * sinv16) >> 16 for n < 1024, S <= 32

    // cell records of the 32 leaves [b0, b0 + 32) of the list, their prefix sums and image shifts
    auto load_batch = [&](uint32_t b0) {
        leaf_batch L;
        L.first = 0; L.cnt = 0; L.shx = L.shy = L.shz = 0.0f;
        uint32_t img = 0;
        if (b0 + lane < n) {
            const uint32_t e = lst[b0 + lane];
            img = e >> DSK_CELL_BITS;
            const dsk_cellrec r = cell[e & ((1u << DSK_CELL_BITS) - 1u)];
            L.first = r.first; L.cnt = r.count;
            if (periodic) {
                const int im = (int)img, side = 2 * DSK_WS + 1;
                L.shz = (float)(im % side - DSK_WS) * box;
                L.shy = (float)((im / side) % side - DSK_WS) * box;
                L.shx = (float)(im / (side * side) - DSK_WS) * box;
            }
        }
        uint32_t x = L.cnt;
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        L.total = __shfl_sync(0xffffffffu, x, 31);
        L.pref = x - L.cnt;
        // Runs: the walk emits sibling leaves next to each other, and siblings are neighbours in the sorted array, so
        // a leaf that starts where the previous lane's leaf ends (same image) continues its run and ONE bulk copy
        // moves the whole run (the copies are issued one lane at a time, ~10 instructions each).
        const uint32_t pend = __shfl_up_sync(0xffffffffu, L.first + L.cnt, 1), pimg = __shfl_up_sync(0xffffffffu, img, 1);
        const bool head = L.cnt != 0u && (lane == 0 || pend != L.first || pimg != img);
        const uint32_t heads = __ballot_sync(0xffffffffu, head);
        const uint32_t above = lane < 31 ? heads >> (lane + 1) : 0u;
        const int nh = above ? lane + __ffs((int)above) : 31;              // lane of the next run's first leaf
        const uint32_t npref = __shfl_sync(0xffffffffu, L.pref, nh);
        L.mcnt = head ? (above ? npref : L.total) - L.pref : 0u;
        return L;
    };
    // my part of window [lo, lo + P2P_TILE) of batch L: particles [i0, i1) of my leaf
    auto my_part = [&](const leaf_batch &L, uint32_t lo, uint32_t &i0, uint32_t &i1) {
        const uint32_t hi = min(lo + (uint32_t)P2P_TILE, L.total), e = min(L.pref + L.cnt, hi);
        i0 = max(L.pref, lo) - L.pref;
        i1 = e > L.pref ? e - L.pref : 0u;
    };
    // copy window [lo, lo + P2P_TILE) of batch L into buffer b: one cp.async.bulk per leaf run (a per-particle
    // LDGSTS loop kept 3.8 of 32 lanes busy and made 16 % of the kernel's instructions)
    auto issue = [&](const leaf_batch &L, uint32_t lo, int b) {
        const uint32_t hiw = min(lo + (uint32_t)P2P_TILE, L.total), ew = min(L.pref + L.mcnt, hiw);
        const uint32_t i0 = max(L.pref, lo) - L.pref, i1 = ew > L.pref ? ew - L.pref : 0u;      // my run's part of the window
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // earlier generic reads of the buffer are done
        if (lane == 0) p2p_mbar_expect(&bar_all[warp][b], (min(lo + (uint32_t)P2P_TILE, L.total) - lo) * 16u);
        __syncwarp();
        if (i1 > i0) p2p_bulk(src_all[warp][b] + ((L.pref + i0) - lo), spos + L.first + i0, (i1 - i0) * 16u, &bar_all[warp][b]);
    };

    if (lane == 0) { p2p_mbar_init(&bar_all[warp][0]); p2p_mbar_init(&bar_all[warp][1]); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncwarp();
    uint32_t phase = 0;                           // bit b: parity of the next completion of buffer b's mbarrier
    leaf_batch cur = load_batch(0), nxt = load_batch(32);
    uint32_t bcur = 0, lo = 0;                    // current window: batch at list position bcur, offset lo
    int buf = 0;
    if (cur.total) issue(cur, 0, 0);
    while (bcur < n) {
        // the window after this one
        const bool same = lo + (uint32_t)P2P_TILE < cur.total;
        p2p_mbar_wait(&bar_all[warp][buf], (phase >> buf) & 1u);
        phase ^= 1u << buf;
        float4 *src = src_all[warp][buf];
        const uint32_t nt = min((uint32_t)P2P_TILE, cur.total - lo);
        if (periodic && (cur.shx != 0.0f || cur.shy != 0.0f || cur.shz != 0.0f)) {
            uint32_t i0, i1;
            my_part(cur, lo, i0, i1);
            for (uint32_t i = i0; i < i1; i++) {
                float4 v = src[cur.pref - lo + i];
                v.x += cur.shx; v.y += cur.shy; v.z += cur.shz;
                src[cur.pref - lo + i] = v;
            }
        }
        __syncwarp();
        if (same) {
            issue(cur, lo + P2P_TILE, buf ^ 1);
        } else if (bcur + 32 < n) {
            issue(nxt, 0, buf ^ 1);
        }
        if (t.active && cur.total) {
            f2 ax = f2_dup(0.0f), ay = f2_dup(0.0f), az = f2_dup(0.0f), pot = f2_dup(0.0f);
            auto pair = [&](const float4 s) {
                const f2 dx = f2_sub(f2_dup(s.x), X), dy = f2_sub(f2_dup(s.y), Y), dz = f2_sub(f2_dup(s.z), Z);
                if constexpr (K1) {
                    f2 r2 = f2_mul(dx, dx);
                    r2 = f2_fma(dy, dy, r2);
                    r2 = f2_fma(dz, dz, r2);
                    const f2 u = f2_mul(r2, f2_dup(hinv2));
                    const f2 rs = f2_make(rsqrtf(fmaxf(f2_lo(r2), 1e-37f)), rsqrtf(fmaxf(f2_hi(r2), 1e-37f)));
                    const f2 n3 = f2_mul(f2_mul(rs, rs), rs);
                    const f2 pf = f2_mul(f2_fma(f2_fma(f2_dup(8.4375f), u, f2_dup(-18.375f)), u, f2_dup(10.9375f)), f2_dup(hinv3));
                    const bool in_lo = f2_lo(u) < 1.0f, in_hi = f2_hi(u) < 1.0f;
                    const f2 f = f2_make(in_lo ? f2_lo(pf) : f2_lo(n3), in_hi ? f2_hi(pf) : f2_hi(n3));
                    const f2 mf = f2_mul(f2_dup(s.w), f);
                    ax = f2_fma(dx, mf, ax); ay = f2_fma(dy, mf, ay); az = f2_fma(dz, mf, az);
                    if (POT) {
                        const f2 pp = f2_mul(f2_fma(f2_fma(f2_fma(f2_dup(-1.40625f), u, f2_dup(4.59375f)), u, f2_dup(-5.46875f)), u, f2_dup(3.28125f)),
                                             f2_dup(hinv));
                        const f2 ph = f2_make(in_lo ? f2_lo(pp) : f2_lo(rs), in_hi ? f2_hi(pp) : f2_hi(rs));
                        pot = f2_sub(pot, f2_mul(f2_dup(s.w), ph));
                    }
                    return;
                }
                f2 r2 = f2_fma(dx, dx, E2);
                r2 = f2_fma(dy, dy, r2);
                r2 = f2_fma(dz, dz, r2);
                const f2 ri = f2_rsqrt(r2);
                const f2 ri2 = f2_mul(ri, ri), mri = f2_mul(f2_dup(s.w), ri), mri3 = f2_mul(mri, ri2);
                ax = f2_fma(dx, mri3, ax); ay = f2_fma(dy, mri3, ay); az = f2_fma(dz, mri3, az);
                if (POT) pot = f2_sub(pot, mri);
            };
            // my sub-group's sources: src[sub], src[sub + S], ...; pointer stepping keeps index arithmetic out of the loop
            const float4 *q = src + t.sub;
            const int S1 = t.S, S2 = 2 * t.S, S3 = 3 * t.S, S4 = 4 * t.S;
            int left = (int)(((nt - (uint32_t)t.sub + (uint32_t)t.S - 1u) * sinv16) >> 16);   // = ceil((nt - sub) / S), nt <= P2P_TILE < 1024
            for (; left >= 4; left -= 4, q += S4) {
                const float4 s0 = q[0], s1 = q[S1], s2 = q[S2], s3 = q[S3];
                pair(s0); pair(s1); pair(s2); pair(s3);
            }
            for (; left > 0; left--, q += S1) pair(q[0]);
            acc_fold(A, ax, ay, az, pot, POT);
        }
        __syncwarp();
        if (same) {
            lo += P2P_TILE;
        } else {
            bcur += 32; lo = 0;
            cur = nxt;
            nxt = load_batch(bcur + 32);
        }
        buf ^= 1;
    }
    // the sink's own leaf is always in the list: remove its self term -m_i/eps from the potential (once)
    if (POT && t.active && t.sub == 0) {
        const float self = K1 ? 3.28125f * hinv : rsqrtf(eps2);          // -m phi(0): m/eps (Plummer), (105/32) m/h (K1)
        f2_fold(A.hi[3], A.lo[3], f2_make(ma.w * self, mb.w * self));
    }
    __syncwarp();
    task_store(t, A, reinterpret_cast<double *>(src_all[warp][0]), sacc, sacc_lo);
}

// the next batch of groups [g0, g1): the longest run whose three lists fit their buffers
struct batch_cut { uint32_t g1, t0, t1, pad; uint64_t mb, pb, lb; };
__global__ void k_batch_cut(uint32_t g0, uint32_t ng, const uint64_t *__restrict__ moff, const uint64_t *__restrict__ poff,
                            const uint64_t *__restrict__ loff, const uint32_t *__restrict__ taskoff, uint32_t ntask, uint64_t cap_m,
                            uint64_t cap_p, uint64_t cap_l, batch_cut *out)
{
    // largest g1 in [g0, ng] with off[g1] - off[g0] <= cap for every list (the offsets are non-decreasing)
    uint32_t lo = g0, hi = ng;
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo + 1) >> 1);
        const bool fits = moff[mid] - moff[g0] <= cap_m && poff[mid] - poff[g0] <= cap_p && (!loff || loff[mid] - loff[g0] <= cap_l);
        if (fits) lo = mid; else hi = mid - 1;
    }
    out->g1 = lo; out->t0 = taskoff[g0]; out->t1 = lo < ng ? taskoff[lo] : ntask; out->pad = 0;
    out->mb = moff[g0]; out->pb = poff[g0]; out->lb = loff ? loff[g0] : 0;
}

static int eval_batch(dsk_ctx *c, uint32_t g0, uint32_t g1, uint32_t t0, uint32_t t1, uint64_t mb, uint64_t pb, uint64_t lb,
                      int want_pot, bool fill)
{
    cudaStream_t s = c->stream;
    if (fill) {
        int e = dsk_walk_fill(c, g0, g1, mb, pb, lb);
        if (e) return e;
        if (c->walk_predicted) {             // slots sized from the previous evaluation (walk.cu): did every list fit?
            unsigned long long ovf = 0;
            DSK_CUDA(cudaMemcpyAsync(&ovf, &c->dstate->scratch[0], sizeof(ovf), cudaMemcpyDeviceToHost, s));
            DSK_CUDA(cudaStreamSynchronize(s));
            if (ovf) return DSK_RETRY_WALK;
        }
    }
    cudaEventRecord(c->ev[8], s);
    const float e2 = c->eps * c->eps;
    {
        int e = dsk_order_tasks(c, t0, t1, c->g_p2p_src, 6);      // longest first (m2p.cu)
        if (e) return e;
    }
    {
        const unsigned grid = (t1 - t0 + FW - 1) / FW;
        auto launch = [&](auto kern) {
            kern<<<grid, FW * 32, 0, s>>>(t0, t1, c->g_task_sorted, c->periodic, c->box, e2, c->cell, c->spos, c->gfirst, c->gcount,
                                          c->list_p2p, c->g_p2p_off, pb, c->g_p2p_len, c->sacc, c->sacc_lo);
        };
        if (c->soft_kind == 1) { if (want_pot) launch(k_p2p<true, true>); else launch(k_p2p<false, true>); }
        else { if (want_pot) launch(k_p2p<true, false>); else launch(k_p2p<false, false>); }
    }
    cudaEventRecord(c->ev[9], s);
    {
        int e = dsk_launch_m2p(c, t0, t1, mb, want_pot);
        if (e) return e;
    }
    if (c->periodic && c->bg) {                      // the cubes kept outside the groups' windows (background.cu)
        int e = dsk_run_bg_left(c, g0, g1, lb, want_pot);
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
    c->pending_force_ms = 0;
    if (reuse) {
        int e = eval_batch(c, 0, ng, 0, c->hstate->ntask, 0, 0, 0, want_pot, false);
        if (e) return e;
        c->pending_force_ms = 1;                      // the event times are read after the call's one closing synchronisation (dsk_api.cu)
        c->stats.ms_walk = 0.0f;
        return DSK_OK;
    }
    c->stats.ms_walk = 0.0f;
    if (c->walk_onepass) {                        // the lists are already there (walk.cu): one batch, no FILL pass
        int e = eval_batch(c, 0, ng, 0, c->hstate->ntask, 0, 0, 0, want_pot, false);
        if (e) return e;
        c->pending_force_ms = 2;
        c->stats.nbatch = 1;
        c->lists_valid = 1; c->lists_theta = c->theta;
        return DSK_OK;
    }
    // totals of the COUNT pass
    const bool BG = c->periodic && c->bg;
    uint64_t tot[3] = {0, 0, 0};
    DSK_CUDA(cudaMemcpyAsync(&tot[0], c->g_m2p_off + ng, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaMemcpyAsync(&tot[1], c->g_p2p_off + ng, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
    if (BG) DSK_CUDA(cudaMemcpyAsync(&tot[2], c->g_left_off + ng, sizeof(uint64_t), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaStreamSynchronize(s));
    // reset the interaction counters (filled by the FILL pass)
    DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_m2p_list, 0, sizeof(unsigned long long) * 5, s));
    DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_left_list, 0, sizeof(unsigned long long), s));
    DSK_CUDA(cudaMemsetAsync(&c->dstate->scratch[0], 0, sizeof(unsigned long long), s));          // overflow flag of a predicted fill
    // diagnostic modes 3 / 4 (dsk_set_walk_mode): pretend the list buffers are small (batches on small inputs) or tiny
    // (not even one group fits: DSK_ELISTOVERFLOW)
    const size_t cap_m = c->walk_two_pass_only == 3 ? (size_t)65536 : c->walk_two_pass_only == 4 ? (size_t)256 : c->list_m2p_cap;
    const size_t cap_p = c->walk_two_pass_only == 3 ? (size_t)8192 : c->walk_two_pass_only == 4 ? (size_t)8 : c->list_p2p_cap;
    const size_t cap_l = BG ? c->list_left_cap : (size_t)1;
    if (tot[0] <= cap_m && tot[1] <= cap_p && tot[2] <= cap_l) {
        int e = eval_batch(c, 0, ng, 0, c->hstate->ntask, 0, 0, 0, want_pot, true);
        if (e) return e;
        c->pending_force_ms = 2;
        c->stats.nbatch = 1;
        c->lists_valid = !c->walk_predicted; c->lists_theta = c->theta;      // (predicted slots are not tight: the cached-list path assumes nothing about that, but keep it simple)
        if (!c->gact_cur) dsk_walk_remember(c);
        return DSK_OK;
    }
    // batches: cut the group range where a list would overflow.  The cut is found on the device (binary search over the three
    // offset arrays) and 48 bytes come back per batch: copying the offsets of 3.4 M groups to the host took 80 MB and ~10 ms per
    // evaluation at 512^3.
    batch_cut *dcut = reinterpret_cast<batch_cut *>(c->task_hist);          // scratch, free between the task sorts
    uint32_t g0 = 0;
    int nb = 0, rc = DSK_OK;
    while (g0 < ng) {
        batch_cut h;
        k_batch_cut<<<1, 1, 0, s>>>(g0, ng, c->g_m2p_off, c->g_p2p_off, BG ? c->g_left_off : nullptr, c->g_taskoff, c->hstate->ntask,
                                    (uint64_t)cap_m, (uint64_t)cap_p, (uint64_t)cap_l, dcut);
        if (cudaMemcpyAsync(&h, dcut, sizeof(h), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess) { rc = DSK_ECUDA; break; }
        const uint32_t g1 = h.g1;
        if (g1 == g0) { rc = DSK_ELISTOVERFLOW; break; }           // one group alone does not fit
        cudaEventRecord(c->ev[11], s);
        rc = eval_batch(c, g0, g1, h.t0, h.t1, h.mb, h.pb, h.lb, want_pot, true);
        if (rc) break;
        if (cudaStreamSynchronize(s) != cudaSuccess) { rc = DSK_ECUDA; break; }
        add_ms(c->ev[11], c->ev[8], &c->stats.ms_walk);
        add_ms(c->ev[8], c->ev[9], &c->stats.ms_p2p);
        add_ms(c->ev[9], c->ev[10], &c->stats.ms_m2p);
        g0 = g1; nb++;
    }
    DSK_COUNT(c, nb);
    if (rc == DSK_OK && !c->gact_cur) dsk_walk_remember(c);
    c->stats.nbatch = nb;
    c->lists_valid = 0;
    return rc;
}
