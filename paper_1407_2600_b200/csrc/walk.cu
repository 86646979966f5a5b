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

#ifndef WW
#define WW 1                 // warps (groups) per block: walks differ in length, a block ends with its longest
#endif
#define WRESERVE 160         // stack entries kept free for the depth-first tail (7 per level, 21 levels)
#ifndef WEPL
#define WEPL 2               // stack entries per lane and trip
#endif
#ifndef WSTACK
#define WSTACK 2048          // stack entries per warp
#endif

__device__ __forceinline__ void image_shift(int img, int periodic, float box, float sh[3])
{
    if (!periodic) { sh[0] = sh[1] = sh[2] = 0.0f; return; }
    const int side = 2 * DSK_WS + 1;
    int iz = img % side - DSK_WS, iy = (img / side) % side - DSK_WS, ix = img / (side * side) - DSK_WS;
    sh[0] = ix * box; sh[1] = iy * box; sh[2] = iz * box;
}

template <int MODE>          // 0 COUNT, 1 FILL at the scanned offsets, 2 ONE pass into a fixed capacity per group
__global__ void __launch_bounds__(WW * 32) k_walk(uint32_t g0, uint32_t g1, int periodic, float box,
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
                                                  uint64_t *__restrict__ p2p_off_out, dsk_devstate *st)
{
    constexpr bool FILL = MODE != 0;
    __shared__ uint32_t stack[WW][WSTACK];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t g = g0 + blockIdx.x * WW + warp;
    if (g >= g1) return;
    if (gact && !gact[g]) {                          // no active sink in this group (dsk_accel_active): empty lists
        if (MODE != 1 && lane == 0) {
            m2p_len[g] = 0; p2p_len[g] = 0; p2p_src[g] = 0;
            if (MODE == 2) { m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p; }
        }
        return;
    }
    const float4 blo = gbox[2 * (size_t)g], bhi = gbox[2 * (size_t)g + 1];
    uint32_t *stk = stack[warp];
    const int nimg = periodic ? (2 * DSK_WS + 1) * (2 * DSK_WS + 1) * (2 * DSK_WS + 1) : 1;
    for (int i = lane; i < nimg; i += 32) stk[i] = (uint32_t)i << DSK_CELL_BITS;   // root of every image
    __syncwarp();
    int sp = nimg;
    uint32_t nm = 0, np = 0, nsrc = 0;
    uint64_t mo = 0, po = 0;
    if (MODE == 1) { mo = m2p_off[g] - m2p_base; po = p2p_off[g] - p2p_base; }
    if (MODE == 2) { mo = (uint64_t)g * cap_m; po = (uint64_t)g * cap_p; }
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
                const uint32_t c = e[q] & ((1u << DSK_CELL_BITS) - 1u);
                h[q] = wmac[2 * (size_t)c];            // com.xyz, critical radius s/theta + delta
                rr[q] = wmac[2 * (size_t)c + 1];       // the cell record (same sector)
            }
        uint32_t push[WEPL], ptot = 0;
#pragma unroll
        for (int q = 0; q < WEPL; q++) {
            accept[q] = false; leaf[q] = false; nchild[q] = 0; child0[q] = 0;
            uint32_t cnt = 0;
            if (act[q]) {
                float sh[3];
                image_shift((int)(e[q] >> DSK_CELL_BITS), periodic, box, sh);
                const float zx = h[q].x + sh[0], zy = h[q].y + sh[1], zz = h[q].z + sh[2];
                const float dx = fmaxf(fmaxf(blo.x - zx, zx - bhi.x), 0.0f);
                const float dy = fmaxf(fmaxf(blo.y - zy, zy - bhi.y), 0.0f);
                const float dz = fmaxf(fmaxf(blo.z - zz, zz - bhi.z), 0.0f);
                const float d2 = dx * dx + dy * dy + dz * dz;
                accept[q] = d2 > h[q].w * h[q].w;
                if (!accept[q]) {
                    nchild[q] = __float_as_uint(rr[q].w) & 255u; child0[q] = __float_as_uint(rr[q].z); cnt = __float_as_uint(rr[q].y);
                    leaf[q] = nchild[q] == 0;
                }
            }
            const uint32_t bm = __ballot_sync(0xffffffffu, accept[q]);
            const uint32_t bl = __ballot_sync(0xffffffffu, leaf[q]);
            if (FILL) {
                const uint32_t im = nm + __popc(bm & lt), ip = np + __popc(bl & lt);
                if (accept[q] && (MODE == 1 || im < cap_m)) list_m2p[mo + im] = e[q];
                if (leaf[q] && (MODE == 1 || ip < cap_p)) list_p2p[po + ip] = e[q];
            }
            nm += __popc(bm); np += __popc(bl);
            if (leaf[q]) nsrc += cnt;
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
            const uint32_t img = e[q] & ~((1u << DSK_CELL_BITS) - 1u);
            for (uint32_t k = 0; k < push[q]; k++) stk[at + k] = img | (child0[q] + k);
            at += push[q];
        }
        sp += (int)tot;
        __syncwarp();
    }
    for (int o = 16; o; o >>= 1) nsrc += __shfl_xor_sync(0xffffffffu, nsrc, o);
    if (lane == 0) {
        if (MODE != 1) { m2p_len[g] = nm; p2p_len[g] = np; p2p_src[g] = nsrc; }
        if (MODE == 2) {
            m2p_off_out[g] = (uint64_t)g * cap_m; p2p_off_out[g] = (uint64_t)g * cap_p;
            if (nm > cap_m || np > cap_p) st->scratch[0] = 1ull;      // a list did not fit: the host falls back to two passes
        }
        if (FILL) {
            const unsigned long long ns = gcount[g];
            atomicAdd(&st->n_m2p, ns * nm);
            atomicAdd(&st->n_p2p, ns * nsrc);
            atomicAdd(&st->tot_m2p_list, (unsigned long long)nm);
            atomicAdd(&st->tot_p2p_list, (unsigned long long)np);
            atomicAdd(&st->tot_p2p_src, (unsigned long long)nsrc);
        }
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

// the 32 bytes the walk reads per tested cell: centre of mass and critical radius s/theta + delta | the cell record
__global__ void __launch_bounds__(256) k_walk_mac(uint32_t ncell, float box, float inv_theta,
                                                  const dsk_cellrec *__restrict__ cell, const float4 *__restrict__ whdr,
                                                  float4 *__restrict__ wmac)
{
    const uint32_t c = blockIdx.x * 256 + threadIdx.x;
    if (c >= ncell) return;
    float4 h = whdr[c];
    const int level = (int)(cell[c].meta >> 8);
    const float s = box * exp2f((float)-level);
    h.w = s * inv_theta + h.w;
    wmac[2 * (size_t)c] = h;
    // the cell record rides in the same 32-byte sector: a rejected cell needs it, and a second, dependent load would
    // double the latency of every walk iteration
    const dsk_cellrec r = cell[c];
    wmac[2 * (size_t)c + 1] = make_float4(__uint_as_float(r.first), __uint_as_float(r.count), __uint_as_float(r.child0),
                                          __uint_as_float(r.meta));
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
    k_walk_mac<<<(nc + 255) / 256, 256, 0, s>>>(nc, c->box, inv_theta, c->cell, c->whdr, c->wmac);
    DSK_COUNT(c, 1);
    c->walk_onepass = 0;
    const uint64_t cap_m = ng ? c->list_m2p_cap / ng : 0, cap_p = ng ? c->list_p2p_cap / ng : 0;
    const bool tiny = c->walk_two_pass_only == 2;          // diagnostic: capacities that overflow, to exercise the fallback
    if (cap_m >= 4096 && cap_p >= 512 && (c->onepass_bad_theta != c->theta || tiny) && c->walk_two_pass_only != 1 &&
        c->walk_two_pass_only < 3) {
        DSK_CUDA(cudaMemsetAsync(&c->dstate->tot_m2p_list, 0, sizeof(unsigned long long) * 5, s));
        DSK_CUDA(cudaMemsetAsync(&c->dstate->scratch[0], 0, sizeof(unsigned long long), s));
        const uint32_t cm = tiny ? 64u : (uint32_t)(cap_m > 0xffffff00ull ? 0xffffff00ull : cap_m),
                       cp = tiny ? 8u : (uint32_t)(cap_p > 0xffffff00ull ? 0xffffff00ull : cap_p);
        k_walk<2><<<(ng + WW - 1) / WW, WW * 32, 0, s>>>(0, ng, c->periodic, c->box, c->cell, c->wmac, c->gbox, c->gcount,
                                                         c->g_m2p_len, c->g_p2p_len, c->g_p2p_src, nullptr, nullptr, 0, 0,
                                                         c->list_m2p, c->list_p2p, c->gact_cur, cm, cp, c->g_m2p_off,
                                                         c->g_p2p_off, c->dstate);
        DSK_COUNT(c, 1);
        unsigned long long ovf = 0;
        DSK_CUDA(cudaMemcpyAsync(&ovf, &c->dstate->scratch[0], sizeof(ovf), cudaMemcpyDeviceToHost, s));
        DSK_CUDA(cudaStreamSynchronize(s));
        if (!ovf) { c->walk_onepass = 1; return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA; }
        c->onepass_bad_theta = c->theta;
    }
    k_walk<0><<<(ng + WW - 1) / WW, WW * 32, 0, s>>>(0, ng, c->periodic, c->box, c->cell, c->wmac,
                                                     c->gbox, c->gcount, c->g_m2p_len, c->g_p2p_len,
                                                     c->g_p2p_src, nullptr, nullptr, 0, 0, nullptr, nullptr,
                                                     c->gact_cur, 0, 0, nullptr, nullptr, c->dstate);
    scan64(c, c->g_m2p_len, ng, c->g_m2p_off);
    scan64(c, c->g_p2p_len, ng, c->g_p2p_off);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_walk_fill(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t m2p_base, uint64_t p2p_base)
{
    k_walk<1><<<(g1 - g0 + WW - 1) / WW, WW * 32, 0, c->stream>>>(
        g0, g1, c->periodic, c->box, c->cell, c->wmac, c->gbox, c->gcount, c->g_m2p_len,
        c->g_p2p_len, c->g_p2p_src, c->g_m2p_off, c->g_p2p_off, m2p_base, p2p_base, c->list_m2p, c->list_p2p,
        c->gact_cur, 0, 0, nullptr, nullptr, c->dstate);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
