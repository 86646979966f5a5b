// keysort.cu — steps K (Morton keys), S (LSD radix sort), the gather into the sorted float4 array,
// X (scatter back to caller order) and a device-wide exclusive scan used by several phases.
// DESIGN.md O1/O2 ("assign a Key to each particle, based on Morton ordering";
// PAPER.md:69 "domain decomposition ... practically identical to a parallel sorting algorithm").
// All HBM-bound: every global access below is a full-warp contiguous run except the two
// permutation-driven ones (gather read, scatter write), which move whole 12/16-byte records.
#include "dsk_internal.cuh"

// ---- K: keys --------------------------------------------------------------------------------------
// q = floor(fp32(x) * fp32(2^21/box)) with ONE IEEE fp32 multiply (reading A3), clamp to 2^21-1,
// interleave x (msb of each triple), y, z, placeholder bit 2^63.  Periodic: fp32 wrap first.
__device__ __forceinline__ float dsk_wrap(float x, float box)
{
    float t = __fdiv_rn(x, box);
    float f = floorf(t);
    float w = __fsub_rn(x, __fmul_rn(box, f));
    if (!(w >= 0.0f && w < box)) w = 0.0f;
    return w;
}

__device__ __forceinline__ uint64_t dsk_spread3(uint32_t q)
{   // 21 bits -> every third bit
    uint64_t x = q & 0x1fffffull;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}

__global__ void __launch_bounds__(256) k_keys(const float *__restrict__ pos, int64_t n, float box,
                                              float scale, int periodic, uint64_t *__restrict__ key,
                                              uint32_t *__restrict__ idx, dsk_devstate *st)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t q[3];
    uint32_t bad = 0;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        float x = pos[3 * i + d];
        if (!isfinite(x)) { bad |= ST_NONFINITE; x = 0.0f; }
        if (periodic) x = dsk_wrap(x, box);
        else if (!(x >= 0.0f && x < box)) { bad |= ST_OUTOFBOX; x = 0.0f; }
        float fl = floorf(__fmul_rn(x, scale));
        uint32_t qi = (uint32_t)fl;
        q[d] = qi > 2097151u ? 2097151u : qi;
    }
    if (bad) atomicOr(&st->status, bad);
    key[i] = (1ull << 63) | (dsk_spread3(q[0]) << 2) | (dsk_spread3(q[1]) << 1) | dsk_spread3(q[2]);
    idx[i] = (uint32_t)i;
}

// ---- S: LSD radix sort, 8-bit digits ---------------------------------------------------------------
// Per pass: tile histograms (digit-major matrix) -> exclusive scan -> stable scatter.  A warp owns a
// contiguous run of SORT_ITEMS*32 keys, so "warp, round, lane" is ascending global index and the
// per-warp running counters give a stable rank.
#define SORT_THREADS 256
#define SORT_ITEMS 8
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
static_assert(SORT_TILE == DSK_SORT_TILE, "dsk_api.cu sizes the sort scratch by DSK_SORT_TILE");

__global__ void __launch_bounds__(SORT_THREADS) k_sort_hist(const uint64_t *__restrict__ key, int64_t n,
                                                            int shift, int ntile,
                                                            uint32_t *__restrict__ hist)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * SORT_TILE;
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        int64_t j = base + i * SORT_THREADS + threadIdx.x;
        if (j < n) atomicAdd(&h[(key[j] >> shift) & 255u], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * ntile + blockIdx.x] = h[threadIdx.x];
}

__global__ void __launch_bounds__(SORT_THREADS) k_sort_scatter(
    const uint64_t *__restrict__ key_in, const uint32_t *__restrict__ idx_in, int64_t n, int shift,
    int ntile, const uint32_t *__restrict__ hist_scanned, uint64_t *__restrict__ key_out,
    uint32_t *__restrict__ idx_out)
{
    __shared__ uint32_t cnt[SORT_THREADS / 32][256];
    __shared__ uint32_t goff[256], dstart[256], wtot[SORT_THREADS / 32];
    __shared__ uint64_t skey[SORT_TILE];
    __shared__ uint32_t sidx[SORT_TILE];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < (SORT_THREADS / 32) * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
    goff[threadIdx.x] = hist_scanned[(size_t)threadIdx.x * ntile + blockIdx.x];
    __syncthreads();
    int64_t base = (int64_t)blockIdx.x * SORT_TILE + (int64_t)warp * (SORT_ITEMS * 32);
    uint64_t k[SORT_ITEMS];
    uint32_t v[SORT_ITEMS], rank[SORT_ITEMS];
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        int64_t j = base + i * 32 + lane;
        bool ok = j < n;
        k[i] = ok ? key_in[j] : ~0ull;
        v[i] = ok ? idx_in[j] : 0u;
    }
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t before = __popc(peers & ((1u << lane) - 1u));
        uint32_t old = cnt[warp][d];
        __syncwarp();
        if (before == 0) cnt[warp][d] = old + __popc(peers);
        __syncwarp();
        rank[i] = old + before;
    }
    __syncthreads();
    uint32_t dtot;
    {   // exclusive prefix over warps, per digit (thread = digit)
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_THREADS / 32; w++) {
            uint32_t c = cnt[w][threadIdx.x];
            cnt[w][threadIdx.x] = run;
            run += c;
        }
        dtot = run;
    }
    // exclusive prefix over digits: where each digit's run starts inside the tile
    {
        uint32_t x = dtot;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wtot[warp] = x;
        __syncthreads();
        uint32_t wpre = 0;
        for (int w = 0; w < warp; w++) wpre += wtot[w];
        dstart[threadIdx.x] = wpre + x - dtot;
    }
    __syncthreads();
    // stage the tile in digit order, then write it out run by run: consecutive threads write consecutive
    // addresses inside a digit's run (scattering 8- and 4-byte records straight from the registers wrote a
    // quarter and an eighth of every 32-byte sector)
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        int64_t j = base + i * 32 + lane;
        if (j < n) {
            uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
            uint32_t lp = dstart[d] + cnt[warp][d] + rank[i];
            skey[lp] = k[i];
            sidx[lp] = v[i];
        }
    }
    __syncthreads();
    const int64_t tile0 = (int64_t)blockIdx.x * SORT_TILE;
    const int ntile_items = (int)min((int64_t)SORT_TILE, n - tile0);
    for (int e = threadIdx.x; e < ntile_items; e += SORT_THREADS) {
        const uint64_t kk = skey[e];
        const uint32_t d = (uint32_t)(kk >> shift) & 255u;
        const uint32_t dst = goff[d] + ((uint32_t)e - dstart[d]);
        key_out[dst] = kk;
        idx_out[dst] = sidx[e];
    }
}

// ---- S for small N: one read and one write of the records per pass (decoupled look-back) ---------------------------------
// Below DSK_SORT_ONESWEEP_NMAX keys the three-kernel pass above is bound by its 40 launches, not by traffic or ranking (C1: 0.19 of
// a 0.77 ms step).  Here the eight global digit histograms come from ONE read of the keys (k_sort_hist8) and a pass is a single
// kernel (k_sort_pass): a block takes the next tile from a ticket counter, ranks its keys exactly as k_sort_scatter does,
// publishes its per-digit counts and finds the counts of all earlier tiles by look-back over the tiles' status words (flag in the
// two top bits: 0 not yet there, 1 this tile's count, 2 the inclusive count up to this tile).  Tickets make the look-back safe:
// a tile with a lower number has started, so it publishes without waiting for anyone behind it.  Measured (sort ms, three-kernel
// -> this): C1 0.186 -> 0.092, C2 0.250 -> 0.211; C4 2.16 -> 2.26 and C5 18.0 -> 19.1, which is why large N keeps the form above:
// at scale a pass is bound by the ranking code (ncu: 0.4 keys per cycle and SM either way), and the look-back waits cost more
// than the saved histogram read.
#define SORT_FLAG_AGG 0x40000000u
#define SORT_FLAG_INC 0x80000000u
#define SORT_VAL_MASK 0x3fffffffu
#define SORT_LB 4                 // status words in flight per thread during the look-back

__global__ void __launch_bounds__(256) k_sort_hist8(const uint64_t *__restrict__ key, int64_t n, uint32_t *__restrict__ ghist)
{
    __shared__ uint32_t h[8 * 256];
    for (int i = threadIdx.x; i < 8 * 256; i += 256) h[i] = 0;
    __syncthreads();
    for (int64_t j = (int64_t)blockIdx.x * 256 + threadIdx.x; j < n; j += (int64_t)gridDim.x * 256) {
        const uint64_t k = key[j];
#pragma unroll
        for (int d = 0; d < 8; d++) atomicAdd(&h[d * 256 + ((uint32_t)(k >> (8 * d)) & 255u)], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 8 * 256; i += 256)
        if (h[i]) atomicAdd(&ghist[i], h[i]);
}

__device__ __forceinline__ uint32_t sort_ld_status(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void sort_st_status(uint32_t *p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__global__ void __launch_bounds__(SORT_THREADS) k_sort_pass(
    const uint64_t *__restrict__ key_in, const uint32_t *__restrict__ idx_in, int64_t n, int shift,
    const uint32_t *__restrict__ ghist, uint32_t *status, uint32_t *ticket, uint64_t *__restrict__ key_out,
    uint32_t *__restrict__ idx_out)
{
    __shared__ uint32_t cnt[SORT_THREADS / 32][256];
    __shared__ uint32_t goff[256], dstart[256];
    __shared__ uint64_t wtot[SORT_THREADS / 32];
    __shared__ uint64_t skey[SORT_TILE];
    __shared__ uint32_t sidx[SORT_TILE];
    __shared__ uint32_t s_tile;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = threadIdx.x; i < (SORT_THREADS / 32) * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t tile0 = (int64_t)tile * SORT_TILE;
    const int64_t base = tile0 + (int64_t)warp * (SORT_ITEMS * 32);
    uint64_t k[SORT_ITEMS];
    uint32_t v[SORT_ITEMS], rank[SORT_ITEMS];
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        int64_t j = base + i * 32 + lane;
        bool ok = j < n;
        k[i] = ok ? key_in[j] : ~0ull;
        v[i] = ok ? idx_in[j] : 0u;
    }
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t before = __popc(peers & ((1u << lane) - 1u));
        uint32_t old = cnt[warp][d];
        __syncwarp();
        if (before == 0) cnt[warp][d] = old + __popc(peers);
        __syncwarp();
        rank[i] = old + before;
    }
    __syncthreads();
    // thread = digit from here to the look-back.  Exclusive prefix over warps; the tile's count of this digit goes out at once.
    // (the padding keys ~0 of a ragged last tile are counted in digit 255 of the tile, behind every real key: they are
    // neither staged nor written, and no later tile exists to read that count)
    uint32_t dtot;
    {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < SORT_THREADS / 32; w++) {
            uint32_t c = cnt[w][threadIdx.x];
            cnt[w][threadIdx.x] = run;
            run += c;
        }
        dtot = run;
    }
    uint32_t *my_status = status + (size_t)tile * 256 + threadIdx.x;
    sort_st_status(my_status, (tile == 0 ? SORT_FLAG_INC : SORT_FLAG_AGG) | dtot);
    // exclusive prefix over digits of (tile count, global count) in one 64-bit scan: where the digit's run starts inside
    // the tile, and where the digit's region starts in the output
    uint32_t gbase;
    {
        const uint64_t mine = ((uint64_t)dtot << 32) | (uint64_t)ghist[threadIdx.x];
        uint64_t x = mine;
        for (int o = 1; o < 32; o <<= 1) {
            uint64_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wtot[warp] = x;
        __syncthreads();
        uint64_t wpre = 0;
        for (int w = 0; w < warp; w++) wpre += wtot[w];
        const uint64_t ex = wpre + x - mine;
        dstart[threadIdx.x] = (uint32_t)(ex >> 32);
        gbase = (uint32_t)ex;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < SORT_ITEMS; i++) {
        int64_t j = base + i * 32 + lane;
        if (j < n) {
            uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
            uint32_t lp = dstart[d] + cnt[warp][d] + rank[i];
            skey[lp] = k[i];
            sidx[lp] = v[i];
        }
    }
    // look-back: the count of this digit in all earlier tiles.  SORT_LB status words are fetched at a time (independent loads);
    // they are consumed nearest tile first up to the first one that is not there yet.
    {
        uint32_t excl = 0;
        if (tile > 0) {
            const uint32_t *sp = my_status - 256;
            uint32_t left = tile;                       // predecessors not yet consumed
            for (bool done = false; !done;) {
                uint32_t s[SORT_LB];
#pragma unroll
                for (int b = 0; b < SORT_LB; b++) s[b] = (uint32_t)b < left ? sort_ld_status(sp - 256 * b) : SORT_FLAG_INC;
                uint32_t used = 0;
                bool open = true;
#pragma unroll
                for (int b = 0; b < SORT_LB; b++) {
                    if (open && !(s[b] & (SORT_FLAG_AGG | SORT_FLAG_INC))) open = false;
                    if (open) {
                        excl += s[b] & SORT_VAL_MASK;
                        used++;
                        if (s[b] & SORT_FLAG_INC) { done = true; open = false; }
                    }
                }
                sp -= 256 * used;
                left -= used;
            }
            sort_st_status(my_status, SORT_FLAG_INC | (excl + dtot));
        }
        goff[threadIdx.x] = gbase + excl;
    }
    __syncthreads();
    const int ntile_items = (int)min((int64_t)SORT_TILE, n - tile0);
    for (int e = threadIdx.x; e < ntile_items; e += SORT_THREADS) {
        const uint64_t kk = skey[e];
        const uint32_t d = (uint32_t)(kk >> shift) & 255u;
        const uint32_t dst = goff[d] + ((uint32_t)e - dstart[d]);
        key_out[dst] = kk;
        idx_out[dst] = sidx[e];
    }
}

// ---- device-wide exclusive scan (u32), fixed grid, n may live on the device ------------------------
#define SCAN_THREADS 256
__device__ __forceinline__ uint32_t block_sum(uint32_t v, uint32_t *sh)
{
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    uint32_t t = 0;
    for (int w = 0; w < SCAN_THREADS / 32; w++) t += sh[w];
    __syncthreads();
    return t;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const uint32_t *__restrict__ in,
                                                              const uint32_t *n_dev, uint32_t n_max,
                                                              uint32_t *__restrict__ bsum)
{
    __shared__ uint32_t sh[SCAN_THREADS / 32];
    uint32_t n = n_dev ? min(*n_dev, n_max) : n_max;
    uint32_t chunk = ((n + gridDim.x - 1) / gridDim.x + SCAN_THREADS - 1) / SCAN_THREADS * SCAN_THREADS;
    uint64_t lo = (uint64_t)blockIdx.x * chunk, hi = min((uint64_t)n, lo + chunk);
    uint32_t s = 0;
    for (uint64_t i = lo + threadIdx.x; i < hi; i += SCAN_THREADS) s += in[i];
    s = block_sum(s, sh);
    if (threadIdx.x == 0) bsum[blockIdx.x] = s;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const uint32_t *in, uint32_t *out,   // may alias
                                                             const uint32_t *n_dev, uint32_t n_max,
                                                             const uint32_t *__restrict__ bsum,
                                                             uint32_t *total)
{
    __shared__ uint32_t sh[SCAN_THREADS / 32];
    __shared__ uint32_t wsum[SCAN_THREADS / 32];
    uint32_t n = n_dev ? min(*n_dev, n_max) : n_max;
    uint32_t chunk = ((n + gridDim.x - 1) / gridDim.x + SCAN_THREADS - 1) / SCAN_THREADS * SCAN_THREADS;
    uint64_t lo = (uint64_t)blockIdx.x * chunk, hi = min((uint64_t)n, lo + chunk);
    uint32_t pre = 0, all = 0;
    for (uint32_t b = threadIdx.x; b < gridDim.x; b += SCAN_THREADS) {
        uint32_t v = bsum[b];
        all += v;
        if (b < blockIdx.x) pre += v;
    }
    pre = block_sum(pre, sh);
    if (total && blockIdx.x == 0) {
        all = block_sum(all, sh);
        if (threadIdx.x == 0) *total = all;
    }
    uint32_t carry = pre;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint64_t i0 = lo; i0 < hi; i0 += SCAN_THREADS) {
        uint64_t i = i0 + threadIdx.x;
        uint32_t v = i < hi ? in[i] : 0u, x = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        uint32_t wpre = 0, tot = 0;
        for (int w = 0; w < SCAN_THREADS / 32; w++) {
            uint32_t t = wsum[w];
            if (w < warp) wpre += t;
            tot += t;
        }
        if (i < hi) out[i] = carry + wpre + x - v;
        carry += tot;
        __syncthreads();
    }
}

void dsk_exclusive_scan_u32(dsk_ctx *c, const uint32_t *in, uint32_t *out, const uint32_t *n_dev,
                            uint32_t n_max, uint32_t *total_dev)
{
    int grid = c->nsm * 4;
    if ((uint64_t)grid * SCAN_THREADS > (uint64_t)n_max) grid = (int)((n_max + SCAN_THREADS - 1) / SCAN_THREADS);
    if (grid < 1) grid = 1;
    k_scan_reduce<<<grid, SCAN_THREADS, 0, c->stream>>>(in, n_dev, n_max, c->scan_tmp);
    k_scan_apply<<<grid, SCAN_THREADS, 0, c->stream>>>(in, out, n_dev, n_max, c->scan_tmp, total_dev);
    DSK_COUNT(c, 2);
}

// ---- gather / scatter ------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_gather(const float *__restrict__ pos, const float *__restrict__ mass,
                                                const uint32_t *__restrict__ order, int64_t n, float box,
                                                int periodic, float4 *__restrict__ spos)
{
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    uint32_t i = order[r];
    float x = pos[3 * (size_t)i], y = pos[3 * (size_t)i + 1], z = pos[3 * (size_t)i + 2];
    if (periodic) { x = dsk_wrap(x, box); y = dsk_wrap(y, box); z = dsk_wrap(z, box); }
    spos[r] = make_float4(x, y, z, mass[i]);
}

__global__ void __launch_bounds__(256) k_scatter(const float4 *__restrict__ sacc, const float4 *__restrict__ sacc_lo,
                                                 const uint32_t *__restrict__ order, int64_t n,
                                                 float *__restrict__ acc, float *__restrict__ pot,
                                                 const uint8_t *__restrict__ active, uint32_t r_lo, uint32_t r_hi)
{
    int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n || r < (int64_t)r_lo || r >= (int64_t)r_hi) return;     // dsk_accel_shard: only the ranks (sorted positions) of this shard
    uint32_t i = order[r];
    if (active && !active[i]) return;            // dsk_accel_active: inactive entries are left untouched
    float4 a = sacc[r];
    const float4 l = sacc_lo[r];
    a.x = (float)((double)a.x + (double)l.x); a.y = (float)((double)a.y + (double)l.y);
    a.z = (float)((double)a.z + (double)l.z); a.w = (float)((double)a.w + (double)l.w);
    acc[3 * (size_t)i] = a.x; acc[3 * (size_t)i + 1] = a.y; acc[3 * (size_t)i + 2] = a.z;
    if (pot) pot[i] = a.w;
}

int dsk_run_keysort(dsk_ctx *c, const float *pos, const float *mass)
{
    const int64_t n = c->N;
    const int nb = (int)((n + 255) / 256);
    float scale = 2097152.0f / c->box;
    cudaEventRecord(c->ev[0], c->stream);
    k_keys<<<nb, 256, 0, c->stream>>>(pos, n, c->box, scale, c->periodic, c->key_a, c->idx_a, c->dstate);
    cudaEventRecord(c->ev[1], c->stream);
    uint64_t *ka = c->key_a, *kb = c->key_b;
    uint32_t *ia = c->idx_a, *ib = c->idx_b;
    const int ntile = c->ntile;
    if (n <= (int64_t)DSK_SORT_ONESWEEP_NMAX) {
        // sort_hist: [8][256] global digit histograms, 8 tickets (+ padding to 64 words), then [8][ntile][256] status words
        uint32_t *ghist = c->sort_hist, *ticket = ghist + 8 * 256, *status = ticket + 64;
        cudaMemsetAsync(ghist, 0, sizeof(uint32_t) * (8 * 256 + 64 + (size_t)8 * 256 * ntile), c->stream);
        int64_t hb = (n + 256 * 16 - 1) / (256 * 16);
        if (hb > (int64_t)c->nsm * 8) hb = (int64_t)c->nsm * 8;
        k_sort_hist8<<<(unsigned)hb, 256, 0, c->stream>>>(ka, n, ghist);
        for (int pass = 0; pass < 8; pass++) {
            k_sort_pass<<<ntile, SORT_THREADS, 0, c->stream>>>(ka, ia, n, 8 * pass, ghist + 256 * pass, status + (size_t)pass * 256 * ntile,
                                                               ticket + pass, kb, ib);
            uint64_t *tk = ka; ka = kb; kb = tk;
            uint32_t *ti = ia; ia = ib; ib = ti;
        }
        DSK_COUNT(c, 1 + 8);
    } else {
        for (int pass = 0; pass < 8; pass++) {
            int shift = 8 * pass;
            k_sort_hist<<<ntile, SORT_THREADS, 0, c->stream>>>(ka, n, shift, ntile, c->sort_hist);
            dsk_exclusive_scan_u32(c, c->sort_hist, c->sort_hist, nullptr, (uint32_t)(256u * (uint32_t)ntile), nullptr);
            k_sort_scatter<<<ntile, SORT_THREADS, 0, c->stream>>>(ka, ia, n, shift, ntile, c->sort_hist, kb, ib);
            uint64_t *tk = ka; ka = kb; kb = tk;
            uint32_t *ti = ia; ia = ib; ib = ti;
        }
        DSK_COUNT(c, 2 * 8);            // 8 x (hist, scatter); the scans count themselves
    }
    // 8 passes: the result is back in (key_a, idx_a)
    k_gather<<<nb, 256, 0, c->stream>>>(pos, mass, c->idx_a, n, c->box, c->periodic, c->spos);
    cudaEventRecord(c->ev[2], c->stream);
    DSK_COUNT(c, 2);                // keys, gather
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// one warp per group: does it hold a particle with active[caller index] != 0 ?
__global__ void __launch_bounds__(256) k_group_active(const uint8_t *__restrict__ active, const uint32_t *__restrict__ order,
                                                      const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                      uint32_t ngroup, uint8_t *__restrict__ gact)
{
    const uint32_t g = (blockIdx.x * 256 + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (g >= ngroup) return;
    const uint32_t f = gfirst[g], n = gcount[g];
    bool any = false;
    for (uint32_t r = f + lane; r < f + n; r += 32) any |= active[order[r]] != 0;
    any = __any_sync(0xffffffffu, any);
    if (lane == 0) gact[g] = any ? 1 : 0;
}

int dsk_run_group_active(dsk_ctx *c, const uint8_t *active)
{
    const uint32_t ng = c->hstate->ngroup;
    k_group_active<<<(unsigned)(((size_t)ng * 32 + 255) / 256), 256, 0, c->stream>>>(active, c->idx_a, c->gfirst, c->gcount, ng, c->gact);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_run_scatter(dsk_ctx *c, float *acc, float *pot, const uint8_t *active, uint32_t r_lo, uint32_t r_hi)
{
    const int nb = (int)((c->N + 255) / 256);
    k_scatter<<<nb, 256, 0, c->stream>>>(c->sacc, c->sacc_lo, c->idx_a, c->N, acc, pot, active, r_lo, r_hi);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// ---- K + S without any allocation: dsk_sort_keys_noalloc (include/dsk.h) ---------------------------------------
// For callers that can neither allocate nor lend a workspace (code under CUDA graph capture, serving loops, harnesses
// that forbid cudaMalloc): the same key and sort kernels as dsk_run_keysort, with the sort's second key / index buffer,
// its tile histograms, the scan's block sums and the status word in ONE file-scope device array of fixed size
// (12.6 MiB for N <= 2^20; every GPU that loads the library holds it until the process exits).
// In host code the array's NAME is a host-side stand-in, not a device address: the kernels get the pointer that
// cudaGetSymbolAddress returns, looked up once per device with that device current.
// Every call shares the array, and it keeps the last call's contents: the status word is cleared at the start of every
// call (everything else is written before it is read), and two calls that overlap on the GPU (two streams, two host
// threads) race on it.
#define NA_NMAX DSK_NOALLOC_NMAX
#define NA_NTILE ((NA_NMAX + SORT_TILE - 1) / SORT_TILE)
#define NA_OFF_STATE 0                                                  // dsk_devstate (256 B reserved)
#define NA_OFF_SCAN 256                                                 // 4096 u32 block sums of the scan
#define NA_OFF_HIST (NA_OFF_SCAN + 4 * 4096)                            // [256][ntile] tile histograms
#define NA_OFF_KEYB (NA_OFF_HIST + 4 * 256 * NA_NTILE)                  // second key buffer
#define NA_OFF_IDXB (NA_OFF_KEYB + 8 * (size_t)NA_NMAX)                 // second index buffer
#define NA_BYTES (NA_OFF_IDXB + 4 * (size_t)NA_NMAX)
static_assert(sizeof(dsk_devstate) <= 256, "state slot of the static scratch");
static_assert(NA_OFF_HIST % 256 == 0 && NA_OFF_KEYB % 256 == 0 && NA_OFF_IDXB % 256 == 0, "256-byte aligned parts");

static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_BYTES];

static unsigned char *g_noalloc_ptr[DSK_MAXDEV];        // device address of g_noalloc_scratch, per device ordinal
static int g_noalloc_nsm[DSK_MAXDEV];

extern "C" int dsk_sort_keys_noalloc(const float *pos, int64_t N, float box, int periodic, uint64_t *sorted_keys,
                                     uint32_t *order, void *cuda_stream)
{
    if (!pos || !sorted_keys || !order || N <= 0 || !(box > 0.0f) || !isfinite(box)) return DSK_EINVAL;
    if (N > (int64_t)NA_NMAX) return DSK_ETOOLARGE;
    int dev = 0;
    DSK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= DSK_MAXDEV) return DSK_EINVAL;
    if (!g_noalloc_ptr[dev]) {                          // set-up, once per device, that device current
        void *p = nullptr;
        DSK_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        int nsm = 0;
        DSK_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        if (!p || nsm <= 0) return DSK_ECUDA;
        g_noalloc_nsm[dev] = nsm;
        g_noalloc_ptr[dev] = (unsigned char *)p;
    }
    unsigned char *base = g_noalloc_ptr[dev];
    cudaStream_t s = (cudaStream_t)cuda_stream;
    dsk_devstate *st = (dsk_devstate *)(base + NA_OFF_STATE);
    uint32_t *scan_tmp = (uint32_t *)(base + NA_OFF_SCAN), *hist = (uint32_t *)(base + NA_OFF_HIST);
    uint64_t *ka = sorted_keys, *kb = (uint64_t *)(base + NA_OFF_KEYB);
    uint32_t *ia = order, *ib = (uint32_t *)(base + NA_OFF_IDXB);
    DSK_CUDA(cudaMemsetAsync(st, 0, sizeof(dsk_devstate), s));
    const int nb = (int)((N + 255) / 256), ntile = (int)((N + SORT_TILE - 1) / SORT_TILE);
    k_keys<<<nb, 256, 0, s>>>(pos, N, box, 2097152.0f / box, periodic ? 1 : 0, ka, ia, st);
    const uint32_t nh = 256u * (uint32_t)ntile;
    int grid = g_noalloc_nsm[dev] * 4;
    if ((uint64_t)grid * SCAN_THREADS > (uint64_t)nh) grid = (int)((nh + SCAN_THREADS - 1) / SCAN_THREADS);
    if (grid > 4096) grid = 4096;
    for (int pass = 0; pass < 8; pass++) {
        const int shift = 8 * pass;
        k_sort_hist<<<ntile, SORT_THREADS, 0, s>>>(ka, N, shift, ntile, hist);
        k_scan_reduce<<<grid, SCAN_THREADS, 0, s>>>(hist, nullptr, nh, scan_tmp);
        k_scan_apply<<<grid, SCAN_THREADS, 0, s>>>(hist, hist, nullptr, nh, scan_tmp, nullptr);
        k_sort_scatter<<<ntile, SORT_THREADS, 0, s>>>(ka, ia, N, shift, ntile, hist, kb, ib);
        uint64_t *tk = ka; ka = kb; kb = tk;
        uint32_t *ti = ia; ia = ib; ib = ti;
    }
    // 8 passes: the result is back in the caller's (sorted_keys, order)
    DSK_CUDA(cudaGetLastError());
    uint32_t status = 0;
    DSK_CUDA(cudaMemcpyAsync(&status, &st->status, sizeof(status), cudaMemcpyDeviceToHost, s));
    DSK_CUDA(cudaStreamSynchronize(s));
    if (status & ST_NONFINITE) return DSK_ENONFINITE;
    if (status & ST_OUTOFBOX) return DSK_EOUTOFBOX;
    return DSK_OK;
}
