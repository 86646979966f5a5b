// tree.cu — steps T (canonical octree over the sorted keys) and G (sink groups).
// DESIGN.md O3/O5 ("The Morton ordered key labeling scheme implicitly defines the topology
// of the tree"; PAPER.md:71-73 sink cells whose particles share one interaction list).
// Integer-only: a cell (level l, prefix) owns the contiguous rank range of keys with that prefix; it is
// split iff count > NLEAF and l < 21; children = non-empty octants.  Built breadth-first, one level
// per pair of launches, so cells come out in canonical (ascending hotkey = level-major) order.
// Level sizes stay on the device (dsk_devstate.lvl_start); kernels use a fixed grid and each block
// takes a contiguous chunk of the level, which makes the child-offset scan a two-launch affair.
#include "dsk_internal.cuh"
#include <cooperative_groups.h>
namespace cg = cooperative_groups;

#define TB 256

__global__ void k_tree_init(dsk_cellrec *cell, uint64_t *hotkey, uint32_t *parent, uint32_t n,
                            dsk_devstate *st)
{
    cell[0].first = 0; cell[0].count = n; cell[0].child0 = 0; cell[0].meta = 0;
    hotkey[0] = 1ull;
    parent[0] = 0xffffffffu;
    st->ncell = 1; st->lvl_start[0] = 0; st->lvl_start[1] = 1; st->nlevel = 1; st->nleaf_cells = 0;
    for (int l = 2; l < DSK_KEY_LEVELS + 3; l++) st->lvl_start[l] = 1;
}

__device__ __forceinline__ void level_chunk(const dsk_devstate *st, int l, uint32_t &lo, uint32_t &hi)
{
    uint32_t s = st->lvl_start[l], e = st->lvl_start[l + 1], n = e - s;
    uint32_t chunk = ((n + gridDim.x - 1) / gridDim.x + TB - 1) / TB * TB;
    uint64_t a = (uint64_t)s + (uint64_t)blockIdx.x * chunk;
    lo = (uint32_t)min(a, (uint64_t)e);
    hi = (uint32_t)min(a + chunk, (uint64_t)e);
}

// (the arrays written by one phase and read by the next inside the fused kernel carry no __restrict__/const:
// they must not be read through the non-coherent path)
__device__ __forceinline__ void tree_count_level(int l, const uint64_t *__restrict__ key, const dsk_cellrec *cell,
                                                 uint32_t *nchild_tmp, uint32_t *cbounds, uint32_t *bsum,
                                                 const dsk_devstate *st, uint32_t *sh)
{
    uint32_t lo, hi;
    level_chunk(st, l, lo, hi);
    const int shift = 3 * (DSK_KEY_LEVELS - 1 - l);
    uint32_t s = 0;
    // eight lanes per cell, lane o finds the first rank whose digit is >= o: the seven binary searches of a cell
    // (20 dependent loads each near the root) run side by side instead of one after the other, and the
    // bounds are kept for the emit phase
    const int lane = threadIdx.x & 31, sub = lane & 7;
    for (uint32_t c0 = lo + (threadIdx.x >> 5) * 4; c0 < hi; c0 += TB / 8) {
        const uint32_t c = c0 + (lane >> 3);
        const bool valid = c < hi;
        dsk_cellrec r;
        r.first = 0; r.count = 0; r.child0 = 0; r.meta = 0;
        if (valid) r = cell[c];
        const bool split = valid && r.count > DSK_NLEAF && l < DSK_KEY_LEVELS;
        uint32_t b = r.first;
        if (split && sub > 0) {
            uint32_t a = r.first, e = r.first + r.count;
            while (a < e) {
                const uint32_t mid = a + ((e - a) >> 1);
                if (((key[mid] >> shift) & 7ull) < (uint64_t)sub) a = mid + 1; else e = mid;
            }
            b = a;
        }
        uint32_t nb = __shfl_down_sync(0xffffffffu, b, 1, 8);
        if (sub == 7) nb = r.first + r.count;
        const uint32_t bal = __ballot_sync(0xffffffffu, split && nb > b);
        const uint32_t nc = __popc((bal >> (lane & 24)) & 0xffu);
        if (valid) {
            cbounds[(size_t)c * 8 + sub] = b;
            if (sub == 0) { nchild_tmp[c] = nc; s += nc; }
        }
    }
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < TB / 32; w++) t += sh[w];
        bsum[blockIdx.x] = t;
    }
}

__device__ __forceinline__ void tree_emit_level(int l, const uint64_t *__restrict__ key,
                                                dsk_cellrec *cell, uint64_t *hotkey, uint32_t *parent,
                                                const uint32_t *nchild_tmp, const uint32_t *cbounds, const uint32_t *bsum,
                                                uint32_t ncell_cap, dsk_devstate *st, uint32_t *sh, uint32_t *wsum, uint32_t &s_pre,
                                                uint32_t &s_all)
{
    // offset of this block's chunk = sum of the sums of the blocks before it
    uint32_t pre = 0, all = 0;
    for (uint32_t b = threadIdx.x; b < gridDim.x; b += TB) {
        uint32_t v = bsum[b];
        all += v;
        if (b < blockIdx.x) pre += v;
    }
    for (int o = 16; o; o >>= 1) { pre += __shfl_xor_sync(0xffffffffu, pre, o); all += __shfl_xor_sync(0xffffffffu, all, o); }
    if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5] = pre; wsum[threadIdx.x >> 5] = all; }
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t p = 0, a = 0;
        for (int w = 0; w < TB / 32; w++) { p += sh[w]; a += wsum[w]; }
        s_pre = p; s_all = a;
    }
    __syncthreads();
    const uint32_t child_base = st->lvl_start[l + 1];
    const bool overflow = (uint64_t)child_base + s_all > (uint64_t)ncell_cap;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (overflow) { atomicOr(&st->status, ST_CELLOVF); }
        uint32_t tot = overflow ? 0u : s_all;
        st->lvl_start[l + 2] = child_base + tot;
        for (int k = l + 3; k < DSK_KEY_LEVELS + 3; k++) st->lvl_start[k] = child_base + tot;
        st->ncell = child_base + tot;
        if (tot) st->nlevel = l + 2;
    }
    uint32_t lo, hi;
    level_chunk(st, l, lo, hi);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t carry = s_pre;
    __syncthreads();
    for (uint32_t c0 = lo; c0 < hi; c0 += TB) {
        uint32_t c = c0 + threadIdx.x;
        uint32_t v = c < hi ? nchild_tmp[c] : 0u, x = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        uint32_t wpre = 0, tot = 0;
        for (int w = 0; w < TB / 32; w++) { uint32_t t = wsum[w]; if (w < warp) wpre += t; tot += t; }
        if (c < hi) {
            dsk_cellrec r = cell[c];
            if (v == 0 || overflow) {
                r.child0 = 0; r.meta = (uint32_t)l << 8;
                cell[c] = r;
                atomicAdd(&st->nleaf_cells, 1u);
            } else {
                uint32_t ch = child_base + carry + wpre + x - v;
                r.child0 = ch; r.meta = v | ((uint32_t)l << 8);
                cell[c] = r;
                uint32_t b[9];
#pragma unroll
                for (int o = 0; o < 8; o++) b[o] = cbounds[(size_t)c * 8 + o];
                b[8] = r.first + r.count;
                uint64_t hk = hotkey[c];
#pragma unroll
                for (int o = 0; o < 8; o++)
                    if (b[o + 1] > b[o]) {
                        dsk_cellrec k;
                        k.first = b[o]; k.count = b[o + 1] - b[o]; k.child0 = 0; k.meta = (uint32_t)(l + 1) << 8;
                        cell[ch] = k;
                        hotkey[ch] = (hk << 3) | (uint64_t)o;
                        parent[ch] = c;
                        ch++;
                    }
            }
        }
        carry += tot;
        __syncthreads();
    }
}

// T in ONE cooperative launch: all levels, a grid barrier between the count and emit phases of a level and
// between levels; the loop ends at the first level that produces no children.  (One launch pair per level
// cost 44 launches of ~15-25 us each, most of them on empty levels.)
__global__ void __launch_bounds__(TB) k_tree_build(const uint64_t *__restrict__ key, dsk_cellrec *cell,
                                                   uint64_t *hotkey, uint32_t *parent, uint32_t *nchild_tmp,
                                                   uint32_t *cbounds, uint32_t *bsum, uint32_t ncell_cap, dsk_devstate *st)
{
    __shared__ uint32_t sh[TB / 32];
    __shared__ uint32_t wsum[TB / 32];
    __shared__ uint32_t s_pre, s_all;
    cg::grid_group grid = cg::this_grid();
    for (int l = 0; l <= DSK_KEY_LEVELS; l++) {
        tree_count_level(l, key, cell, nchild_tmp, cbounds, bsum, st, sh);
        grid.sync();
        tree_emit_level(l, key, cell, hotkey, parent, nchild_tmp, cbounds, bsum, ncell_cap, st, sh, wsum, s_pre, s_all);
        grid.sync();
        const volatile dsk_devstate *vs = st;
        if (vs->lvl_start[l + 2] == vs->lvl_start[l + 1]) break;      // no cells at level l + 1
    }
}

// ---- G: groups ---------------------------------------------------------------------------------------
// a cell is a group iff count <= NCRIT and (it is the root or its parent has count > NCRIT); a leaf
// with count > NCRIT (only possible at level 21) is cut into consecutive chunks of NCRIT.  Groups tile
// [0,N) so marking their first ranks and compacting over the ranks yields them in Morton order.
__global__ void __launch_bounds__(TB) k_group_mark(const dsk_cellrec *__restrict__ cell,
                                                   const uint32_t *__restrict__ parent,
                                                   uint32_t *__restrict__ gmark, const dsk_devstate *st)
{
    uint32_t n = st->ncell;
    for (uint32_t c = blockIdx.x * TB + threadIdx.x; c < n; c += gridDim.x * TB) {
        dsk_cellrec r = cell[c];
        uint32_t nchild = r.meta & 255u;
        if (r.count <= DSK_NCRIT) {
            if (c == 0 || cell[parent[c]].count > DSK_NCRIT) gmark[r.first] = c + 1;
        } else if (nchild == 0) {
            for (uint32_t k = 0; k < r.count; k += DSK_NCRIT) gmark[r.first + k] = c + 1;
        }
    }
}

__global__ void __launch_bounds__(TB) k_group_flag(const uint32_t *__restrict__ gmark, uint32_t n,
                                                   uint32_t *__restrict__ flag)
{
    uint32_t i = blockIdx.x * TB + threadIdx.x;
    if (i < n) flag[i] = gmark[i] != 0;
}

__global__ void __launch_bounds__(TB) k_group_emit(const uint32_t *__restrict__ gmark,
                                                   const uint32_t *__restrict__ gscan, uint32_t n,
                                                   uint32_t ngroup_cap, uint32_t *__restrict__ gfirst,
                                                   uint32_t *__restrict__ gcell, dsk_devstate *st)
{
    uint32_t i = blockIdx.x * TB + threadIdx.x;
    if (i >= n) return;
    uint32_t m = gmark[i];
    if (!m) return;
    uint32_t g = gscan[i];
    if (g >= ngroup_cap) { atomicOr(&st->status, ST_CELLOVF); return; }
    gfirst[g] = i;
    gcell[g] = m - 1;
}

// one warp per group: count, exact fp32 AABB of the members
__global__ void __launch_bounds__(TB) k_group_bbox(const float4 *__restrict__ spos,
                                                   const uint32_t *__restrict__ gfirst,
                                                   uint32_t *__restrict__ gcount, float4 *__restrict__ gbox,
                                                   uint32_t *__restrict__ ntask, uint32_t n, uint32_t ngroup_cap,
                                                   const dsk_devstate *st)
{
    // more groups than the workspace holds (k_group_emit has set ST_CELLOVF, the call will fail): stay inside the arrays
    if (st->status & ST_CELLOVF) return;
    // the number of groups is known on the device only: a bounded grid strides over them (a grid sized for the capacity, N/4 groups,
    // launched 4 M blocks at 512^3 of which 3 % had a group: 3.4 of the 4.6 ms of the group phase)
    const uint32_t ng = min(st->ngroup, ngroup_cap);
    const int lane = threadIdx.x & 31;
    for (uint32_t g = (blockIdx.x * TB + threadIdx.x) >> 5; g < ng; g += gridDim.x * (TB / 32)) {
    uint32_t f = gfirst[g], e = (g + 1 < ng) ? gfirst[g + 1] : n;
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (uint32_t r = f + lane; r < e; r += 32) {
        float4 p = spos[r];
        lo[0] = fminf(lo[0], p.x); lo[1] = fminf(lo[1], p.y); lo[2] = fminf(lo[2], p.z);
        hi[0] = fmaxf(hi[0], p.x); hi[1] = fmaxf(hi[1], p.y); hi[2] = fmaxf(hi[2], p.z);
    }
    for (int o = 16; o; o >>= 1)
#pragma unroll
        for (int d = 0; d < 3; d++) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
    if (lane == 0) {
        ntask[g] = dsk_task_parts(min(e - f, (uint32_t)DSK_NCRIT));
        gcount[g] = e - f;
        gbox[2 * (size_t)g] = make_float4(lo[0], lo[1], lo[2], 0.0f);
        gbox[2 * (size_t)g + 1] = make_float4(hi[0], hi[1], hi[2], 0.0f);
    }
    }
}

// task -> (group, part) map for the warp-task force kernels
__global__ void __launch_bounds__(TB) k_task_fill(const uint32_t *__restrict__ taskoff, uint32_t *__restrict__ task,
                                                  uint32_t ngroup_cap, dsk_devstate *st)
{
    if (st->status & ST_CELLOVF) return;
    const uint32_t ng = min(st->ngroup, ngroup_cap);
    for (uint32_t g = blockIdx.x * TB + threadIdx.x; g < ng; g += gridDim.x * TB) {
        const uint32_t a = taskoff[g], b = (g + 1 < ng) ? taskoff[g + 1] : st->ntask;
        for (uint32_t k = a; k < b; k++) task[k] = (g << 2) | (k - a);
    }
}

int dsk_run_build(dsk_ctx *c)
{
    const uint32_t n = (uint32_t)c->N;
    cudaStream_t s = c->stream;
    int grid = c->nsm * 4;
    k_tree_init<<<1, 1, 0, s>>>(c->cell, c->hotkey, c->parent, n, c->dstate);
    {
        const uint64_t *key = c->key_a;
        uint32_t cap = (uint32_t)c->ncell_cap;
        void *args[] = {(void *)&key, (void *)&c->cell, (void *)&c->hotkey, (void *)&c->parent, (void *)&c->nchild_tmp,
                        (void *)&c->cbounds, (void *)&c->scan_tmp, (void *)&cap, (void *)&c->dstate};
        // blocks of the cooperative launch: every level costs two grid barriers, whose price grows with the number of blocks, and the top
        // levels have no work to share - one block per SM up to 4 M particles, more where the deep levels are wide
        // (build ms with 1 / 2 / 4 / 6 blocks per SM: C1 0.050 / 0.055 / 0.060 / 0.067, C2 0.248 / 0.276 / 0.306 / 0.325,
        //  C4 0.636 / 0.613 / 0.598 / 0.642, C5 1.92 / 1.62 / 1.43 / 1.39)
        const int bgrid = c->nsm * (c->N <= (1ll << 22) ? 1 : (c->N <= (1ll << 25) ? 4 : 6));
        DSK_CUDA(cudaLaunchCooperativeKernel((const void *)k_tree_build, dim3(bgrid), dim3(TB), args, 0, s));
    }
    cudaEventRecord(c->ev[3], s);
    // groups
    cudaMemsetAsync(c->gmark, 0, sizeof(uint32_t) * (size_t)n, s);
    k_group_mark<<<grid * 2, TB, 0, s>>>(c->cell, c->parent, c->gmark, c->dstate);
    const int nb = (int)((n + TB - 1) / TB);
    k_group_flag<<<nb, TB, 0, s>>>(c->gmark, n, c->gscan);
    dsk_exclusive_scan_u32(c, c->gscan, c->gscan, nullptr, n, &c->dstate->ngroup);
    k_group_emit<<<nb, TB, 0, s>>>(c->gmark, c->gscan, n, (uint32_t)c->ngroup_cap, c->gfirst, c->gcell, c->dstate);
    // a warp per group, striding: ngroup is read on the device (capacity N/4; usually N/60 groups)
    int64_t nwarp_blocks = (c->ngroup_cap * 32 + TB - 1) / TB;
    if (nwarp_blocks > (int64_t)c->nsm * 64) nwarp_blocks = (int64_t)c->nsm * 64;
    k_group_bbox<<<(unsigned)nwarp_blocks, TB, 0, s>>>(c->spos, c->gfirst, c->gcount, c->gbox, c->g_taskoff, n, (uint32_t)c->ngroup_cap, c->dstate);
    dsk_exclusive_scan_u32(c, c->g_taskoff, c->g_taskoff, &c->dstate->ngroup, (uint32_t)c->ngroup_cap, &c->dstate->ntask);
    int64_t fill_blocks = (c->ngroup_cap + TB - 1) / TB;
    if (fill_blocks > (int64_t)c->nsm * 32) fill_blocks = (int64_t)c->nsm * 32;
    k_task_fill<<<(unsigned)fill_blocks, TB, 0, s>>>(c->g_taskoff, c->g_task, (uint32_t)c->ngroup_cap, c->dstate);
    cudaEventRecord(c->ev[4], s);
    DSK_COUNT(c, 1 + 1 + 5);   // init, the fused level loop, mark/flag/emit/bbox/taskfill
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
