// force_task.cuh — work decomposition and small vector abstraction shared by the force kernels
// F1 (force.cu, P2P) and F2 (m2p.cu, M2P).  DESIGN.md section 5.
//
// One WARP per task, TWO SINKS PER LANE: the two fp32 halves of every packed f32x2 register belong to two
// sinks, and a source (cell coefficient, particle coordinate) enters FFMA2/FMUL2/FADD2 as a scalar operand
// broadcast to both halves (SASS "R.F32"; measured 2.2 cycles per FFMA2 per SMSP against 2.0 for three packed
// operands).  Sources therefore sit in shared memory exactly as they sit in global memory (no interleaving
// pass), one LDS.128 brings four coefficients, and a warp covers up to 64 sinks.
// Groups hold 1..NCRIT = 192 sinks (most far fewer: groups are tree cells), so a group of n sinks is cut into
// k <= 4 tasks of ~n/k sinks; a task of ns sinks uses W = ceil(ns/2) lanes per sub-group and S = 32 / W sub-groups
// that take alternate sources of a tile and are summed at the end through shared memory; k maximises the share
// of busy lanes n S / (64 k) (ncu: 29.3 of 32 threads per instruction on the Plummer workload).
#pragma once
#include "dsk_internal.cuh"
#include <type_traits>


// ---- T = f2 (two sinks per op, packed f32x2) or float ------------------------------------------------
__device__ __forceinline__ f2 vfma(f2 a, f2 b, f2 c) { return f2_fma(a, b, c); }
__device__ __forceinline__ f2 vmul(f2 a, f2 b) { return f2_mul(a, b); }
__device__ __forceinline__ f2 vadd(f2 a, f2 b) { return f2_add(a, b); }
__device__ __forceinline__ f2 vsub(f2 a, f2 b) { return f2_sub(a, b); }
__device__ __forceinline__ f2 vrsqrt(f2 a) { return f2_rsqrt(a); }
__device__ __forceinline__ float vfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float vmul(float a, float b) { return a * b; }
__device__ __forceinline__ float vadd(float a, float b) { return a + b; }
__device__ __forceinline__ float vsub(float a, float b) { return a - b; }
__device__ __forceinline__ float vrsqrt(float a) { return rsqrtf(a); }
template <typename T> __device__ __forceinline__ T vdup(float x);
template <> __device__ __forceinline__ f2 vdup<f2>(float x) { return f2_dup(x); }
template <> __device__ __forceinline__ float vdup<float>(float x) { return x; }
template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

struct MI { int a, b, c, l; };
__host__ __device__ constexpr MI dsk_mi(int i)
{
    int l = 0;
    while ((l + 1) * (l + 2) * (l + 3) / 6 <= i) l++;
    int rem = i - l * (l + 1) * (l + 2) / 6, k = 0;
    while ((k + 1) * (k + 2) / 2 <= rem) k++;
    int c = rem - k * (k + 1) / 2;
    return MI{l - k, k - c, c, l};
}

struct warp_task {
    uint32_t g, first, ns;       // group, rank of the task's first sink, sinks in the task
    int W, S, sub, j;            // lanes per sub-group, number of sub-groups, my sub-group, my lane in it
    uint32_t sa, sb;             // ranks of my two sinks (sb == sa when the task has an odd sink left over)
    bool valid, active, has_b;   // task exists; this lane belongs to a sub-group; second sink is a real one
};
// taskmap entry = group << 2 | part
__device__ __forceinline__ warp_task make_task(uint32_t t0, uint32_t t1, int fw, const uint32_t *__restrict__ taskmap,
                                               const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount)
{
    warp_task t;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t task = t0 + blockIdx.x * fw + warp;      // fw = warps (tasks) per block
    t.valid = false; t.active = false; t.has_b = false;
    t.g = 0; t.first = 0; t.ns = 0; t.W = 32; t.S = 1; t.sub = 0; t.j = 0; t.sa = t.sb = 0;
    if (task >= t1) return t;
    const uint32_t m = taskmap[task], part = m & 3u;
    t.g = m >> 2;
    uint32_t off, ns;
    dsk_task_range(gcount[t.g], part, off, ns);
    t.valid = true;
    t.ns = ns;
    t.first = gfirst[t.g] + off;
    t.W = (int)((t.ns + 1u) >> 1);
    t.S = 32 / t.W;
    t.sub = lane / t.W;
    t.active = t.sub < t.S;
    t.j = lane - t.sub * t.W;
    if (!t.active) { t.sub = 0; t.j = 0; }
    t.has_b = 2u * (uint32_t)t.j + 1u < t.ns;
    t.sa = t.first + 2u * (uint32_t)t.j;
    t.sb = t.has_b ? t.sa + 1u : t.sa;
    return t;
}

// two-float running sums of (ax, ay, az, pot) for the lane's two sinks, PACKED like the arithmetic: component c
// of both sinks in one f32x2 (lo half = sink a, hi half = sink b), so a TwoSum fold is six packed adds
struct sink_acc {
    f2 hi[4], lo[4];
};
__device__ __forceinline__ float f2_half(f2 v, int h) { return h ? f2_hi(v) : f2_lo(v); }
__device__ __forceinline__ f2 f2_with(f2 v, int h, float x) { return h ? f2_make(f2_lo(v), x) : f2_make(x, f2_hi(v)); }
__device__ __forceinline__ void acc_zero(sink_acc &a)
{
#pragma unroll
    for (int c = 0; c < 4; c++) a.hi[c] = a.lo[c] = f2_dup(0.0f);
}
__device__ __forceinline__ void acc_load(sink_acc &a, const warp_task &t, const float4 *__restrict__ sacc,
                                         const float4 *__restrict__ sacc_lo)
{
    acc_zero(a);
    if (t.active && t.sub == 0) {
        const float4 ha = sacc[t.sa], la = sacc_lo[t.sa];
        float4 hb = make_float4(0.f, 0.f, 0.f, 0.f), lb = hb;
        if (t.has_b) { hb = sacc[t.sb]; lb = sacc_lo[t.sb]; }
        a.hi[0] = f2_make(ha.x, hb.x); a.hi[1] = f2_make(ha.y, hb.y); a.hi[2] = f2_make(ha.z, hb.z); a.hi[3] = f2_make(ha.w, hb.w);
        a.lo[0] = f2_make(la.x, lb.x); a.lo[1] = f2_make(la.y, lb.y); a.lo[2] = f2_make(la.z, lb.z); a.lo[3] = f2_make(la.w, lb.w);
    }
}
// (hi, lo) += t without losing the rounding error of the addition (TwoSum), both sinks at once
__device__ __forceinline__ void f2_fold(f2 &hi, f2 &lo, f2 t)
{
    const f2 s = f2_add(hi, t);
    const f2 bb = f2_sub(s, hi);
    lo = f2_add(lo, f2_add(f2_sub(hi, f2_sub(s, bb)), f2_sub(t, bb)));
    hi = s;
}
// fold one tile's plain-fp32 sums into the running sums
__device__ __forceinline__ void acc_fold(sink_acc &a, f2 ax, f2 ay, f2 az, f2 pot, bool want_pot)
{
    f2_fold(a.hi[0], a.lo[0], ax); f2_fold(a.hi[1], a.lo[1], ay); f2_fold(a.hi[2], a.lo[2], az);
    if (want_pot) f2_fold(a.hi[3], a.lo[3], pot);
}
// scalar access: component c of sink h
__device__ __forceinline__ void acc_fold1(sink_acc &a, int h, int c, float t)
{
    float hi = f2_half(a.hi[c], h), lo = f2_half(a.lo[c], h);
    dsk_fold(hi, lo, t);
    a.hi[c] = f2_with(a.hi[c], h, hi); a.lo[c] = f2_with(a.lo[c], h, lo);
}
__device__ __forceinline__ void acc_add_double(sink_acc &a, int h, int c, double v)
{
    const double s = ((double)f2_half(a.hi[c], h) + (double)f2_half(a.lo[c], h)) + v;
    const float hi = (float)s;
    a.hi[c] = f2_with(a.hi[c], h, hi); a.lo[c] = f2_with(a.lo[c], h, (float)(s - (double)hi));
}

// Add the sub-groups' two-float accumulators (in double, through the warp's scratch: >= 32 x 8 doubles,
// 16-byte aligned, free for reuse) and store; lane j < W of sub-group 0 owns sinks 2j, 2j+1.
__device__ __forceinline__ void task_store(const warp_task &t, const sink_acc &a, double *scratch,
                                           float4 *__restrict__ sacc, float4 *__restrict__ sacc_lo)
{
    const int lane = threadIdx.x & 31;
    double d[8];
#pragma unroll
    for (int h = 0; h < 2; h++)
#pragma unroll
        for (int c = 0; c < 4; c++) d[4 * h + c] = (double)f2_half(a.hi[c], h) + (double)f2_half(a.lo[c], h);
    if (t.S > 1) {
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 8; q++) scratch[q * 32 + lane] = t.active ? d[q] : 0.0;
        __syncwarp();
        if (lane < t.W)
            for (int s = 1; s < t.S; s++)
#pragma unroll
                for (int q = 0; q < 8; q++) d[q] += scratch[q * 32 + lane + s * t.W];
    }
    if (lane < t.W) {
#pragma unroll
        for (int h = 0; h < 2; h++) {
            if (h == 1 && !t.has_b) break;
            float4 oh, ol;
            oh.x = (float)d[4 * h]; oh.y = (float)d[4 * h + 1]; oh.z = (float)d[4 * h + 2]; oh.w = (float)d[4 * h + 3];
            ol.x = (float)(d[4 * h] - (double)oh.x); ol.y = (float)(d[4 * h + 1] - (double)oh.y);
            ol.z = (float)(d[4 * h + 2] - (double)oh.z); ol.w = (float)(d[4 * h + 3] - (double)oh.w);
            const uint32_t r = h ? t.sb : t.sa;
            sacc[r] = oh; sacc_lo[r] = ol;
        }
    }
}
