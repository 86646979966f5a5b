// force_task.cuh — work decomposition and small vector abstraction shared by the force kernels
// F1 (force.cu, P2P) and F2 (m2p.cu, M2P).  DESIGN.md section 5.
//
// One WARP per task; task = (group, half): sinks [32 half, 32 half + 32) of the group, so a group of <= 32
// sinks is one warp and nothing waits at a block barrier.  Groups are tree cells, so many hold few sinks
// (mean 18 of 64 on the Plummer workload): a task with ns <= 16 sinks splits the warp into S = 32 / ns
// sub-groups of W = ns lanes that take alternate source pairs of a tile; their partial sums are added at
// the end through shared memory.  Lanes >= W * S idle.
#pragma once
#include "dsk_internal.cuh"
#include <type_traits>

#define FW 4                 // warps (tasks) per block

// ---- T = f2 (two sources per op, packed f32x2) or float ----------------------------------------------
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
template <typename T> __device__ __forceinline__ T vld(const float2 *p, int half);
template <> __device__ __forceinline__ f2 vld<f2>(const float2 *p, int)
{
    f2 r;
    r.v = *reinterpret_cast<const unsigned long long *>(p);
    return r;
}
template <> __device__ __forceinline__ float vld<float>(const float2 *p, int half)
{
    return reinterpret_cast<const float *>(p)[half];
}
__device__ __forceinline__ float vsum(f2 a) { return f2_lo(a) + f2_hi(a); }
__device__ __forceinline__ float vsum(float a) { return a; }

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
    int W, S, sub, j;            // sub-group width, number of sub-groups, my sub-group, my sink in the task
    bool valid, active;          // task exists; this lane belongs to a sub-group
};
__device__ __forceinline__ warp_task make_task(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap,
                                               const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount)
{
    warp_task t;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t task = t0 + blockIdx.x * FW + warp;
    t.valid = false; t.active = false;
    t.g = 0; t.first = 0; t.ns = 0; t.W = 32; t.S = 1; t.sub = 0; t.j = 0;
    if (task >= t1) return t;
    const uint32_t m = taskmap[task], h = m & 1u;
    t.g = m >> 1;
    const uint32_t count = gcount[t.g];
    t.valid = true;
    t.ns = min(32u, count - 32u * h);
    t.first = gfirst[t.g] + 32u * h;
    t.W = (int)t.ns;
    t.S = 32 / t.W;
    t.sub = lane / t.W;
    t.active = t.sub < t.S;
    t.j = lane - t.sub * t.W;
    if (!t.active) { t.sub = 0; t.j = 0; }
    return t;
}

// Add the sub-groups' two-float accumulators (in double, through the warp's scratch: >= 32 x 4 doubles,
// 16-byte aligned, free for reuse) and store; lane j < ns owns sink j.
__device__ __forceinline__ void task_store(const warp_task &t, float4 hi, float4 lo, double *scratch,
                                           float4 *__restrict__ sacc, float4 *__restrict__ sacc_lo)
{
    const int lane = threadIdx.x & 31;
    double d[4] = {(double)hi.x + (double)lo.x, (double)hi.y + (double)lo.y, (double)hi.z + (double)lo.z,
                   (double)hi.w + (double)lo.w};
    if (t.S > 1) {
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 4; q++) scratch[q * 32 + lane] = t.active ? d[q] : 0.0;
        __syncwarp();
        if (lane < (int)t.ns)
            for (int s = 1; s < t.S; s++)
#pragma unroll
                for (int q = 0; q < 4; q++) d[q] += scratch[q * 32 + lane + s * t.W];
    }
    if (lane < (int)t.ns) {
        float4 oh, ol;
        oh.x = (float)d[0]; oh.y = (float)d[1]; oh.z = (float)d[2]; oh.w = (float)d[3];
        ol.x = (float)(d[0] - (double)oh.x); ol.y = (float)(d[1] - (double)oh.y); ol.z = (float)(d[2] - (double)oh.z);
        ol.w = (float)(d[3] - (double)oh.w);
        sacc[t.first + lane] = oh; sacc_lo[t.first + lane] = ol;
    }
}
