// force.cu — steps F1 (P2P) and F2 (M2P): evaluation of the interaction lists.
// DESIGN.md O6 ("bundle a set of m source cells which have interactions in common with a
// set of n sink particles ... perform the full m x n interactions on this block"; PAPER.md:75 direct
// interactions near the leaves, quadrupole/hexadecapole cell interactions for the rest).
//
// One warp per (group, 32-sink half) task, one sink per lane (sub-warp tiling for small tasks, below).
// Source tiles are staged through per-warp shared memory in PAIR-INTERLEAVED form {A,B}, read back with
// broadcast LDS.64/128 and consumed with packed f32x2 arithmetic: every thread handles 1 sink x 2 sources
// per instruction (FFMA2 is the
// only way to reach the FP32 peak with three distinct operands on sm_100, see dsk_internal.cuh).
// All coordinates are taken relative to the group's cell centre c_g (exact subtraction for nearby
// values), which keeps fp32 differences accurate and absorbs the periodic image shift.
//
// F1: Plummer pair, acc_i += m_j d / (|d|^2+eps^2)^(3/2), pot_i -= m_j / sqrt(...), d = x_j - x_i.
// F2: derivatives D_n = d^n g, g = (|rho|^2 + eps~^2)^(-1/2), in cell-scaled coordinates rho = r/s:
//       l R^2 D_n + (2l-1) sum_i n_i rho_i D_{n-e_i} + (l-1) sum_i n_i (n_i-1) D_{n-2e_i} = 0,  l = |n|
//     pot_i -= (1/s) sum_{|n|<=p} Mhat_n D_n ,  acc_i += (1/s^2) sum_{|n|<=p} Mhat_n D_{n+e_i}
//     (Mhat carries (-1)^|n|/n!/s^|n|, so there are no per-term factors).
#include "dsk_internal.cuh"
#include <type_traits>

#define P2P_TILE 128         // sources per warp tile

int dsk_walk_fill(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t m2p_base, uint64_t p2p_base);   // walk.cu

// ---- small vector abstraction: T = f2 (two sources per op) or float ---------------------------------
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

// ---- F2 body: one sink against one cell (float) or a pair of cells (f2) ------------------------------
// tile row layout (float2 = {cell A, cell B}): [0..2] com' xyz, [3] 1/s, [4] eps^2/s^2, [5+n] Mhat_n
#define M2P_HDR 5
template <int P, typename T, bool POT>
__device__ __forceinline__ void m2p_body(T xs, T ys, T zs, const float2 *__restrict__ row, int half,
                                         T &pot, T &ax, T &ay, T &az)
{
    constexpr int NP1 = dsk_np(P + 1);
    const T sinv = vld<T>(row + 3, half);
    const T rx = vmul(vsub(xs, vld<T>(row + 0, half)), sinv);
    const T ry = vmul(vsub(ys, vld<T>(row + 1, half)), sinv);
    const T rz = vmul(vsub(zs, vld<T>(row + 2, half)), sinv);
    T R2 = vfma(rx, rx, vld<T>(row + 4, half));
    R2 = vfma(ry, ry, R2);
    R2 = vfma(rz, rz, R2);
    T D[NP1];
    D[0] = vrsqrt(R2);
    const T q = vmul(D[0], D[0]);
    const float2 *Mh = row + M2P_HDR;
    T phi = vmul(vld<T>(Mh, half), D[0]);
    T gx = vdup<T>(0.0f), gy = vdup<T>(0.0f), gz = vdup<T>(0.0f);
    static_for<1, P + 2>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int beg = l * (l + 1) * (l + 2) / 6, end = (l + 1) * (l + 2) * (l + 3) / 6;
        const T A = vmul(q, vdup<T>(-(float)(2 * l - 1) / (float)l));
        T ux[l + 1], uy[l + 1], uz[l + 1], w[l + 1];
        ux[1] = vmul(A, rx); uy[1] = vmul(A, ry); uz[1] = vmul(A, rz);
        static_for<2, l + 1>([&](auto K) {
            constexpr int k = decltype(K)::value;
            ux[k] = vadd(ux[k - 1], ux[1]); uy[k] = vadd(uy[k - 1], uy[1]); uz[k] = vadd(uz[k - 1], uz[1]);
            w[k] = vmul(q, vdup<T>(-(float)(l - 1) * (float)(k * (k - 1)) / (float)l));
        });
        static_for<beg, end>([&](auto I) {
            constexpr int i = decltype(I)::value;
            constexpr MI m = dsk_mi(i);
            T v;
            // first-order terms (at least one of a,b,c is >= 1)
            if constexpr (m.a >= 1) {
                v = vmul(ux[m.a], D[dsk_midx(m.a - 1, m.b, m.c)]);
                if constexpr (m.b >= 1) v = vfma(uy[m.b], D[dsk_midx(m.a, m.b - 1, m.c)], v);
                if constexpr (m.c >= 1) v = vfma(uz[m.c], D[dsk_midx(m.a, m.b, m.c - 1)], v);
            } else if constexpr (m.b >= 1) {
                v = vmul(uy[m.b], D[dsk_midx(m.a, m.b - 1, m.c)]);
                if constexpr (m.c >= 1) v = vfma(uz[m.c], D[dsk_midx(m.a, m.b, m.c - 1)], v);
            } else {
                v = vmul(uz[m.c], D[dsk_midx(m.a, m.b, m.c - 1)]);
            }
            if constexpr (m.a >= 2) v = vfma(w[m.a], D[dsk_midx(m.a - 2, m.b, m.c)], v);
            if constexpr (m.b >= 2) v = vfma(w[m.b], D[dsk_midx(m.a, m.b - 2, m.c)], v);
            if constexpr (m.c >= 2) v = vfma(w[m.c], D[dsk_midx(m.a, m.b, m.c - 2)], v);
            D[i] = v;
            if constexpr (POT && l <= P) phi = vfma(vld<T>(Mh + i, half), v, phi);
            if constexpr (m.a >= 1) gx = vfma(vld<T>(Mh + dsk_midx(m.a - 1, m.b, m.c), half), v, gx);
            if constexpr (m.b >= 1) gy = vfma(vld<T>(Mh + dsk_midx(m.a, m.b - 1, m.c), half), v, gy);
            if constexpr (m.c >= 1) gz = vfma(vld<T>(Mh + dsk_midx(m.a, m.b, m.c - 1), half), v, gz);
        });
    });
    const T sinv2 = vmul(sinv, sinv);
    if constexpr (POT) pot = vfma(phi, sinv, pot);        // caller subtracts
    ax = vfma(gx, sinv2, ax); ay = vfma(gy, sinv2, ay); az = vfma(gz, sinv2, az);
}

// ---- work decomposition shared by F1 and F2 -----------------------------------------------------------
// One WARP per task; task = (group, half): sinks [32 half, 32 half + 32) of the group, so a group of <= 32
// sinks is one warp and nothing waits at a block barrier (ncu on the first version, one 64-thread CTA per
// group: 6 barrier-stall cycles per issue, FMA pipe 45 % active, ~18 of 64 lanes useful on the Plummer
// workload).  Groups are cells, so many hold few sinks: a task with ns <= 16 (<= 8) sinks splits the warp
// into 2 (4) sub-groups that take alternate source pairs of a tile and are summed at the end.
struct warp_task {
    uint32_t g, first, ns;       // group, rank of the task's first sink, sinks in the task
    int W, S, sub, j;            // sub-group width, number of sub-groups, my sub-group, my sink in the task
    bool valid;
};
__device__ __forceinline__ warp_task make_task(uint32_t t0, uint32_t t1, int fw, const uint32_t *__restrict__ taskmap,
                                               const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount)
{
    warp_task t;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t task = t0 + blockIdx.x * fw + warp;
    t.valid = false;
    t.g = 0; t.first = 0; t.ns = 0; t.W = 32; t.S = 1; t.sub = 0; t.j = 0;
    if (task >= t1) return t;
    const uint32_t m = taskmap[task], h = m & 1u;
    t.g = m >> 1;
    const uint32_t count = gcount[t.g];
    t.valid = true;
    t.ns = min(32u, count - 32u * h);
    t.first = gfirst[t.g] + 32u * h;
    t.W = t.ns <= 8 ? 8 : (t.ns <= 16 ? 16 : 32);
    t.S = 32 / t.W;
    t.sub = lane / t.W;
    t.j = min(lane % t.W, (int)t.ns - 1);
    return t;
}
// sum the sub-groups' two-float accumulators (in double) and store; lanes of sub-group 0 own the sinks
__device__ __forceinline__ void task_store(const warp_task &t, float4 hi, float4 lo, float4 *__restrict__ sacc,
                                           float4 *__restrict__ sacc_lo)
{
    double d[4] = {(double)hi.x + (double)lo.x, (double)hi.y + (double)lo.y, (double)hi.z + (double)lo.z,
                   (double)hi.w + (double)lo.w};
    for (int o = 16; o >= t.W; o >>= 1)
#pragma unroll
        for (int q = 0; q < 4; q++) d[q] += __shfl_xor_sync(0xffffffffu, d[q], o);
    const int lane = threadIdx.x & 31;
    if (lane < (int)t.ns) {
        float4 oh, ol;
        oh.x = (float)d[0]; oh.y = (float)d[1]; oh.z = (float)d[2]; oh.w = (float)d[3];
        ol.x = (float)(d[0] - (double)oh.x); ol.y = (float)(d[1] - (double)oh.y); ol.z = (float)(d[2] - (double)oh.z);
        ol.w = (float)(d[3] - (double)oh.w);
        sacc[t.first + lane] = oh; sacc_lo[t.first + lane] = ol;
    }
}

#define FW 4                 // warps (tasks) per block

template <int P, bool POT, bool PACKED>
__global__ void __launch_bounds__(FW * 32) k_m2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic, float box, float eps2,
                                                 const float *__restrict__ rows, const float4 *__restrict__ spos,
                                                 const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                 const uint32_t *__restrict__ gcell, const uint32_t *__restrict__ list,
                                                 const uint64_t *__restrict__ off, uint64_t base,
                                                 const uint32_t *__restrict__ len, float4 *__restrict__ sacc,
                                                 float4 *__restrict__ sacc_lo)
{
    constexpr int NP = dsk_np(P), ROW = dsk_rowlen(P), TROW = M2P_HDR + NP;
    constexpr int TC = (P <= 6) ? 32 : 16;                  // cells per tile (one per lane at most)
    __shared__ uint32_t s_cell_all[FW][TC];
    __shared__ __align__(16) float2 tile_all[FW][TC / 2][TROW];
    const warp_task t = make_task(t0, t1, FW, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *s_cell = s_cell_all[warp];
    float2(*tile)[TROW] = tile_all[warp];
    const float *grow = rows + (size_t)gcell[t.g] * ROW;
    const float cgx = grow[0], cgy = grow[1], cgz = grow[2];
    const float4 me = spos[t.first + t.j];
    const uint32_t n = len[t.g];
    const uint32_t *lst = list + (off[t.g] - base);
    using T = typename std::conditional<PACKED, f2, float>::type;
    // running sums as two-float (hi, lo) pairs, continued from the P2P kernel (sub-group 0 carries them);
    // each tile is summed from zero in plain fp32 and folded in with TwoSum, so no addition ever rounds at
    // the size of the total
    float4 hi = make_float4(0.f, 0.f, 0.f, 0.f), lo = hi;
    if (t.sub == 0 && lane < (int)t.ns) { hi = sacc[t.first + lane]; lo = sacc_lo[t.first + lane]; }
    const T X = vdup<T>(me.x - cgx), Y = vdup<T>(me.y - cgy), Z = vdup<T>(me.z - cgz);
    const int quantum = PACKED ? 2 * t.S : t.S;             // cells consumed per round of the sub-groups
    for (uint32_t b0 = 0; b0 < n; b0 += TC) {
        const int ntc = (int)min((uint32_t)TC, n - b0);
        const int npad = (ntc + quantum - 1) / quantum * quantum;
        if (lane < npad) {
            float cx = 1.0e5f, cy = 1.0e5f, cz = 1.0e5f, sinv = 1.0f;       // dummy cell: far away, no mass
            uint32_t cidx = 0xffffffffu;
            if (lane < ntc) {
                const uint32_t e = lst[b0 + lane];
                cidx = e & ((1u << DSK_CELL_BITS) - 1u);
                const float *r = rows + (size_t)cidx * ROW;
                const float4 h0 = *reinterpret_cast<const float4 *>(r);
                const float4 h1 = *reinterpret_cast<const float4 *>(r + 4);
                float shx = 0.0f, shy = 0.0f, shz = 0.0f;
                if (periodic) {
                    const int img = (int)(e >> DSK_CELL_BITS), side = 2 * DSK_WS + 1;
                    shz = (float)(img % side - DSK_WS) * box;
                    shy = (float)((img / side) % side - DSK_WS) * box;
                    shx = (float)(img / (side * side) - DSK_WS) * box;
                }
                cx = ((h0.x - cgx) + shx) + h1.x; cy = ((h0.y - cgy) + shy) + h1.y; cz = ((h0.z - cgz) + shz) + h1.z;
                sinv = h0.w;
            }
            s_cell[lane] = cidx;
            float *hd = reinterpret_cast<float *>(&tile[lane >> 1][0]) + (lane & 1);
            hd[0] = cx; hd[2] = cy; hd[4] = cz; hd[6] = sinv; hd[8] = eps2 * sinv * sinv;
        }
        __syncwarp();
        for (int idx = lane; idx < npad * NP; idx += 32) {
            const int ci = idx / NP, k = idx - ci * NP;
            const uint32_t cidx = s_cell[ci];
            const float v = cidx != 0xffffffffu ? rows[(size_t)cidx * ROW + 8 + k] : 0.0f;
            reinterpret_cast<float *>(&tile[ci >> 1][M2P_HDR + k])[ci & 1] = v;
        }
        __syncwarp();
        {
            T pot = vdup<T>(0.0f), ax = vdup<T>(0.0f), ay = vdup<T>(0.0f), az = vdup<T>(0.0f);
            if constexpr (PACKED) {
                const int npair = npad >> 1;
                for (int k = t.sub; k < npair; k += t.S) m2p_body<P, T, POT>(X, Y, Z, tile[k], 0, pot, ax, ay, az);
            } else {
                for (int k = t.sub; k < npad; k += t.S) m2p_body<P, T, POT>(X, Y, Z, tile[k >> 1], k & 1, pot, ax, ay, az);
            }
            dsk_fold(hi.x, lo.x, vsum(ax)); dsk_fold(hi.y, lo.y, vsum(ay)); dsk_fold(hi.z, lo.z, vsum(az));
            if (POT) dsk_fold(hi.w, lo.w, -vsum(pot));
        }
        __syncwarp();
    }
    task_store(t, hi, lo, sacc, sacc_lo);
}

// ---- F1 ----------------------------------------------------------------------------------------------
template <bool POT>
__global__ void __launch_bounds__(FW * 32) k_p2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic, float box, float eps2,
                                                 int rowlen, const float *__restrict__ rows,
                                                 const dsk_cellrec *__restrict__ cell, const float4 *__restrict__ spos,
                                                 const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                 const uint32_t *__restrict__ gcell, const uint32_t *__restrict__ list,
                                                 const uint64_t *__restrict__ off, uint64_t base,
                                                 const uint32_t *__restrict__ len, float4 *__restrict__ sacc,
                                                 float4 *__restrict__ sacc_lo)
{
    __shared__ uint32_t s_first_all[FW][32];
    __shared__ uint32_t s_pref_all[FW][33];
    __shared__ float s_sh_all[FW][32][3];
    __shared__ __align__(16) float4 tA_all[FW][P2P_TILE / 2], tB_all[FW][P2P_TILE / 2];   // {xA,xB,yA,yB}, {zA,zB,mA,mB}
    const warp_task t = make_task(t0, t1, FW, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *s_first = s_first_all[warp], *s_pref = s_pref_all[warp];
    float(*s_sh)[3] = s_sh_all[warp];
    float4 *tA = tA_all[warp], *tB = tB_all[warp];
    const float *grow = rows + (size_t)gcell[t.g] * rowlen;
    const float cgx = grow[0], cgy = grow[1], cgz = grow[2];
    const float4 me = spos[t.first + t.j];
    const f2 X = f2_dup(me.x - cgx), Y = f2_dup(me.y - cgy), Z = f2_dup(me.z - cgz);
    const f2 E2 = f2_dup(eps2);
    const uint32_t n = len[t.g];
    const uint32_t *lst = list + (off[t.g] - base);
    float4 hi = make_float4(0.f, 0.f, 0.f, 0.f), lo = hi;     // two-float running sums (see k_m2p)
    const uint32_t quantum = 2u * (uint32_t)t.S;
    for (uint32_t b0 = 0; b0 < n; b0 += 32) {
        // one leaf (segment of sources) per lane; exclusive scan of the segment lengths
        uint32_t cnt = 0;
        if (b0 + lane < n) {
            const uint32_t e = lst[b0 + lane];
            const dsk_cellrec r = cell[e & ((1u << DSK_CELL_BITS) - 1u)];
            s_first[lane] = r.first; cnt = r.count;
            float shx = 0.0f, shy = 0.0f, shz = 0.0f;
            if (periodic) {
                const int img = (int)(e >> DSK_CELL_BITS), side = 2 * DSK_WS + 1;
                shz = (float)(img % side - DSK_WS) * box;
                shy = (float)((img / side) % side - DSK_WS) * box;
                shx = (float)(img / (side * side) - DSK_WS) * box;
            }
            s_sh[lane][0] = shx; s_sh[lane][1] = shy; s_sh[lane][2] = shz;
        }
        uint32_t x = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        const uint32_t total = __shfl_sync(0xffffffffu, x, 31);
        s_pref[lane] = x - cnt;
        if (lane == 0) s_pref[32] = total;
        __syncwarp();
        for (uint32_t t0 = 0; t0 < total; t0 += P2P_TILE) {
            const uint32_t nt = min((uint32_t)P2P_TILE, total - t0);
            const uint32_t npad = (nt + quantum - 1) / quantum * quantum;
            for (uint32_t j = lane; j < npad; j += 32) {
                float sx = 1.0e10f, sy = 1.0e10f, sz = 1.0e10f, sm = 0.0f;      // pad: far away, massless
                if (j < nt) {
                    const uint32_t gj = t0 + j;
                    int a = 0, b = 32;                        // last segment with pref <= gj
                    while (b - a > 1) {
                        const int mid = (a + b) >> 1;
                        if (s_pref[mid] <= gj) a = mid; else b = mid;
                    }
                    const float4 p = spos[s_first[a] + (gj - s_pref[a])];
                    sx = (p.x - cgx) + s_sh[a][0]; sy = (p.y - cgy) + s_sh[a][1]; sz = (p.z - cgz) + s_sh[a][2];
                    sm = p.w;
                }
                float *pa = reinterpret_cast<float *>(&tA[j >> 1]) + (j & 1);
                float *pb = reinterpret_cast<float *>(&tB[j >> 1]) + (j & 1);
                pa[0] = sx; pa[2] = sy; pb[0] = sz; pb[2] = sm;
            }
            __syncwarp();
            {
                f2 ax = f2_dup(0.0f), ay = f2_dup(0.0f), az = f2_dup(0.0f), pot = f2_dup(0.0f);
                const int npair = (int)(npad >> 1);
#pragma unroll 4
                for (int k = t.sub; k < npair; k += t.S) {
                    const ulonglong2 qa = *reinterpret_cast<const ulonglong2 *>(&tA[k]);
                    const ulonglong2 qb = *reinterpret_cast<const ulonglong2 *>(&tB[k]);
                    f2 sx, sy, sz, sm;
                    sx.v = qa.x; sy.v = qa.y; sz.v = qb.x; sm.v = qb.y;
                    const f2 dx = f2_sub(sx, X), dy = f2_sub(sy, Y), dz = f2_sub(sz, Z);
                    f2 r2 = f2_fma(dx, dx, E2);
                    r2 = f2_fma(dy, dy, r2);
                    r2 = f2_fma(dz, dz, r2);
                    const f2 ri = f2_rsqrt(r2);
                    const f2 ri2 = f2_mul(ri, ri), mri = f2_mul(sm, ri), mri3 = f2_mul(mri, ri2);
                    ax = f2_fma(dx, mri3, ax); ay = f2_fma(dy, mri3, ay); az = f2_fma(dz, mri3, az);
                    if (POT) pot = f2_sub(pot, mri);
                }
                dsk_fold(hi.x, lo.x, vsum(ax)); dsk_fold(hi.y, lo.y, vsum(ay)); dsk_fold(hi.z, lo.z, vsum(az));
                if (POT) dsk_fold(hi.w, lo.w, vsum(pot));
            }
            __syncwarp();
        }
    }
    // the sink's own leaf is always in the list: remove its self term -m_i/eps from the potential (once)
    if (POT && t.sub == 0) dsk_fold(hi.w, lo.w, me.w * rsqrtf(eps2));
    task_store(t, hi, lo, sacc, sacc_lo);
}

template <int P>
static void launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot)
{
    const float e2 = c->eps * c->eps;
    constexpr bool PACKED = (P <= 6);
    if (want_pot)
        k_m2p<P, true, PACKED><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, c->stream>>>(t0, t1, c->g_task, c->periodic, c->box, e2, c->rows, c->spos, c->gfirst,
                                                              c->gcount, c->gcell, c->list_m2p, c->g_m2p_off, base,
                                                              c->g_m2p_len, c->sacc, c->sacc_lo);
    else
        k_m2p<P, false, PACKED><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, c->stream>>>(t0, t1, c->g_task, c->periodic, c->box, e2, c->rows, c->spos, c->gfirst,
                                                               c->gcount, c->gcell, c->list_m2p, c->g_m2p_off, base,
                                                               c->g_m2p_len, c->sacc, c->sacc_lo);
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
    const int rowlen = dsk_rowlen(c->p);
    if (want_pot)
        k_p2p<true><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, s>>>(t0, t1, c->g_task, c->periodic, c->box, e2, rowlen, c->rows, c->cell, c->spos, c->gfirst,
                                           c->gcount, c->gcell, c->list_p2p, c->g_p2p_off, pb, c->g_p2p_len, c->sacc, c->sacc_lo);
    else
        k_p2p<false><<<(t1 - t0 + FW - 1) / FW, FW * 32, 0, s>>>(t0, t1, c->g_task, c->periodic, c->box, e2, rowlen, c->rows, c->cell, c->spos, c->gfirst,
                                            c->gcount, c->gcell, c->list_p2p, c->g_p2p_off, pb, c->g_p2p_len, c->sacc, c->sacc_lo);
    cudaEventRecord(c->ev[9], s);
    switch (c->p) {
    case 2: launch_m2p<2>(c, t0, t1, mb, want_pot); break;
    case 4: launch_m2p<4>(c, t0, t1, mb, want_pot); break;
    case 6: launch_m2p<6>(c, t0, t1, mb, want_pot); break;
    case 8: launch_m2p<8>(c, t0, t1, mb, want_pot); break;
    default: return DSK_EINVAL;
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
