// kdk.cu — step I: kick and drift kernels of the comoving leapfrog (O9; PAPER.md:63
// "symplectic integrator").  Pure streaming: 24 B/particle read + 12 B written per kernel.
// The factors K (int dt/a) and D (int dt/a^2) are computed in fp64 on the host (dsk_api.cu).
#include "dsk_internal.cuh"

__global__ void __launch_bounds__(256) k_kick(float *__restrict__ vel, const float *__restrict__ acc, int64_t n3, float k)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n3) vel[i] = fmaf(acc[i], k, vel[i]);
}

__global__ void __launch_bounds__(256) k_drift(float *__restrict__ pos, const float *__restrict__ vel, int64_t n3,
                                               float d, float box, int periodic)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n3) return;
    float x = fmaf(vel[i], d, pos[i]);
    if (periodic) {       // the fp32 wrap of reading O1
        float t = __fdiv_rn(x, box);
        float w = __fsub_rn(x, __fmul_rn(box, floorf(t)));
        if (!(w >= 0.0f && w < box)) w = 0.0f;
        x = w;
    }
    pos[i] = x;
}

int dsk_run_kick(dsk_ctx *c, float *vel, const float *acc, float k)
{
    int64_t n3 = 3 * c->N;
    k_kick<<<(unsigned)((n3 + 255) / 256), 256, 0, c->stream>>>(vel, acc, n3, k);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_run_drift(dsk_ctx *c, float *pos, const float *vel, float d)
{
    int64_t n3 = 3 * c->N;
    k_drift<<<(unsigned)((n3 + 255) / 256), 256, 0, c->stream>>>(pos, vel, n3, d, c->box, c->periodic);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// ---- hierarchical (block) time steps (O9c; "adaptive symplectic integrator (Quinn et al.
// 1997)") -------------------------------------------------------------------------------------------------
// nsub = 2^rmax substeps per block step; a particle on rung r takes steps of L(r) = nsub >> r substeps.
// A rung above rmax (an array carried over from a call with a deeper hierarchy, or never initialised) is read as rmax:
// without the clamp nsub >> r is 0 (a device modulo by zero) and k[r] lies past the table.
struct dsk_rung_factors { float k[DSK_RMAX + 1]; };
__device__ __forceinline__ uint32_t dsk_rung_clamped(uint8_t r, uint32_t rmax) { return r > rmax ? rmax : (uint32_t)r; }

// v += acc * k[rung] for the particles whose step starts (mode 0: s % L == 0) or ends (mode 1: active) now
__global__ void __launch_bounds__(256) k_kick_rung(float *__restrict__ vel, const float *__restrict__ acc,
                                                   const uint8_t *__restrict__ rung, int64_t n, uint32_t s,
                                                   uint32_t nsub, uint32_t rmax, dsk_rung_factors f)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t r = dsk_rung_clamped(rung[i], rmax), L = nsub >> r;
    if (s % L) return;
    const float k = f.k[r];
#pragma unroll
    for (int d = 0; d < 3; d++) vel[3 * i + d] = fmaf(acc[3 * i + d], k, vel[3 * i + d]);
}

__global__ void __launch_bounds__(256) k_rung_active(const uint8_t *__restrict__ rung, int64_t n, uint32_t t,
                                                     uint32_t nsub, uint32_t rmax, uint8_t *__restrict__ active)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) active[i] = (t % (nsub >> dsk_rung_clamped(rung[i], rmax))) == 0 ? 1 : 0;
}

// the step criterion, decided in fp32: step_i = eta sqrt(eps / |acc_i|), wanted rung = ceil(log2(da / step_i)) in
// [0, rmax]; a particle that just ended a step moves to a finer rung at once, to a coarser one by one level and
// only when t is a multiple of the coarser step
__global__ void __launch_bounds__(256) k_rung_update(const float *__restrict__ acc, const uint8_t *__restrict__ active,
                                                     uint8_t *__restrict__ rung, int64_t n, uint32_t t, uint32_t nsub,
                                                     int rmax, float da, float eta, float eps)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || !active[i]) return;
    const float ax = acc[3 * i], ay = acc[3 * i + 1], az = acc[3 * i + 2];
    const float amag = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(ax, ax), __fmul_rn(ay, ay)), __fmul_rn(az, az)));
    const float step = __fmul_rn(eta, __fsqrt_rn(__fdiv_rn(eps, amag)));
    const float w = ceilf(log2f(__fdiv_rn(da, step)));
    int want = isfinite(w) ? (int)fminf(fmaxf(w, 0.0f), (float)rmax) : 0;
    const int r = (int)dsk_rung_clamped(rung[i], (uint32_t)rmax);
    if (want > r) rung[i] = (uint8_t)want;
    else if (want < r && r > 0 && (t % (nsub >> (r - 1))) == 0) rung[i] = (uint8_t)(r - 1);
    else rung[i] = (uint8_t)r;                   // writes the clamped value back when the input was out of range
}

int dsk_run_kick_rung(dsk_ctx *c, float *vel, const float *acc, const uint8_t *rung, uint32_t s, uint32_t nsub,
                      int rmax, const float *k)
{
    dsk_rung_factors f;
    for (int r = 0; r <= DSK_RMAX; r++) f.k[r] = k[r];
    k_kick_rung<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(vel, acc, rung, c->N, s, nsub, (uint32_t)rmax, f);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_run_rung_active(dsk_ctx *c, const uint8_t *rung, uint32_t t, uint32_t nsub, int rmax, uint8_t *active)
{
    k_rung_active<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(rung, c->N, t, nsub, (uint32_t)rmax, active);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_run_rung_update(dsk_ctx *c, const float *acc, const uint8_t *active, uint8_t *rung, uint32_t t, uint32_t nsub,
                        int rmax, float da, float eta)
{
    k_rung_update<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(acc, active, rung, c->N, t, nsub, rmax, da, eta, c->eps);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
