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
