// peak.cu — FP32 issue-rate probe: the measured denominator of the force kernels' roofline (SURVEY.md section 7:
// "a pure-FFMA microbenchmark that measures the sustained FP32 peak and the SM clock it runs at").
// Three operand forms of the instruction the force kernels are made of, each as independent dependency chains long
// enough to hide the pipe latency, nothing else in the loop:
//   variant 0  FFMA2, three packed register operands                  a = fma(x, y, a)     x, y, a: 64-bit register pairs
//   variant 1  FFMA2, one operand a scalar broadcast to both halves   a = fma(a, {s,s}, y) the form M2P/P2P feed sources in
//   variant 2  scalar FFMA, three distinct registers                  a = fma(x, y, a)
//   variant 3  FFMA2, the two source operands shared by all chains    a_k = fma(a_k, {s,s}, y)   (operand-reuse cache hits)
//   variant 4  scalar FFMA, the two source operands shared            a_k = fma(a_k, s, y)
//   variant 5  the M2P body's pattern: a_k = fma({s_i,s_i}, m_k, a_k), a new scalar s_i every instruction, m_k and a_k distinct
//   variant 6  the same with each scalar used by TWO consecutive instructions (what four sinks per lane would give)
// Variants 0-2 read five or six, three distinct registers per instruction and are bound by register-file bandwidth (measured:
// one FFMA2 per 2.6 - 3.0 cycles, one FFMA per 1.5); 3 and 4 show what the pipe itself issues when operands repeat, which is
// what a real inner loop (one coefficient against many monomials) looks like.
// Reported: TFLOP/s (2 flop per lane and FMA) from CUDA events, cycles per warp instruction per SM sub-partition from
// clock64() inside the kernel, and the SM clock the kernel ran at (clock64 cycles over globaltimer nanoseconds).
#include "dsk_internal.cuh"

#define PK_CHAINS 8          // independent accumulators per thread
#define PK_UNROLL 16         // loop body = PK_UNROLL x PK_CHAINS instructions
#define PK_THREADS 1024      // one block per SM: 32 warps = 8 per sub-partition (two blocks of 512 per SM did not always
#define PK_BLOCKS_PER_SM 1   // land two to an SM: the event time then read 25 % below what the SMs' own clocks showed)

__device__ __forceinline__ unsigned long long pk_globaltimer()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

template <int VARIANT>
__global__ void __launch_bounds__(PK_THREADS, PK_BLOCKS_PER_SM) k_fp32_peak(int iters, const float *__restrict__ seed,
                                                                           float *__restrict__ out,
                                                                           unsigned long long *__restrict__ clk)
{
    const float s0 = seed[0], s1 = seed[1];                  // run-time values: nothing folds at compile time
    const unsigned long long t0 = pk_globaltimer();
    const long long c0 = clock64();
    float res = 0.0f;
    if (VARIANT == 5 || VARIANT == 6) {
        f2 a[PK_CHAINS], m[PK_CHAINS];
        float sc[PK_CHAINS];
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) {
            a[k] = f2_make(s0 + (float)k, s1 + (float)k);
            m[k] = f2_make(s1 * 1e-3f + 1e-4f * (float)(k + threadIdx.x), s0 * 1e-3f + 2e-4f * (float)k);
            sc[k] = s1 * 0.5f + 1e-3f * (float)k;
        }
        for (int it = 0; it < iters; it++)
#pragma unroll
            for (int u = 0; u < PK_UNROLL; u++)
#pragma unroll
                for (int k = 0; k < PK_CHAINS; k++) a[k] = f2_fma(f2_dup(sc[VARIANT == 5 ? k : (k >> 1)]), m[k], a[k]);
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) res += f2_lo(a[k]) + f2_hi(a[k]);
    } else if (VARIANT == 4) {
        float a[PK_CHAINS];
        const float x = s1 + 1e-3f * (float)threadIdx.x, y = s0 * 0.5f;
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) a[k] = s0 + (float)k;
        for (int it = 0; it < iters; it++)
#pragma unroll
            for (int u = 0; u < PK_UNROLL; u++)
#pragma unroll
                for (int k = 0; k < PK_CHAINS; k++) a[k] = fmaf(a[k], x, y);
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) res += a[k];
    } else if (VARIANT == 2) {
        float a[PK_CHAINS], x[PK_CHAINS], y[PK_CHAINS];
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) { a[k] = s0 + (float)k; x[k] = s1 + 1e-3f * (float)(k + threadIdx.x); y[k] = s0 * 0.5f + 1e-3f * (float)k; }
        for (int it = 0; it < iters; it++)
#pragma unroll
            for (int u = 0; u < PK_UNROLL; u++)
#pragma unroll
                for (int k = 0; k < PK_CHAINS; k++) a[k] = fmaf(x[k], y[k], a[k]);
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) res += a[k];
    } else {
        f2 a[PK_CHAINS], x[PK_CHAINS], y[PK_CHAINS];
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) {
            a[k] = f2_make(s0 + (float)k, s1 + (float)k);
            x[k] = f2_make(s1 + 1e-3f * (float)(k + threadIdx.x), s0 + 2e-3f * (float)k);
            y[k] = f2_make(s0 * 0.5f + 1e-3f * (float)k, s1 * 0.25f + 1e-3f * (float)k);
        }
        float sc[PK_CHAINS];
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) sc[k] = s1 * 1e-3f + 1e-6f * (float)k;
        for (int it = 0; it < iters; it++)
#pragma unroll
            for (int u = 0; u < PK_UNROLL; u++)
#pragma unroll
                for (int k = 0; k < PK_CHAINS; k++) {
                    if (VARIANT == 0) a[k] = f2_fma(x[k], y[k], a[k]);
                    else if (VARIANT == 1) a[k] = f2_fma(a[k], f2_dup(sc[k]), y[k]);
                    else a[k] = f2_fma(a[k], f2_dup(sc[0]), y[0]);
                }
#pragma unroll
        for (int k = 0; k < PK_CHAINS; k++) res += f2_lo(a[k]) + f2_hi(a[k]);
    }
    const long long c1 = clock64();
    const unsigned long long t1 = pk_globaltimer();
    out[(size_t)blockIdx.x * PK_THREADS + threadIdx.x] = res;
    if (threadIdx.x == 0) { clk[2 * blockIdx.x] = (unsigned long long)(c1 - c0); clk[2 * blockIdx.x + 1] = t1 - t0; }
}

// Host pointers.  Allocates and frees its own few MB of device memory (it is a diagnostic, not part of the path).
static int probe_impl(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz, double *tflops_by_cycles);
extern "C" int dsk_probe_fp32_peak(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz)
{
    return probe_impl(variant, tflops, cycles_per_inst_smsp, sm_mhz, nullptr);
}
// the same plus the rate implied by the in-kernel cycle counters (a cross-check of the event timing)
extern "C" int dsk_probe_fp32_peak_ex(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz, double *tflops_by_cycles)
{
    if (!tflops_by_cycles) return DSK_EINVAL;
    return probe_impl(variant, tflops, cycles_per_inst_smsp, sm_mhz, tflops_by_cycles);
}
static int probe_impl(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz, double *tflops_by_cycles)
{
    if (variant < 0 || variant > 6 || !tflops || !cycles_per_inst_smsp || !sm_mhz) return DSK_EINVAL;
    int dev = 0, nsm = 0;
    DSK_CUDA(cudaGetDevice(&dev));
    DSK_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    const int grid = nsm * PK_BLOCKS_PER_SM, iters = 2048;
    float *out = nullptr, *seed = nullptr;
    unsigned long long *clk = nullptr;
    DSK_CUDA(cudaMalloc(&out, sizeof(float) * (size_t)grid * PK_THREADS));
    DSK_CUDA(cudaMalloc(&seed, sizeof(float) * 2));
    DSK_CUDA(cudaMalloc(&clk, sizeof(unsigned long long) * 2 * grid));
    const float hs[2] = {1.0f, 0.999f};
    DSK_CUDA(cudaMemcpy(seed, hs, sizeof(hs), cudaMemcpyHostToDevice));
    cudaEvent_t e0, e1;
    DSK_CUDA(cudaEventCreate(&e0));
    DSK_CUDA(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 6; rep++) {                      // first repetitions warm the clocks up
        cudaEventRecord(e0);
        if (variant == 0) k_fp32_peak<0><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else if (variant == 1) k_fp32_peak<1><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else if (variant == 2) k_fp32_peak<2><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else if (variant == 3) k_fp32_peak<3><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else if (variant == 4) k_fp32_peak<4><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else if (variant == 5) k_fp32_peak<5><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        else k_fp32_peak<6><<<grid, PK_THREADS>>>(iters, seed, out, clk);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 2 && ms < best) best = ms;
    }
    unsigned long long *h = new unsigned long long[2 * grid];
    cudaError_t err = cudaMemcpy(h, clk, sizeof(unsigned long long) * 2 * grid, cudaMemcpyDeviceToHost);
    double cyc = 0.0, ns = 0.0;
    for (int b = 0; b < grid; b++) { cyc += (double)h[2 * b]; ns += (double)h[2 * b + 1]; }
    delete[] h;
    cudaFree(out); cudaFree(seed); cudaFree(clk);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (err != cudaSuccess || cudaGetLastError() != cudaSuccess || best > 1e29f) return DSK_ECUDA;
    const double inst_per_thread = (double)iters * PK_UNROLL * PK_CHAINS;
    const double lanes = (variant == 2 || variant == 4) ? 1.0 : 2.0;
    *tflops = inst_per_thread * 2.0 * lanes * (double)grid * PK_THREADS / ((double)best * 1e-3) / 1e12;
    if (tflops_by_cycles) {      // the same from the SMs' own cycle counters: flop per block / (its cycles / its clock), all blocks at once
        const double sec = (cyc / grid) / (cyc / ns * 1e9);
        *tflops_by_cycles = inst_per_thread * 2.0 * lanes * (double)grid * PK_THREADS / sec / 1e12;
    }
    // warp instructions issued by one sub-partition while a block's clock ran: the SM holds PK_BLOCKS_PER_SM blocks of
    // PK_THREADS / 32 warps, a quarter of them on each sub-partition
    const double warps_per_smsp = (double)PK_BLOCKS_PER_SM * (PK_THREADS / 32) / 4.0;
    *cycles_per_inst_smsp = (cyc / grid) / (inst_per_thread * warps_per_smsp);
    *sm_mhz = cyc / ns * 1e3;
    return DSK_OK;
}
