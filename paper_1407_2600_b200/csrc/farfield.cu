// farfield.cu — step F3: periodic far field as an order-8 local expansion about the box centre.
// DESIGN.md O7 ("periodic boundary conditions using a high-order (p=8) multipole local
// expansion (Challacombe et al. 1997; Metchnik 2009)").  The (2 WS+1)^3 nearest images are summed by
// the tree walk; everything else (all farther images + the neutralising background) is the smooth field
//   Phi_far(u) = psi_Ewald(u) + sum_{|n|_inf <= WS} 1/|u - nL|
// whose Taylor coefficients T_n (|n| <= 8) are computed once per context on the host in fp64.
// Per force evaluation: (a) root moments M_k = sum m (x - c)^k, |k| <= 8, fp64 block partials;
// (b) Lambda_n = sum_k (-1)^|k| C(n+k,k) M_k T_{n+k}; (c) per particle pot += sum Lambda_n X^n,
// acc_i -= sum n_i Lambda_n X^(n-e_i).
#include "dsk_internal.cuh"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <type_traits>
#include <vector>

#define NF DSK_NFAR
#define FO DSK_FAR_ORDER

// ---------------------------------------------------------------------------------------------------
// host: lattice tensors.  Truncated polynomial algebra in three variables (degree <= 8).
namespace {
struct Poly {
    double c[NF];
    Poly() { memset(c, 0, sizeof(c)); }
};
struct Tab {
    int a[NF], b[NF], c[NF], l[NF];
    Tab()
    {
        for (int L = 0; L <= FO; L++)
            for (int A = L; A >= 0; A--)
                for (int B = L - A; B >= 0; B--) {
                    int C = L - A - B, i = dsk_midx(A, B, C);
                    a[i] = A; b[i] = B; c[i] = C; l[i] = L;
                }
    }
};
const Tab &tab()
{
    static Tab t;
    return t;
}
Poly mul(const Poly &x, const Poly &y)
{
    const Tab &t = tab();
    Poly r;
    for (int i = 0; i < NF; i++) {
        if (x.c[i] == 0.0) continue;
        for (int j = 0; j < NF && t.l[i] + t.l[j] <= FO; j++)
            r.c[dsk_midx(t.a[i] + t.a[j], t.b[i] + t.b[j], t.c[i] + t.c[j])] += x.c[i] * y.c[j];
    }
    return r;
}
// out += sum_k coef[k] * delta^k, k = 0..FO  (delta has no constant term)
void compose(const double coef[FO + 1], const Poly &delta, Poly &out)
{
    Poly pw;
    pw.c[0] = 1.0;
    for (int k = 0; k <= FO; k++) {
        if (k) pw = mul(pw, delta);
        for (int i = 0; i < NF; i++) out.c[i] += coef[k] * pw.c[i];
    }
}
}   // namespace

void dsk_lattice_tensors(double L, int ws, double *T)
{
    const double PI = 3.14159265358979323846, alpha = 2.0 / L, sqpi = sqrt(PI);
    Poly out;
    out.c[0] = PI / (alpha * alpha * L * L * L);
    // real-space images.  s = |u - a|^2 = s0 + delta(u), delta = -2 a.u + |u|^2.
    // Taylor coefficients in delta of F(s): F^(k)(s0)/k!, with d/ds = -(1/2) * (-(1/r) d/dr).
    const double rcut = 6.5 / alpha;
    const int nmax = (int)ceil(rcut / L) + ws + 1;
    for (int ix = -nmax; ix <= nmax; ix++)
        for (int iy = -nmax; iy <= nmax; iy++)
            for (int iz = -nmax; iz <= nmax; iz++) {
                const bool inblock = abs(ix) <= ws && abs(iy) <= ws && abs(iz) <= ws;
                const double a[3] = {ix * L, iy * L, iz * L};
                const double s0 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
                Poly delta;
                delta.c[dsk_midx(2, 0, 0)] = delta.c[dsk_midx(0, 2, 0)] = delta.c[dsk_midx(0, 0, 2)] = 1.0;
                delta.c[dsk_midx(1, 0, 0)] = -2 * a[0]; delta.c[dsk_midx(0, 1, 0)] = -2 * a[1];
                delta.c[dsk_midx(0, 0, 1)] = -2 * a[2];
                double coef[FO + 1];
                if (s0 == 0.0) {
                    // in-block image at the origin: erf(alpha r)/r = 2 alpha/sqrt(pi) sum_k (-alpha^2 s)^k/(k!(2k+1))
                    double f = 2.0 * alpha / sqpi, kf = 1.0;
                    for (int k = 0; k <= FO; k++) {
                        if (k) { f *= -alpha * alpha; kf *= k; }
                        coef[k] = f / (kf * (2 * k + 1));
                    }
                } else {
                    const double r = sqrt(s0);
                    if (!inblock && r > rcut + 2 * L) continue;
                    // E_k = (-(1/r) d/dr)^k [erfc(alpha r)/r],  N_k = (-(1/r) d/dr)^k [1/r] = (2k-1)!!/r^(2k+1)
                    double E = erfc(alpha * r) / r, N = 1.0 / r, g = exp(-alpha * alpha * s0) / (alpha * sqpi);
                    double tw = 1.0, sc = 1.0;
                    for (int k = 0; k <= FO; k++) {
                        if (k) {
                            tw *= 2.0 * alpha * alpha;
                            E = ((2 * k - 1) * E + tw * g) / s0;
                            N = (2 * k - 1) * N / s0;
                            sc *= -0.5 / k;
                        }
                        coef[k] = sc * (inblock ? (N - E) : -E);     // +erf/r inside the block, -erfc/r outside
                    }
                }
                compose(coef, delta, out);
            }
    // reciprocal space: -(1/(pi L)) sum_h h^-2 exp(-pi^2 h^2/(alpha L)^2) cos(w.u), w = 2 pi h / L
    const Tab &t = tab();
    double fact[FO + 1];
    fact[0] = 1.0;
    for (int i = 1; i <= FO; i++) fact[i] = fact[i - 1] * i;
    const int hmax = (int)ceil(sqrt(42.0) * alpha * L / PI) + 1;
    for (int hx = -hmax; hx <= hmax; hx++)
        for (int hy = -hmax; hy <= hmax; hy++)
            for (int hz = -hmax; hz <= hmax; hz++) {
                const int h2 = hx * hx + hy * hy + hz * hz;
                if (!h2) continue;
                const double ex = PI * PI * h2 / (alpha * alpha * L * L);
                if (ex > 42.0) continue;
                const double amp = -exp(-ex) / (h2 * PI * L);
                const double w[3] = {2 * PI * hx / L, 2 * PI * hy / L, 2 * PI * hz / L};
                double pwx[FO + 1], pwy[FO + 1], pwz[FO + 1];
                pwx[0] = pwy[0] = pwz[0] = 1.0;
                for (int e = 1; e <= FO; e++) { pwx[e] = pwx[e - 1] * w[0]; pwy[e] = pwy[e - 1] * w[1]; pwz[e] = pwz[e - 1] * w[2]; }
                for (int i = 0; i < NF; i++) {
                    if (t.l[i] & 1) continue;
                    const double sg = ((t.l[i] >> 1) & 1) ? -1.0 : 1.0;
                    out.c[i] += amp * sg * pwx[t.a[i]] * pwy[t.b[i]] * pwz[t.c[i]] / (fact[t.a[i]] * fact[t.b[i]] * fact[t.c[i]]);
                }
            }
    memcpy(T, out.c, sizeof(double) * NF);
}

// ---------------------------------------------------------------------------------------------------
// device
__constant__ uint8_t f_ea[NF], f_eb[NF], f_ec[NF];
static bool g_far_tables[DSK_MAXDEV];
static int far_tables()
{
    bool *done = dsk_device_flag(g_far_tables);
    if (*done) return DSK_OK;
    const Tab &t = tab();
    uint8_t a[NF], b[NF], c[NF];
    for (int i = 0; i < NF; i++) { a[i] = (uint8_t)t.a[i]; b[i] = (uint8_t)t.b[i]; c[i] = (uint8_t)t.c[i]; }
    DSK_CUDA(cudaMemcpyToSymbol(f_ea, a, NF));
    DSK_CUDA(cudaMemcpyToSymbol(f_eb, b, NF));
    DSK_CUDA(cudaMemcpyToSymbol(f_ec, c, NF));
    *done = true;
    return DSK_OK;
}

#define FM_THREADS 192
#define FM_WARPS 8
template <int I, int N, typename F>
__device__ __forceinline__ void sfor(F &&f)
{
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        sfor<I + 1, N>(f);
    }
}
// (a) block partials of the root moments about the box centre, fp64.  A thread keeps running sums of a third of
// the 165 moments (55 doubles) in registers over its particles and the block is reduced once at the end, so the inner
// loop is one DFMA per moment and particle with no shuffles; the three thirds are blockIdx.y (positions are read three
// times, 48 B per particle).  (Earlier forms: one moment per thread walking the particles serially, 3.9 ms at N = 2^21;
// one particle per lane with a butterfly sum per monomial, 0.53 ms; this one 0.1 ms.)
#define FM_PARTS 3
#define FM_PER ((NF + FM_PARTS - 1) / FM_PARTS)
template <int PART>
__device__ __forceinline__ void far_moments_part(const float4 *__restrict__ spos, uint32_t n, float half_box,
                                                 double *__restrict__ partial, double (*red)[FM_PER])
{
    constexpr int LO = PART * FM_PER, HI = (LO + FM_PER < NF) ? LO + FM_PER : NF;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double acc[FM_PER];
#pragma unroll
    for (int k = 0; k < FM_PER; k++) acc[k] = 0.0;
    const uint32_t stride = gridDim.x * FM_WARPS * 32;
    for (uint32_t i = blockIdx.x * FM_WARPS * 32 + threadIdx.x; i < n; i += stride) {
        const float4 p = spos[i];
        const double X = (double)p.x - (double)half_box, Y = (double)p.y - (double)half_box, Z = (double)p.z - (double)half_box;
        double px[FO + 1], py[FO + 1], pz[FO + 1];
        px[0] = (double)p.w; py[0] = 1.0; pz[0] = 1.0;
#pragma unroll
        for (int e = 1; e <= FO; e++) { px[e] = px[e - 1] * X; py[e] = py[e - 1] * Y; pz[e] = pz[e - 1] * Z; }
        sfor<0, FO + 1>([&](auto LL) {
            constexpr int l = decltype(LL)::value;
            sfor<0, l + 1>([&](auto KK) {
                constexpr int k = decltype(KK)::value;          // k = b + c, a = l - k
                sfor<0, k + 1>([&](auto CC) {
                    constexpr int c = decltype(CC)::value, b = k - c, a = l - k;
                    constexpr int idx = dsk_midx(a, b, c);
                    if constexpr (idx >= LO && idx < HI) acc[idx - LO] = fma(px[a], py[b] * pz[c], acc[idx - LO]);
                });
            });
        });
    }
#pragma unroll
    for (int k = 0; k < FM_PER; k++) {
        double v = acc[k];
#pragma unroll
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][k] = v;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < HI - LO; t += FM_WARPS * 32) {
        double sum = 0.0;
#pragma unroll
        for (int w = 0; w < FM_WARPS; w++) sum += red[w][t];
        partial[(size_t)blockIdx.x * NF + LO + t] = sum;
    }
}
__global__ void __launch_bounds__(FM_WARPS * 32, 1) k_far_moments(const float4 *__restrict__ spos, uint32_t n,
                                                                  float half_box, double *__restrict__ partial)
{
    __shared__ double red[FM_WARPS][FM_PER];
    if (blockIdx.y == 0) far_moments_part<0>(spos, n, half_box, partial, red);
    else if (blockIdx.y == 1) far_moments_part<1>(spos, n, half_box, partial, red);
    else far_moments_part<2>(spos, n, half_box, partial, red);
}

// (b) reduce partials, then Lambda_n = sum_{|k| <= 8-|n|} (-1)^|k| C(n+k,k) M_k T_{n+k}
// bg (reading O4b): the operator acts on the NEUTRAL box, M_k -= rho_bar int_box (y - c)^k d^3y = M_0 prod_i (L/2)^k_i / (k_i + 1)
// for even k_i (0 otherwise) — exact: the zero-mean Ewald potential integrates to 0 over the box, so int_box rho_bar Phi_far
// is the potential of the homogeneous image block, which the tree side now carries.
__global__ void __launch_bounds__(FM_THREADS) k_far_lambda(const double *__restrict__ partial, int nblk,
                                                           const double *__restrict__ T, double *__restrict__ M,
                                                           double *__restrict__ lambda, int bg, double half_box)
{
    __shared__ double sM[NF];
    __shared__ double binom[2 * FO + 1][2 * FO + 1];
    const int t = threadIdx.x;
    if (t < NF) {
        double s = 0.0;
        for (int b = 0; b < nblk; b++) s += partial[(size_t)b * NF + t];
        sM[t] = s; M[t] = s;
    }
    __syncthreads();
    const double m0 = sM[0];
    __syncthreads();
    if (bg && t < NF) {
        const int a = f_ea[t], b = f_eb[t], c = f_ec[t];
        double cube = 0.0;
        if (!((a | b | c) & 1)) cube = pow(half_box, (double)(a + b + c)) / (double)((a + 1) * (b + 1) * (c + 1));
        sM[t] -= m0 * cube;
    }
    if (t == 0)
        for (int i = 0; i <= 2 * FO; i++) {
            binom[i][0] = 1.0;
            for (int j = 1; j <= i; j++) binom[i][j] = (j == i) ? 1.0 : binom[i - 1][j - 1] + binom[i - 1][j];
        }
    __syncthreads();
    if (t < NF) {
        const int a = f_ea[t], b = f_eb[t], c = f_ec[t], l = a + b + c;
        double s = 0.0;
        for (int k = 0; k < NF; k++) {
            const int ka = f_ea[k], kb = f_eb[k], kc = f_ec[k], kl = ka + kb + kc;
            if (l + kl > FO) break;
            const double sg = (kl & 1) ? -1.0 : 1.0;
            s += sg * binom[a + ka][ka] * binom[b + kb][kb] * binom[c + kc][kc] * sM[k] * T[dsk_midx(a + ka, b + kb, c + kc)];
        }
        lambda[t] = s;
    }
}

// (c) per particle: fully unrolled evaluation of the order-8 polynomial and its gradient, in fp64 — the
// far field cancels an O(1) part of the image-block sum, so it is combined with the two-float tree sum
// in double and split back into (hi, lo).
__global__ void __launch_bounds__(128) k_far_eval(const float4 *__restrict__ spos, uint32_t n, float half_box,
                                                  const double *__restrict__ lambda, float4 *__restrict__ sacc,
                                                  float4 *__restrict__ sacc_lo)
{
    __shared__ double sl[NF];
    for (int i = threadIdx.x; i < NF; i += blockDim.x) sl[i] = lambda[i];
    __syncthreads();
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 p = spos[i];
    const double X = (double)p.x - (double)half_box, Y = (double)p.y - (double)half_box, Z = (double)p.z - (double)half_box;
    // nested Horner, innermost in Z, each level carrying the derivatives it needs: 2 FMAs per coefficient in Z,
    // 3 per (a, b) in Y, 4 per a in X (~410 DFMA per particle; the term-by-term form took ~1650 fp64 operations)
    double pot = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    sfor<0, FO + 1>([&](auto AA) {
        constexpr int a = FO - decltype(AA)::value;
        double q = 0.0, qy = 0.0, qz = 0.0;
        sfor<0, FO - a + 1>([&](auto BB) {
            constexpr int b = FO - a - decltype(BB)::value, top = FO - a - b;
            double v = sl[dsk_midx(a, b, top)], dv = 0.0;
            sfor<0, top>([&](auto CC) {
                constexpr int c = top - 1 - decltype(CC)::value;
                if constexpr (c == top - 1) dv = v;
                else dv = fma(dv, Z, v);
                v = fma(v, Z, sl[dsk_midx(a, b, c)]);
            });
            if constexpr (b == FO - a) { q = v; qz = dv; }
            else { qy = fma(qy, Y, q); q = fma(q, Y, v); qz = fma(qz, Y, dv); }
        });
        if constexpr (a == FO) { pot = q; gy = qy; gz = qz; }
        else { gx = fma(gx, X, pot); pot = fma(pot, X, q); gy = fma(gy, X, qy); gz = fma(gz, X, qz); }
    });
    const float4 h = sacc[i], l = sacc_lo[i];
    const double tx = ((double)h.x + (double)l.x) - gx, ty = ((double)h.y + (double)l.y) - gy,
                 tz = ((double)h.z + (double)l.z) - gz, tw = ((double)h.w + (double)l.w) + pot;
    float4 oh, ol;
    oh.x = (float)tx; oh.y = (float)ty; oh.z = (float)tz; oh.w = (float)tw;
    ol.x = (float)(tx - (double)oh.x); ol.y = (float)(ty - (double)oh.y); ol.z = (float)(tz - (double)oh.z);
    ol.w = (float)(tw - (double)oh.w);
    sacc[i] = oh; sacc_lo[i] = ol;
}

int dsk_run_farfield(dsk_ctx *c)
{
    int e = far_tables();
    if (e) return e;
    const uint32_t n = (uint32_t)c->N;
    int nblk = c->nsm * 2;
    if ((int64_t)nblk * FM_WARPS * 32 > c->N) nblk = (int)((c->N + FM_WARPS * 32 - 1) / (FM_WARPS * 32));
    k_far_moments<<<dim3(nblk, FM_PARTS), FM_WARPS * 32, 0, c->stream>>>(c->spos, n, 0.5f * c->box, c->far_partial);
    k_far_lambda<<<1, FM_THREADS, 0, c->stream>>>(c->far_partial, nblk, c->far_T_dev, c->far_M, c->far_lambda, c->bg, 0.5 * (double)c->box);
    k_far_eval<<<(n + 127) / 128, 128, 0, c->stream>>>(c->spos, n, 0.5f * c->box, c->far_lambda, c->sacc, c->sacc_lo);
    DSK_COUNT(c, 3);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
