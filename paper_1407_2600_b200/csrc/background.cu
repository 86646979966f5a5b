// background.cu — background subtraction in periodic boxes (reading O4b of DESIGN.md).
// PAPER.md:63 "Accuracy and error behavior have been improved significantly for cosmological volumes through the use of a
// technique to subtract the uniform background density (Warren 2013)".  Warren (2013) is not available; the reading:
// the sources of a periodic box are  delta rho = particles - rho_bar  (rho_bar = M_tot / box^3), and
//   * every cell of level <= l_b gets a second set of moments, those of delta rho over its cube about the same expansion
//     centre (the particles' centre of mass): Mhat'_n = Mhat_n - (-1)^|n| rho_bar C_n / (n! s^|n|), C_n the closed-form moments
//     of the homogeneous cube about that point.  The walk lists this copy for a cell it accepts OUTSIDE the sink group's
//     window (walk.cu); what it accepts inside the window keeps the particles' moments;
//   * the window — a cube of (w + 2k)^3 level-l_b cells around the group's cell — and the few coarse cubes the walk found
//     sticking out of it hold all the background that no accepted cell carries; their field is the closed-form Newtonian
//     field of a homogeneous cuboid, evaluated here in fp64 per sink;
//   * the far field acts on the neutral box (farfield.cu).
// Why: the monopoles of a nearly uniform box cancel to 1/100 of their size over the 125-image block, which fp32 arithmetic
// does not survive (without subtraction the monopoles are summed in fp64); the moments of delta rho are
// small, so plain fp32 does; and the truncation error at fixed theta, p drops 3x on near-lattice inputs.
#include "dsk_internal.cuh"

// ---- geometry of the cells of level <= l_b (the first ntop cells: canonical order is level-major) ----------------
__device__ __forceinline__ uint32_t bg_compact3(uint64_t x)
{   // every third bit -> 21 contiguous bits
    x &= 0x1249249249249249ull;
    x = (x | x >> 2) & 0x10c30c30c30c30c3ull;
    x = (x | x >> 4) & 0x100f00f00f00f00full;
    x = (x | x >> 8) & 0x1f0000ff0000ffull;
    x = (x | x >> 16) & 0x1f00000000ffffull;
    x = (x | x >> 32) & 0x1fffffull;
    return (uint32_t)x;
}

// topgeo[c] = (qx, qy, qz, level | octant mask of the children << 8): integer coordinates of the cell at its own level
__global__ void __launch_bounds__(256) k_top_geo(uint32_t ntop, const dsk_cellrec *__restrict__ cell,
                                                 const uint64_t *__restrict__ hotkey, int4 *__restrict__ topgeo)
{
    const uint32_t c = blockIdx.x * 256 + threadIdx.x;
    if (c >= ntop) return;
    const dsk_cellrec r = cell[c];
    const int level = (int)(r.meta >> 8), nchild = (int)(r.meta & 255u);
    const uint64_t prefix = hotkey[c] & ~(1ull << (3 * level));
    uint32_t mask = 0;
    for (int k = 0; k < nchild; k++) mask |= 1u << (uint32_t)(hotkey[r.child0 + k] & 7ull);
    topgeo[c] = make_int4((int)bg_compact3(prefix >> 2), (int)bg_compact3(prefix >> 1), (int)bg_compact3(prefix),
                          level | (int)(mask << 8));
}

// ---- masses of the cells of level <= l_b in fp64 ------------------------------------------------------------------
// delta M = M - rho_bar s^3 is a small difference: the fp32 mass of the upward pass (6e-8 M) would put back the very
// rounding error subtraction is there to remove.  Leaves and level-l_b cells sum their particles, the rest their children.
__global__ void __launch_bounds__(256) k_top_mass_leaf(uint32_t ntop, int lb, const dsk_cellrec *__restrict__ cell,
                                                       const float4 *__restrict__ spos, double *__restrict__ mass64)
{
    const uint32_t c = (blockIdx.x * 256 + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (c >= ntop) return;
    const dsk_cellrec r = cell[c];
    if ((int)(r.meta >> 8) != lb && (r.meta & 255u) != 0u) return;
    double m = 0.0;
    for (uint32_t j = r.first + lane; j < r.first + r.count; j += 32) m += (double)spos[j].w;
    for (int o = 16; o; o >>= 1) m += __shfl_xor_sync(0xffffffffu, m, o);
    if (lane == 0) mass64[c] = m;
}
__global__ void __launch_bounds__(256) k_top_mass_up(uint32_t c0, uint32_t c1, const dsk_cellrec *__restrict__ cell,
                                                     double *mass64)
{
    const uint32_t c = c0 + blockIdx.x * 256 + threadIdx.x;
    if (c >= c1) return;
    const dsk_cellrec r = cell[c];
    const uint32_t nchild = r.meta & 255u;
    if (!nchild) return;
    double m = 0.0;
    for (uint32_t k = 0; k < nchild; k++) m += mass64[r.child0 + k];
    mass64[c] = m;
}

// ---- subtracted moment rows ------------------------------------------------------------------------------------------
__constant__ uint8_t b_ea[dsk_np(DSK_PMAX)], b_eb[dsk_np(DSK_PMAX)], b_ec[dsk_np(DSK_PMAX)];
__constant__ double b_sgn_invfact[dsk_np(DSK_PMAX)];      // (-1)^|n| / (a! b! c!)
#include "cube_series.inc"              // bg_series_host[(BG_SER_H + 1)^3], written by gen_cube_series.py
__constant__ double b_series[(BG_SER_H + 1) * (BG_SER_H + 1) * (BG_SER_H + 1)];
static bool g_bg_tables[DSK_MAXDEV];
static int bg_tables()
{
    bool *done = dsk_device_flag(g_bg_tables);
    if (*done) return DSK_OK;
    constexpr int NP = dsk_np(DSK_PMAX);
    uint8_t ea[NP], eb[NP], ec[NP];
    double sif[NP], fact[DSK_PMAX + 1];
    fact[0] = 1.0;
    for (int i = 1; i <= DSK_PMAX; i++) fact[i] = fact[i - 1] * i;
    for (int l = 0; l <= DSK_PMAX; l++)
        for (int a = l; a >= 0; a--)
            for (int b = l - a; b >= 0; b--) {
                const int cc = l - a - b, i = dsk_midx(a, b, cc);
                ea[i] = (uint8_t)a; eb[i] = (uint8_t)b; ec[i] = (uint8_t)cc;
                sif[i] = ((l & 1) ? -1.0 : 1.0) / (fact[a] * fact[b] * fact[cc]);
            }
    DSK_CUDA(cudaMemcpyToSymbol(b_ea, ea, sizeof(ea)));
    DSK_CUDA(cudaMemcpyToSymbol(b_eb, eb, sizeof(eb)));
    DSK_CUDA(cudaMemcpyToSymbol(b_ec, ec, sizeof(ec)));
    DSK_CUDA(cudaMemcpyToSymbol(b_sgn_invfact, sif, sizeof(sif)));
    DSK_CUDA(cudaMemcpyToSymbol(b_series, bg_series_host, sizeof(bg_series_host)));
    *done = true;
    return DSK_OK;
}

// One warp per cell of level <= l_b.  In units of the cell side (e = (com - centre)/s):
//   C_n / s^(|n|+3) = prod_d [ (1/2 - e_d)^(n_d+1) - (-1/2 - e_d)^(n_d+1) ] / (n_d + 1)
// fp64 arithmetic, one rounding to fp32 at the end.  rho_bar = mass64[0] / box^3 (the root holds everything).
__global__ void __launch_bounds__(128) k_bg_rows(uint32_t ntop, int np, int rowlen, float box, const float *__restrict__ rows,
                                                 const double *__restrict__ mass64, float *__restrict__ rows_bg)
{
    const uint32_t c = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (c >= ntop) return;
    const float *row = rows + (size_t)c * rowlen;
    float *out = rows_bg + (size_t)c * rowlen;
    const double s = 1.0 / (double)row[3];
    const double mb = mass64[0] / ((double)box * box * box) * s * s * s;          // rho_bar s^3
    // lane 9 d + k holds the one-dimensional factor of axis d and power k (27 lanes; every lane computing all 27, each with a
    // division, was 30 x the work of the moments themselves)
    double val = 0.0;
    if (lane < 3 * (DSK_PMAX + 1)) {
        const int d = lane / (DSK_PMAX + 1), k = lane - d * (DSK_PMAX + 1);
        const double e = (double)row[4 + d] * (double)row[3];
        const double a = 0.5 - e, b = -0.5 - e;
        double pa = a, pb = b;
        for (int j = 0; j < k; j++) { pa *= a; pb *= b; }
        val = (pa - pb) / (double)(k + 1);
    }
    if (lane < 8) out[lane] = row[lane];
    for (int n0 = 0; n0 < rowlen - 8; n0 += 32) {
        const int n = n0 + lane;
        const bool live = n < np;
        const int ea = live ? b_ea[n] : 0, eb = live ? b_eb[n] : 0, ec = live ? b_ec[n] : 0;
        const double o0 = __shfl_sync(0xffffffffu, val, ea), o1 = __shfl_sync(0xffffffffu, val, (DSK_PMAX + 1) + eb),
                     o2 = __shfl_sync(0xffffffffu, val, 2 * (DSK_PMAX + 1) + ec);
        if (n < rowlen - 8) {
            float v = 0.0f;
            if (live) {
                const double cube = mb * b_sgn_invfact[n] * o0 * o1 * o2;
                const double part = n == 0 ? mass64[c] : (double)row[8 + n];
                v = (float)(part - cube);
            }
            out[8 + n] = v;
        }
    }
}

// ---- closed-form Newtonian field of a homogeneous cuboid, fp64 --------------------------------------------------------
// With r = sqrt(X^2 + Y^2 + Z^2) and (X, Y, Z) = corner - x:
//   I = int d^3y / |y - x|              = sum_corners sign F(X, Y, Z)
//   g = int (y - x)/|y - x|^3 d^3y      : g_x = - sum_corners sign G(X; Y, Z)   (the attractive field of unit density)
//   F = XY ln(Z+r) + YZ ln(X+r) + ZX ln(Y+r) - X^2/2 atan(YZ/(X r)) - Y^2/2 atan(ZX/(Y r)) - Z^2/2 atan(XY/(Z r))
//   G(X; Y, Z) = Y ln(Z+r) + Z ln(Y+r) - X atan(YZ/(X r))
// sign = product over the axes of (+ upper, - lower).  A term whose prefactor is 0 is dropped (its limit is 0: sinks of a
// perfect lattice lie exactly on the planes and edges of the cubes); ln(Z + r) for Z < 0 is ln(rho^2 / (r - Z)).
__device__ __forceinline__ double bg_log_zr(double z, double r, double rho2) { return z >= 0.0 ? log(z + r) : log(rho2 / (r - z)); }

template <bool POT>
__device__ __forceinline__ void bg_cuboid(const double lo[3], const double hi[3], double x, double y, double z, double &I,
                                          double &gx, double &gy, double &gz)
{
    I = 0.0; gx = gy = gz = 0.0;
#pragma unroll 1
    for (int corner = 0; corner < 8; corner++) {
        const int i = corner >> 2, j = (corner >> 1) & 1, k = corner & 1;
        const double X = (i ? hi[0] : lo[0]) - x, Y = (j ? hi[1] : lo[1]) - y, Z = (k ? hi[2] : lo[2]) - z;
        const double sg = ((i + j + k) & 1) ? 1.0 : -1.0;
        const double X2 = X * X, Y2 = Y * Y, Z2 = Z * Z, r = sqrt(X2 + Y2 + Z2);
        const double lx = (Y2 + Z2 > 0.0) ? bg_log_zr(X, r, Y2 + Z2) : 0.0;       // ln(X + r); its prefactors vanish with Y^2 + Z^2
        const double ly = (Z2 + X2 > 0.0) ? bg_log_zr(Y, r, Z2 + X2) : 0.0;
        const double lz = (X2 + Y2 > 0.0) ? bg_log_zr(Z, r, X2 + Y2) : 0.0;
        const double ax = X != 0.0 ? atan(Y * Z / (X * r)) : 0.0;
        const double ay = Y != 0.0 ? atan(Z * X / (Y * r)) : 0.0;
        const double az = Z != 0.0 ? atan(X * Y / (Z * r)) : 0.0;
        gx -= sg * (Y * lz + Z * ly - X * ax);
        gy -= sg * (Z * lx + X * lz - Y * ay);
        gz -= sg * (X * ly + Y * lx - Z * az);
        if (POT) I += sg * (X * Y * lz + Y * Z * lx + Z * X * ly - 0.5 * (X2 * ax + Y2 * ay + Z2 * az));
    }
}

// ---- the same field INSIDE a cube, well away from its faces: Taylor series about the centre -----------------------------------
// Phi(u) = int d^3y / |y - u| over the unit-density cube [-1,1]^3 = sum_{i+j+k <= H} C_ijk a^i b^j c^k with a, b, c = u1^2, u2^2, u3^2
// (gen_cube_series.py: exact derivatives of 1/r at the corners, one quadrature along the edges, Laplace's equation for the rest).
// The series of the harmonic part converges inside the sphere through the edges, |u| < sqrt 2: truncated at degree 2H = 14 it is
// good to 1e-13 for |u|_inf <= 0.21, at 22 for |u|_inf <= 0.36 (checked against the closed form by the generator) - 0.5 k and
// 1.2 k DFMA per sink where the closed form takes eight corners x (3 log + 3 atan + sqrt + divisions) ~ 5 k instructions.
// Returns Phi and grad_u Phi; for a cube of half-width h about ctr: I = h^2 Phi(u), g = grad_x I = h grad_u Phi, u = (x - ctr)/h.
template <int H, bool POT>
__device__ __forceinline__ void bg_cube_series(double u1, double u2, double u3, double &phi, double &g1, double &g2, double &g3)
{
    constexpr int S = BG_SER_H + 1;
    const double a = u1 * u1, b = u2 * u2, c = u3 * u3;
    double pa[H + 1], pb[H + 1];
    pa[0] = 1.0; pb[0] = 1.0;
#pragma unroll
    for (int i = 1; i <= H; i++) { pa[i] = pa[i - 1] * a; pb[i] = pb[i - 1] * b; }
    double da = 0.0, db = 0.0, dc = 0.0, ph = 0.0;      // dPhi/da, dPhi/db, dPhi/dc, Phi
#pragma unroll
    for (int i = 0; i <= H; i++)
#pragma unroll
        for (int j = 0; j <= H - i; j++) {
            // Horner in c with the derivative: p = sum_k C_ijk c^k, dp = dp/dc
            const int K = H - i - j;
            double p = b_series[(i * S + j) * S + K], dp = 0.0;
#pragma unroll
            for (int k = K - 1; k >= 0; k--) { dp = fma(dp, c, p); p = fma(p, c, b_series[(i * S + j) * S + k]); }
            const double ab = pa[i] * pb[j];
            if (POT) ph = fma(ab, p, ph);
            dc = fma(ab, dp, dc);
            if (i) da = fma((double)i * pa[i - 1] * pb[j], p, da);
            if (j) db = fma((double)j * pa[i] * pb[j - 1], p, db);
        }
    phi = ph; g1 = 2.0 * u1 * da; g2 = 2.0 * u2 * db; g3 = 2.0 * u3 * dc;
}

// the window of group g: inclusive index range in level-l_b cells (unwrapped frame of the home image)
__device__ __forceinline__ void bg_window(uint32_t cg, int lb, int k, const dsk_cellrec *__restrict__ cell,
                                          const uint64_t *__restrict__ hotkey, int wlo[3], int whi[3])
{
    const int lg = (int)(cell[cg].meta >> 8);
    const uint64_t prefix = hotkey[cg] & ~(1ull << (3 * lg));
    const int q[3] = {(int)bg_compact3(prefix >> 2), (int)bg_compact3(prefix >> 1), (int)bg_compact3(prefix)};
#pragma unroll
    for (int d = 0; d < 3; d++) {
        int flo, fhi;
        if (lg >= lb) flo = fhi = q[d] >> (lg - lb);
        else { flo = q[d] << (lb - lg); fhi = flo + (1 << (lb - lg)) - 1; }
        wlo[d] = flo - k; whi[d] = fhi + k;
    }
}

__device__ __forceinline__ void bg_add(float4 *__restrict__ sacc, float4 *__restrict__ sacc_lo, uint32_t r, double ax, double ay,
                                       double az, double ph)
{
    const float4 h = sacc[r], l = sacc_lo[r];
    const double tx = ((double)h.x + (double)l.x) + ax, ty = ((double)h.y + (double)l.y) + ay,
                 tz = ((double)h.z + (double)l.z) + az, tw = ((double)h.w + (double)l.w) + ph;
    float4 oh, ol;
    oh.x = (float)tx; oh.y = (float)ty; oh.z = (float)tz; oh.w = (float)tw;
    ol.x = (float)(tx - (double)oh.x); ol.y = (float)(ty - (double)oh.y); ol.z = (float)(tz - (double)oh.z);
    ol.w = (float)(tw - (double)oh.w);
    sacc[r] = oh; sacc_lo[r] = ol;
}

// the window's background at every sink: acc -= rho_bar g(W), pot += rho_bar I(W).  One thread per sink, a warp per 32
// consecutive sinks of one group (the corner loop is uniform; the window is the group's).
// Sinks lie inside the group's cell, hence within w / (w + 2k) of the window's half-width from its centre (w = the footprint of
// the group's cell in level-l_b cells): the series of order 14 up to 0.21 (k >= 2 for a group at or below level l_b), of order
// 22 up to 0.36 (k = 1), the closed form beyond (groups above level l_b: sparse regions), or everywhere with closed != 0.
template <bool POT>
__global__ void __launch_bounds__(128) k_bg_window(uint32_t ngroup, int lb, int k, float box, int closed, const double *__restrict__ mass64,
                                                   const uint32_t *__restrict__ gfirst, const uint32_t *__restrict__ gcount,
                                                   const uint32_t *__restrict__ gcell, const uint8_t *__restrict__ gact,
                                                   const dsk_cellrec *__restrict__ cell, const uint64_t *__restrict__ hotkey,
                                                   const float4 *__restrict__ spos, float4 *__restrict__ sacc,
                                                   float4 *__restrict__ sacc_lo)
{
    const uint32_t g = (blockIdx.x * 128 + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (g >= ngroup) return;
    if (gact && !gact[g]) return;
    int wlo[3], whi[3];
    bg_window(gcell[g], lb, k, cell, hotkey, wlo, whi);
    const double sb = (double)box * exp2((double)-lb), rho = mass64[0] / ((double)box * box * box);
    const double lo[3] = {wlo[0] * sb, wlo[1] * sb, wlo[2] * sb}, hi[3] = {(whi[0] + 1) * sb, (whi[1] + 1) * sb, (whi[2] + 1) * sb};
    const uint32_t f = gfirst[g], n = gcount[g];
    const int side = whi[0] - wlo[0] + 1, w = side - 2 * k;                 // the window is a cube: w + 2k cells a side
    const double h = 0.5 * side * sb, ctr[3] = {0.5 * (lo[0] + hi[0]), 0.5 * (lo[1] + hi[1]), 0.5 * (lo[2] + hi[2])}, hinv = 1.0 / h;
    const int form = closed ? 0 : (100 * w <= 21 * side ? 1 : (100 * w <= 36 * side ? 2 : 0));
    for (uint32_t j = lane; j < n; j += 32) {
        const float4 p = spos[f + j];
        double I, gx, gy, gz;
        if (form == 0) bg_cuboid<POT>(lo, hi, (double)p.x, (double)p.y, (double)p.z, I, gx, gy, gz);
        else {
            const double u1 = ((double)p.x - ctr[0]) * hinv, u2 = ((double)p.y - ctr[1]) * hinv, u3 = ((double)p.z - ctr[2]) * hinv;
            if (form == 1) bg_cube_series<7, POT>(u1, u2, u3, I, gx, gy, gz);
            else bg_cube_series<BG_SER_H, POT>(u1, u2, u3, I, gx, gy, gz);
            I *= h * h; gx *= h; gy *= h; gz *= h;
        }
        bg_add(sacc, sacc_lo, f + j, -rho * gx, -rho * gy, -rho * gz, rho * I);
    }
}

// The cubes kept outside the window (the walk's third list, one record per cube: the inclusive index range in level-l_b cells
// packed as lo | hi << 16 per axis): for every sink of the group, cube minus (cube intersected with the window).  One warp per
// group, after the group's P2P and M2P tasks on the same stream, so nothing else touches its sinks' accumulators.
template <bool POT>
__global__ void __launch_bounds__(128) k_bg_left(uint32_t g0, uint32_t g1, const uint4 *__restrict__ list, const uint64_t *__restrict__ off,
                                                 uint64_t base, const uint32_t *__restrict__ len, int lb, int k, float box,
                                                 const double *__restrict__ mass64, const uint32_t *__restrict__ gfirst,
                                                 const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ gcell,
                                                 const dsk_cellrec *__restrict__ cell, const uint64_t *__restrict__ hotkey,
                                                 const float4 *__restrict__ spos, float4 *__restrict__ sacc,
                                                 float4 *__restrict__ sacc_lo)
{
    const uint32_t g = g0 + ((blockIdx.x * 128 + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    if (g >= g1) return;
    const uint32_t nrec = len[g];
    if (!nrec) return;
    const double sb = (double)box * exp2((double)-lb), rho = mass64[0] / ((double)box * box * box);
    int wlo[3], whi[3];
    bg_window(gcell[g], lb, k, cell, hotkey, wlo, whi);
    const uint32_t f = gfirst[g], n = gcount[g];
    const uint4 *rec = list + (off[g] - base);
    for (uint32_t j = lane; j < n; j += 32) {
        const float4 p = spos[f + j];
        double ax = 0.0, ay = 0.0, az = 0.0, ph = 0.0;
        for (uint32_t q = 0; q < nrec; q++) {
            const uint4 r = rec[q];
            const int clo[3] = {(int)(short)(r.x & 0xffffu), (int)(short)(r.y & 0xffffu), (int)(short)(r.z & 0xffffu)};
            const int chi[3] = {(int)(short)(r.x >> 16), (int)(short)(r.y >> 16), (int)(short)(r.z >> 16)};
            double lo[3], hi[3], olo[3], ohi[3];
            bool overlap = true;
#pragma unroll
            for (int d = 0; d < 3; d++) {
                lo[d] = clo[d] * sb; hi[d] = (chi[d] + 1) * sb;
                const int ol = max(clo[d], wlo[d]), oh = min(chi[d], whi[d]);
                if (ol > oh) overlap = false;
                olo[d] = ol * sb; ohi[d] = (oh + 1) * sb;
            }
            double I, gx, gy, gz;
            bg_cuboid<POT>(lo, hi, (double)p.x, (double)p.y, (double)p.z, I, gx, gy, gz);
            if (overlap) {
                double I2, hx, hy, hz;
                bg_cuboid<POT>(olo, ohi, (double)p.x, (double)p.y, (double)p.z, I2, hx, hy, hz);
                I -= I2; gx -= hx; gy -= hy; gz -= hz;
            }
            ax -= rho * gx; ay -= rho * gy; az -= rho * gz; ph += rho * I;
        }
        bg_add(sacc, sacc_lo, f + j, ax, ay, az, ph);
    }
}

// ---- host ---------------------------------------------------------------------------------------------------------------
int dsk_bg_level(int64_t n)
{
    int lg = 0;
    while ((n >> (lg + 1)) > 0) lg++;
    int l = lg < 6 ? 0 : (lg - 6) / 3;
    return l < 2 ? 2 : l;
}
int dsk_bg_halfwidth(float theta, int lb, int ws)
{
    const int k = (int)ceil(1.0 / (double)theta), kmax = ws << lb;
    return k < kmax ? k : kmax;
}

// after the upward pass of a periodic context with subtraction on: geometry, fp64 masses, subtracted rows, their force rows
int dsk_run_bg_rows(dsk_ctx *c)
{
    int e = bg_tables();
    if (e) return e;
    const uint32_t *ls = c->hstate->lvl_start;
    const int lb = c->bg_level;
    const uint32_t ntop = ls[lb + 1 <= DSK_KEY_LEVELS + 2 ? lb + 1 : DSK_KEY_LEVELS + 2];
    if ((int64_t)ntop > c->ntop_cap) return DSK_ECELLOVERFLOW;
    c->ntop = ntop;
    cudaStream_t s = c->stream;
    k_top_geo<<<(ntop + 255) / 256, 256, 0, s>>>(ntop, c->cell, c->hotkey, c->topgeo);
    k_top_mass_leaf<<<(unsigned)(((size_t)ntop * 32 + 255) / 256), 256, 0, s>>>(ntop, lb, c->cell, c->spos, c->mass64);
    int nl = 0;
    for (int l = lb - 1; l >= 0; l--) {
        const uint32_t c0 = ls[l], c1 = ls[l + 1];
        if (c1 <= c0) continue;
        k_top_mass_up<<<(c1 - c0 + 255) / 256, 256, 0, s>>>(c0, c1, c->cell, c->mass64);
        nl++;
    }
    k_bg_rows<<<(ntop + 3) / 4, 128, 0, s>>>(ntop, dsk_np(c->p), dsk_rowlen(c->p), c->box, c->rows, c->mass64, c->rows_bg);
    DSK_COUNT(c, 3 + nl);
    e = dsk_run_frows_bg(c, ntop);
    if (e) return e;
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// after P2P + M2P of all batches: the exact background of every group's window
int dsk_run_bg_window(dsk_ctx *c, int want_pot)
{
    const uint32_t ng = c->hstate->ngroup;
    cudaStream_t s = c->stream;
    const int k = dsk_bg_halfwidth(c->theta, c->bg_level, c->img_ws);
    const unsigned nb = (unsigned)(((size_t)ng * 32 + 127) / 128);
    if (want_pot)
        k_bg_window<true><<<nb, 128, 0, s>>>(ng, c->bg_level, k, c->box, c->bg_closed, c->mass64, c->gfirst, c->gcount, c->gcell, c->gact_cur,
                                             c->cell, c->hotkey, c->spos, c->sacc, c->sacc_lo);
    else
        k_bg_window<false><<<nb, 128, 0, s>>>(ng, c->bg_level, k, c->box, c->bg_closed, c->mass64, c->gfirst, c->gcount, c->gcell, c->gact_cur,
                                              c->cell, c->hotkey, c->spos, c->sacc, c->sacc_lo);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// per batch of groups, after its M2P: the cubes the walk kept outside the windows (usually none)
int dsk_run_bg_left(dsk_ctx *c, uint32_t g0, uint32_t g1, uint64_t base, int want_pot)
{
    if (g1 <= g0) return DSK_OK;
    cudaStream_t s = c->stream;
    const int k = dsk_bg_halfwidth(c->theta, c->bg_level, c->img_ws);
    const unsigned nb = (unsigned)(((size_t)(g1 - g0) * 32 + 127) / 128);
    if (want_pot)
        k_bg_left<true><<<nb, 128, 0, s>>>(g0, g1, c->list_left, c->g_left_off, base, c->g_left_len, c->bg_level, k, c->box, c->mass64,
                                           c->gfirst, c->gcount, c->gcell, c->cell, c->hotkey, c->spos, c->sacc, c->sacc_lo);
    else
        k_bg_left<false><<<nb, 128, 0, s>>>(g0, g1, c->list_left, c->g_left_off, base, c->g_left_len, c->bg_level, k, c->box, c->mass64,
                                            c->gfirst, c->gcount, c->gcell, c->cell, c->hotkey, c->spos, c->sacc, c->sacc_lo);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// raw subtracted moments in units of the cell side, M'_n / s^|n| (parity tests)
__global__ void k_get_bg_moments(uint32_t ntop, int np, int rowlen, const float *__restrict__ rows_bg, float *__restrict__ mom)
{
    const uint32_t c = blockIdx.x;
    if (c >= ntop) return;
    for (int n = threadIdx.x; n < np; n += blockDim.x)
        mom[(size_t)c * np + n] = (float)((double)rows_bg[(size_t)c * rowlen + 8 + n] / b_sgn_invfact[n]);
}
int dsk_run_get_bg_moments(dsk_ctx *c, float *moments)
{
    if (!c->ntop) return DSK_OK;
    k_get_bg_moments<<<c->ntop, 64, 0, c->stream>>>(c->ntop, dsk_np(c->p), dsk_rowlen(c->p), c->rows_bg, moments);
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}
