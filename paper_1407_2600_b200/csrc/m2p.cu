// m2p.cu — step F2: cell-particle (M2P) evaluation of the interaction lists, and the "force rows" it reads.
// DESIGN.md O6 / section 5.1 (PAPER.md:71 m x n blocks of source cells against the sinks of one sink cell;
// PAPER.md:75 quadrupole / hexadecapole cell interactions).
//
// The order-p field of a cell, pot = -sum_{|n|<=p} (-1)^|n| M_n d^n g / n!, g = (|r|^2+eps^2)^(-1/2), is
// evaluated in the PAIRING FORM ("any algebraically equal arrangement"): every derivative
// of a function of R^2 = |r|^2 + eps^2 is a sum over pairings of indices,
//     M^(l) . d^(l) g = sum_k  l!/(2^k k! (l-2k)!)  f_{l-k}(R)  (Tr^k M^(l)) . r^(l-2k),
//     f_m(R) = (-1)^m (2m-1)!! R^-(2m+1)            (d_i f_m = r_i f_{m+1}),
// so with the scaled monomials mu_j = rho^j / j! (d_i mu_j = mu_{j-e_i}) and per-cell coefficients
//     B^(q,m)_j = c_m 2^-k sum_{|t|=k} (j+2t)!/t! Mhat_{j+2t},   |j| = q, k = m - q, l = 2m - q <= p,
//     c_m = (-1)^m (2m-1)!!,  Mhat_n = (-1)^|n| M_n / (n! s^|n|)  (the upward pass's row),
// the sums S_m = sum_q sum_j B^(q,m)_j mu_j and their gradients G_m,i = sum B^(q,m)_j mu_{j-e_i} give
//     pot = -(1/s) sum_m h_m S_m ,
//     acc_i = (1/s^2) [ sum_m h_m G_m,i - rho_i q sum_m (2m+1) h_m S_m ],  h_m = R^-(2m+1), q = 1/R^2,
// in cell-scaled coordinates rho = r/s, eps~ = eps/s.  This needs about half the FP32 instructions of the
// derivative recurrence (p = 4: 188 against ~410 per interaction) and holds only two degrees of monomials
// in registers.  The coefficients ("force row") are a fixed linear map of the moment row, applied once per
// cell after the upward pass by k_frows.  The dipole (l = 1) vanishes about the centre of mass and is skipped.
#include "force_task.cuh"
#include <vector>

// ---- force-row layout: header of 8 floats as in the moment row, then blocks (q, m) in q-major order ----
__host__ __device__ constexpr bool fr_has(int P, int q, int m) { return m >= q && 2 * m - q <= P && !(q == 1 && m == 1); }
__host__ __device__ constexpr int fr_bsize(int q) { return (q + 1) * (q + 2) / 2; }
__host__ __device__ constexpr int fr_off(int P, int q, int m)
{
    int o = 0;
    for (int qq = 0; qq <= P; qq++)
        for (int mm = qq; mm <= P; mm++) {
            if (qq == q && mm == m) return o;
            if (qq > q) return o;
            if (fr_has(P, qq, mm)) o += fr_bsize(qq);
        }
    return o;
}
__host__ __device__ constexpr int fr_nc(int P) { return fr_off(P, P + 1, 0); }
__host__ __device__ constexpr int fr_rowlen(int P) { return (8 + fr_nc(P) + 3) / 4 * 4; }
__host__ __device__ constexpr int fr_qfirst_S(int P, int m) { return (m == 1 || 2 * m - P < 0) ? 0 : 2 * m - P; }
__host__ __device__ constexpr int fr_qfirst_G(int P, int m) { return 2 * m - P < 1 ? 1 : 2 * m - P; }

int dsk_frow_len(int p) { return p == 2 ? fr_rowlen(2) : p == 4 ? fr_rowlen(4) : p == 6 ? fr_rowlen(6) : fr_rowlen(8); }

// ---- k_frows: moment row -> force row -------------------------------------------------------------------
struct fr_entry { uint32_t src; float w; };

static void build_frow_table(int P, std::vector<uint32_t> &beg, std::vector<fr_entry> &ent)
{
    double fact[2 * DSK_PMAX + 2];
    fact[0] = 1.0;
    for (int i = 1; i < 2 * DSK_PMAX + 2; i++) fact[i] = fact[i - 1] * i;
    beg.clear(); ent.clear();
    for (int q = 0; q <= P; q++)
        for (int m = q; m <= P; m++) {
            if (!fr_has(P, q, m)) continue;
            const int k = m - q;
            double cm = (m & 1) ? -1.0 : 1.0;
            for (int i = 2 * m - 1; i > 0; i -= 2) cm *= i;
            for (int a = q; a >= 0; a--)
                for (int b = q - a; b >= 0; b--) {
                    const int c = q - a - b;
                    beg.push_back((uint32_t)ent.size());
                    for (int ta = k; ta >= 0; ta--)
                        for (int tb = k - ta; tb >= 0; tb--) {
                            const int tc = k - ta - tb;
                            const int na = a + 2 * ta, nb = b + 2 * tb, nc = c + 2 * tc;
                            const double w = cm * ldexp(1.0, -k) * fact[na] * fact[nb] * fact[nc] /
                                             (fact[ta] * fact[tb] * fact[tc]);
                            ent.push_back(fr_entry{(uint32_t)dsk_midx(na, nb, nc), (float)w});
                        }
                }
        }
    beg.push_back((uint32_t)ent.size());
}

__global__ void __launch_bounds__(128) k_frows(uint32_t ncell, int rowlen, int frowlen, int nc,
                                               const uint32_t *__restrict__ beg, const fr_entry *__restrict__ ent,
                                               const float *__restrict__ rows, float *__restrict__ frows)
{
    const uint32_t c = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (c >= ncell) return;
    const float *row = rows + (size_t)c * rowlen;
    float *fr = frows + (size_t)c * frowlen;
    if (lane < 8) fr[lane] = row[lane];
    for (int i = lane; i < frowlen - 8; i += 32) {
        float v = 0.0f;
        if (i < nc)
            for (uint32_t e = beg[i]; e < beg[i + 1]; e++) v = fmaf(ent[e].w, row[8 + ent[e].src], v);
        fr[8 + i] = v;
    }
}

int dsk_run_frows(dsk_ctx *c)
{
    const int P = c->p, nc = P == 2 ? fr_nc(2) : P == 4 ? fr_nc(4) : P == 6 ? fr_nc(6) : fr_nc(8);
    if (c->frow_tab_p != P) {
        std::vector<uint32_t> beg;
        std::vector<fr_entry> ent;
        build_frow_table(P, beg, ent);
        if (beg.size() > DSK_FRTAB_BEG || ent.size() > DSK_FRTAB_ENT) return DSK_EINVAL;
        DSK_CUDA(cudaMemcpyAsync(c->frtab_beg, beg.data(), beg.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
        DSK_CUDA(cudaMemcpyAsync(c->frtab_ent, ent.data(), ent.size() * sizeof(fr_entry), cudaMemcpyHostToDevice, c->stream));
        DSK_CUDA(cudaStreamSynchronize(c->stream));      // the vectors die here
        c->frow_tab_p = P;
    }
    const uint32_t n = c->hstate->ncell;
    k_frows<<<(n + 3) / 4, 128, 0, c->stream>>>(n, dsk_rowlen(P), dsk_frow_len(P), nc, c->frtab_beg,
                                                (const fr_entry *)c->frtab_ent, c->rows, c->frows);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

// ---- F2 body: one sink against one cell (float) or a pair of cells (f2) ------------------------------
// tile row (float2 = {cell A, cell B}): [0..2] com' xyz, [3] 1/s, [4] eps^2/s^2, [5] -1/s^2, [6+i] B_i
#define M2P_HDR 6
template <typename T> __device__ __forceinline__ void vld2(const float2 *p, int half, T &a, T &b);
template <> __device__ __forceinline__ void vld2<f2>(const float2 *p, int, f2 &a, f2 &b)
{
    const ulonglong2 v = *reinterpret_cast<const ulonglong2 *>(p);
    a.v = v.x; b.v = v.y;
}
template <> __device__ __forceinline__ void vld2<float>(const float2 *p, int half, float &a, float &b)
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    a = half ? v.y : v.x; b = half ? v.w : v.z;
}

__host__ __device__ constexpr int mi_comp(MI j, int i) { return i == 0 ? j.a : (i == 1 ? j.b : j.c); }
__host__ __device__ constexpr int mi_lower(MI j, int i)
{
    return dsk_midx(j.a - (i == 0), j.b - (i == 1), j.c - (i == 2));
}
// the non-zero component with the smallest value (monomial mu_j = mu_{j-e_i} * rho_i / j_i)
__host__ __device__ constexpr int mi_pick(MI j)
{
    int best = -1, bv = 1 << 30;
    for (int i = 0; i < 3; i++) {
        const int v = mi_comp(j, i);
        if (v >= 1 && v < bv) { bv = v; best = i; }
    }
    return best;
}

template <int P, typename T, bool POT>
__device__ __forceinline__ void m2p_body(T xs, T ys, T zs, const float2 *__restrict__ row, int half,
                                         T &pot, T &ax, T &ay, T &az)
{
    constexpr int NP = dsk_np(P);
    T cx, cy, cz, sinv, e2s, nsinv2;
    vld2<T>(row + 0, half, cx, cy); vld2<T>(row + 2, half, cz, sinv); vld2<T>(row + 4, half, e2s, nsinv2);
    T rho[3];
    rho[0] = vmul(vsub(xs, cx), sinv); rho[1] = vmul(vsub(ys, cy), sinv); rho[2] = vmul(vsub(zs, cz), sinv);
    T R2 = vfma(rho[0], rho[0], e2s);
    R2 = vfma(rho[1], rho[1], R2);
    R2 = vfma(rho[2], rho[2], R2);
    const T h0 = vrsqrt(R2);
    const T qi = vmul(h0, h0);
    T rd[3][P + 1];                    // rho_i / k
#pragma unroll
    for (int i = 0; i < 3; i++) {
        rd[i][1] = rho[i];
        static_for<2, P + 1>([&](auto K) {
            constexpr int k = decltype(K)::value;
            rd[i][k] = vmul(rho[i], vdup<T>(1.0f / (float)k));
        });
    }
    T mu[NP];                          // scaled monomials rho^j / j!  (mu[0] = 1 is never read)
    mu[1] = rho[0]; mu[2] = rho[1]; mu[3] = rho[2];
    T S[P + 1], G[P + 1][3];
    const float2 *Bp = row + M2P_HDR;
    T bc, bn;                          // coefficients arrive two at a time (one LDS.128)
    static_for<0, P + 1>([&](auto Q) {
        constexpr int q = decltype(Q)::value;
        constexpr int base = q * (q + 1) * (q + 2) / 6;
        if constexpr (q >= 2)
            static_for<0, fr_bsize(q)>([&](auto JJ) {
                constexpr MI j = dsk_mi(base + decltype(JJ)::value);
                constexpr int i = mi_pick(j);
                mu[base + decltype(JJ)::value] = vmul(mu[mi_lower(j, i)], rd[i][mi_comp(j, i)]);
            });
        static_for<q, P + 1>([&](auto M) {
            constexpr int m = decltype(M)::value;
            if constexpr (fr_has(P, q, m)) {
                constexpr int off = fr_off(P, q, m);
                static_for<0, fr_bsize(q)>([&](auto JJ) {
                    constexpr int jj = decltype(JJ)::value, ci = off + jj;
                    T B;
                    if constexpr (ci % 2 == 0) { vld2<T>(Bp + ci, half, bc, bn); B = bc; }
                    else B = bn;
                    if constexpr (q == 0) S[m] = B;
                    else if constexpr (q == fr_qfirst_S(P, m) && jj == 0) S[m] = vmul(B, mu[base + jj]);
                    else S[m] = vfma(B, mu[base + jj], S[m]);
                    if constexpr (m >= 2 && q >= 1)
                        static_for<0, 3>([&](auto I) {
                            constexpr int i = decltype(I)::value;
                            constexpr MI ji = dsk_mi(base + jj);
                            if constexpr (mi_comp(ji, i) >= 1) {
                                if constexpr (q == 1) G[m][i] = B;
                                else if constexpr (q == fr_qfirst_G(P, m) && jj == i) G[m][i] = vmul(B, mu[mi_lower(ji, i)]);
                                else G[m][i] = vfma(B, mu[mi_lower(ji, i)], G[m][i]);
                            }
                        });
                });
            }
        });
    });
    // pot = -(1/s) sum_m h_m S_m ;  acc_i = (1/s^2) [ sum_m h_m G_m,i - rho_i q sum_m (2m+1) h_m S_m ]
    T h = h0;
    T phi = vmul(h, S[0]);
    T tt = phi;
    T g[3];
    static_for<1, P + 1>([&](auto M) {
        constexpr int m = decltype(M)::value;
        h = vmul(h, qi);
        const T w = vmul(h, S[m]);
        if constexpr (POT) phi = vadd(phi, w);
        tt = vfma(w, vdup<T>((float)(2 * m + 1)), tt);
        if constexpr (m == 2) { g[0] = vmul(h, G[m][0]); g[1] = vmul(h, G[m][1]); g[2] = vmul(h, G[m][2]); }
        else if constexpr (m > 2) {
            g[0] = vfma(h, G[m][0], g[0]); g[1] = vfma(h, G[m][1], g[1]); g[2] = vfma(h, G[m][2], g[2]);
        }
    });
    const T sinv2 = vmul(sinv, sinv);
    const T u = vmul(vmul(qi, tt), nsinv2);
    ax = vfma(g[0], sinv2, ax); ay = vfma(g[1], sinv2, ay); az = vfma(g[2], sinv2, az);
    ax = vfma(rho[0], u, ax); ay = vfma(rho[1], u, ay); az = vfma(rho[2], u, az);
    if constexpr (POT) pot = vfma(phi, sinv, pot);        // caller subtracts
}

// ---- F2 kernel ------------------------------------------------------------------------------------------
// Per warp: a tile of up to NPAIR cell pairs in shared memory, PAIR-INTERLEAVED ({cell A, cell B} per float2) so
// one broadcast LDS.128 feeds two packed f32x2 operands.  Staging: one lane per listed cell builds the header
// (centre of mass relative to the sink group's cell centre, image shift absorbed exactly), then the lanes
// copy the coefficient rows 16 bytes at a time (2 LDG.128 -> 2 STS.128 per pair and chunk).
template <int P> struct m2p_cfg {
    static constexpr int NPAIR = (P <= 6) ? 16 : 8;
    static constexpr int FROW = fr_rowlen(P);
    static constexpr int NCH = (FROW - 8) / 4;             // 16-byte chunks of coefficients per cell
    static constexpr int TROW = M2P_HDR + (FROW - 8);      // float2 per pair row
    static constexpr size_t WARP_BYTES = (size_t)NPAIR * TROW * sizeof(float2) + 32 * sizeof(uint32_t);
    static constexpr bool PACKED = (P <= 6);
};

template <int P, bool POT>
__global__ void __launch_bounds__(FW * 32) k_m2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic,
                                                 float box, float eps2, const float *__restrict__ frows,
                                                 const float4 *__restrict__ spos, const uint32_t *__restrict__ gfirst,
                                                 const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ gcell,
                                                 const uint32_t *__restrict__ list, const uint64_t *__restrict__ off,
                                                 uint64_t base, const uint32_t *__restrict__ len,
                                                 float4 *__restrict__ sacc, float4 *__restrict__ sacc_lo)
{
    using C = m2p_cfg<P>;
    constexpr int NPAIR = C::NPAIR, FROW = C::FROW, NCH = C::NCH, TROW = C::TROW;
    constexpr bool PACKED = C::PACKED;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const warp_task t = make_task(t0, t1, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float2(*tile)[TROW] = reinterpret_cast<float2(*)[TROW]>(smem_raw + (size_t)warp * C::WARP_BYTES);
    uint32_t *s_cell = reinterpret_cast<uint32_t *>(smem_raw + (size_t)warp * C::WARP_BYTES + (size_t)NPAIR * TROW * sizeof(float2));
    const float *grow = frows + (size_t)gcell[t.g] * FROW;
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
    // pairs per tile: a multiple of the number of sub-groups, so that they finish together
    const int tp = t.S >= NPAIR ? NPAIR : (NPAIR / t.S) * t.S;
    const uint32_t tc = 2u * (uint32_t)tp;                  // cells per tile (<= 32: one list entry per lane)
    for (uint32_t b0 = 0; b0 < n; b0 += tc) {
        const int ntc = (int)min(tc, n - b0);
        const int npair = (ntc + 1) >> 1;
        if (lane < 2 * npair) {
            float cx = 4.0f * box, cy = cx, cz = cx, sinv = 1.0f / box;     // dummy cell: away from every sink, no mass
            uint32_t cidx = 0xffffffffu;
            if (lane < ntc) {
                const uint32_t e = lst[b0 + lane];
                cidx = e & ((1u << DSK_CELL_BITS) - 1u);
                const float *r = frows + (size_t)cidx * FROW;
                const float4 h0 = __ldg(reinterpret_cast<const float4 *>(r));
                const float4 h1 = __ldg(reinterpret_cast<const float4 *>(r + 4));
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
            hd[0] = cx; hd[2] = cy; hd[4] = cz; hd[6] = sinv; hd[8] = eps2 * sinv * sinv; hd[10] = -sinv * sinv;
        }
        __syncwarp();
        for (int idx = lane; idx < npair * NCH; idx += 32) {
            const int k = idx / NCH, ch = idx - k * NCH;
            const uint32_t ca = s_cell[2 * k], cb = s_cell[2 * k + 1];
            float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a;
            if (ca != 0xffffffffu) a = __ldg(reinterpret_cast<const float4 *>(frows + (size_t)ca * FROW + 8) + ch);
            if (cb != 0xffffffffu) b = __ldg(reinterpret_cast<const float4 *>(frows + (size_t)cb * FROW + 8) + ch);
            float4 *dst = reinterpret_cast<float4 *>(&tile[k][M2P_HDR + 4 * ch]);
            dst[0] = make_float4(a.x, b.x, a.y, b.y);
            dst[1] = make_float4(a.z, b.z, a.w, b.w);
        }
        __syncwarp();
        if (t.active) {
            T pot = vdup<T>(0.0f), ax = vdup<T>(0.0f), ay = vdup<T>(0.0f), az = vdup<T>(0.0f);
            if constexpr (PACKED) {
                for (int k = t.sub; k < npair; k += t.S) m2p_body<P, T, POT>(X, Y, Z, tile[k], 0, pot, ax, ay, az);
            } else {
                for (int k = t.sub; k < 2 * npair; k += t.S) m2p_body<P, T, POT>(X, Y, Z, tile[k >> 1], k & 1, pot, ax, ay, az);
            }
            dsk_fold(hi.x, lo.x, vsum(ax)); dsk_fold(hi.y, lo.y, vsum(ay)); dsk_fold(hi.z, lo.z, vsum(az));
            if (POT) dsk_fold(hi.w, lo.w, -vsum(pot));
        }
        __syncwarp();
    }
    task_store(t, hi, lo, reinterpret_cast<double *>(tile), sacc, sacc_lo);
}

template <int P>
static int launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot)
{
    using C = m2p_cfg<P>;
    static bool attr_done = false;
    const size_t smem = FW * C::WARP_BYTES;
    if (!attr_done) {
        DSK_CUDA(cudaFuncSetAttribute(k_m2p<P, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        DSK_CUDA(cudaFuncSetAttribute(k_m2p<P, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done = true;
    }
    const float e2 = c->eps * c->eps;
    const unsigned grid = (t1 - t0 + FW - 1) / FW;
    if (want_pot)
        k_m2p<P, true><<<grid, FW * 32, smem, c->stream>>>(t0, t1, c->g_task, c->periodic, c->box, e2, c->frows, c->spos, c->gfirst,
                                                           c->gcount, c->gcell, c->list_m2p, c->g_m2p_off, base,
                                                           c->g_m2p_len, c->sacc, c->sacc_lo);
    else
        k_m2p<P, false><<<grid, FW * 32, smem, c->stream>>>(t0, t1, c->g_task, c->periodic, c->box, e2, c->frows, c->spos, c->gfirst,
                                                            c->gcount, c->gcell, c->list_m2p, c->g_m2p_off, base,
                                                            c->g_m2p_len, c->sacc, c->sacc_lo);
    return DSK_OK;
}

int dsk_launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot)
{
    if (t1 <= t0) return DSK_OK;
    switch (c->p) {
    case 2: return launch_m2p<2>(c, t0, t1, base, want_pot);
    case 4: return launch_m2p<4>(c, t0, t1, base, want_pot);
    case 6: return launch_m2p<6>(c, t0, t1, base, want_pot);
    case 8: return launch_m2p<8>(c, t0, t1, base, want_pot);
    default: return DSK_EINVAL;
    }
}
