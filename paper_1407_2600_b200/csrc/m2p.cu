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
// in cell-scaled coordinates rho = r/s, eps~ = eps/s.  This needs well under half the FP32 instructions of the
// derivative recurrence (p = 4: 149 packed instructions = 252 flop per interaction against 636 flop)
// and holds only two degrees of monomials in registers.  The coefficients ("force row") are a fixed linear map of the moment row, applied once per
// cell after the upward pass by k_frows.  The dipole (l = 1) vanishes about the centre of mass and is skipped.
#include "force_task.cuh"
#include <vector>

// ---- force-row layout: header of 8 floats as in the moment row, then blocks (q, m) in q-major order ----
// D: the row carries a dipole block (q = m = 1).  About the centre of mass the particles' dipole vanishes and the block is
// skipped; with background subtraction (reading O4b) the subtracted cube is centred on the cell, not on the centre of mass,
// so the rows of a periodic run with subtraction have it (zero for the plain rows, rho_bar s^3 (com - centre) for the others).
__host__ __device__ constexpr bool fr_has(int P, int q, int m, bool D) { return m >= q && 2 * m - q <= P && (D || !(q == 1 && m == 1)); }
__host__ __device__ constexpr int fr_bsize(int q) { return (q + 1) * (q + 2) / 2; }
__host__ __device__ constexpr int fr_off(int P, int q, int m, bool D)
{
    int o = 0;
    for (int qq = 0; qq <= P; qq++)
        for (int mm = qq; mm <= P; mm++) {
            if (qq == q && mm == m) return o;
            if (qq > q) return o;
            if (fr_has(P, qq, mm, D)) o += fr_bsize(qq);
        }
    return o;
}
__host__ __device__ constexpr int fr_nc(int P, bool D) { return fr_off(P, P + 1, 0, D); }
__host__ __device__ constexpr int fr_rowlen(int P, bool D) { return (8 + fr_nc(P, D) + 3) / 4 * 4; }
__host__ __device__ constexpr int fr_qfirst_S(int P, int m) { return (m == 1 || 2 * m - P < 0) ? 0 : 2 * m - P; }
__host__ __device__ constexpr int fr_qfirst_G(int P, int m) { return 2 * m - P < 1 ? 1 : 2 * m - P; }

static int frow_nc(int p, bool d)
{
    return p == 2 ? fr_nc(2, d) : p == 3 ? fr_nc(3, d) : p == 4 ? fr_nc(4, d) : p == 5 ? fr_nc(5, d) : p == 6 ? fr_nc(6, d) : fr_nc(8, d);
}
int dsk_frow_len(int p, int dip) { return (8 + frow_nc(p, dip != 0) + 3) / 4 * 4; }

// ---- k_frows: moment row -> force row -------------------------------------------------------------------
struct fr_entry { uint32_t src; float w; };

static void build_frow_table(int P, bool D, std::vector<uint32_t> &beg, std::vector<fr_entry> &ent)
{
    double fact[2 * DSK_PMAX + 2];
    fact[0] = 1.0;
    for (int i = 1; i < 2 * DSK_PMAX + 2; i++) fact[i] = fact[i - 1] * i;
    beg.clear(); ent.clear();
    for (int q = 0; q <= P; q++)
        for (int m = q; m <= P; m++) {
            if (!fr_has(P, q, m, D)) continue;
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

// rows [r0, r0 + n) of `rows_in` (moment rows of the current order) -> force rows [f0, f0 + n)
static int run_frows_range(dsk_ctx *c, const float *rows_in, uint32_t n, size_t f0)
{
    const int P = c->p, dip = c->frow_dip, nc = frow_nc(P, dip != 0);
    if (c->frow_tab_p != P || c->frow_tab_dip != dip) {
        std::vector<uint32_t> beg;
        std::vector<fr_entry> ent;
        build_frow_table(P, dip != 0, beg, ent);
        if (beg.size() > DSK_FRTAB_BEG || ent.size() > DSK_FRTAB_ENT) return DSK_EINVAL;
        DSK_CUDA(cudaMemcpyAsync(c->frtab_beg, beg.data(), beg.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
        DSK_CUDA(cudaMemcpyAsync(c->frtab_ent, ent.data(), ent.size() * sizeof(fr_entry), cudaMemcpyHostToDevice, c->stream));
        DSK_CUDA(cudaStreamSynchronize(c->stream));      // the vectors die here
        c->frow_tab_p = P; c->frow_tab_dip = dip;
    }
    if (!n) return DSK_OK;
    const int frl = dsk_frow_len(P, dip);
    k_frows<<<(n + 3) / 4, 128, 0, c->stream>>>(n, dsk_rowlen(P), frl, nc, c->frtab_beg,
                                                (const fr_entry *)c->frtab_ent, rows_in, c->frows + f0 * (size_t)frl);
    DSK_COUNT(c, 1);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

int dsk_run_frows(dsk_ctx *c) { return run_frows_range(c, c->rows, c->hstate->ncell, 0); }
// the background-subtracted copies of the cells of level <= l_b: force rows [ncell, ncell + ntop)   (background.cu)
int dsk_run_frows_bg(dsk_ctx *c, uint32_t ntop) { return run_frows_range(c, c->rows_bg, ntop, c->hstate->ncell); }

// ---- F2 body: the lane's sink(s) against one cell ----------------------------------------------------
// T = f2: two sinks in the halves of every register; T = float: one sink.  The cell's row is read from
// shared memory as scalars (LDS.128 = four coefficients) that enter the packed ops as broadcast operands.
// row (floats): [0..2] -com'/s xyz (com' relative to the sink group's centre), [3] 1/s, [4] eps^2/s^2, [5] -1/s^2,
//               [6] -1/s, [7] 1/s^2, [8+i] B_i
// rho = x/s - com'/s is one FMA per component; both terms are O(d/s) with no cancellation beyond the MAC's
// separation, so this rounds like (x - com')/s.
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

template <int P, typename T, bool POT, bool DIP>
__device__ __forceinline__ void m2p_body(T xs, T ys, T zs, const float *__restrict__ row, T &pot, T &ax, T &ay, T &az)
{
    constexpr int NP = dsk_np(P);
    const float4 hA = *reinterpret_cast<const float4 *>(row), hB = *reinterpret_cast<const float4 *>(row + 4);
    const T sinv = vdup<T>(hA.w);
    T rho[3];
    rho[0] = vfma(xs, sinv, vdup<T>(hA.x)); rho[1] = vfma(ys, sinv, vdup<T>(hA.y));
    rho[2] = vfma(zs, sinv, vdup<T>(hA.z));
    T R2 = vfma(rho[0], rho[0], vdup<T>(hB.x));
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
    const float *Bp = row + 8;
    float4 bq;                         // coefficients arrive four at a time (one LDS.128)
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
            if constexpr (fr_has(P, q, m, DIP)) {
                constexpr int off = fr_off(P, q, m, DIP);
                // A block is homogeneous of degree q, so by Euler's theorem sum_j B_j mu_j = (1/q) rho . grad: from
                // degree 3 on (10 coefficients or more) only the gradient is accumulated (separately) and the value
                // costs 3 FMAs (+ 3 adds to merge the gradient) instead of one FMA per coefficient.
                constexpr bool EUL = (q >= 3);
                T Gt[3];
                static_for<0, fr_bsize(q)>([&](auto JJ) {
                    constexpr int jj = decltype(JJ)::value, ci = off + jj;
                    if constexpr (ci % 4 == 0) bq = *reinterpret_cast<const float4 *>(Bp + ci);
                    const T B = vdup<T>(ci % 4 == 0 ? bq.x : (ci % 4 == 1 ? bq.y : (ci % 4 == 2 ? bq.z : bq.w)));
                    if constexpr (!EUL) {
                        if constexpr (q == 0) S[m] = B;
                        else if constexpr (q == fr_qfirst_S(P, m) && jj == 0) S[m] = vmul(B, mu[base + jj]);
                        else S[m] = vfma(B, mu[base + jj], S[m]);
                    }
                    if constexpr ((m >= 2 || DIP) && q >= 1)
                        static_for<0, 3>([&](auto I) {
                            constexpr int i = decltype(I)::value;
                            constexpr MI ji = dsk_mi(base + jj);
                            if constexpr (mi_comp(ji, i) >= 1) {
                                if constexpr (EUL) {
                                    if constexpr (jj == i) Gt[i] = vmul(B, mu[mi_lower(ji, i)]);
                                    else Gt[i] = vfma(B, mu[mi_lower(ji, i)], Gt[i]);
                                } else {
                                    if constexpr (q == 1) G[m][i] = B;
                                    else if constexpr (q == fr_qfirst_G(P, m) && jj == i) G[m][i] = vmul(B, mu[mi_lower(ji, i)]);
                                    else G[m][i] = vfma(B, mu[mi_lower(ji, i)], G[m][i]);
                                }
                            }
                        });
                });
                if constexpr (EUL) {
                    // the block of highest degree (q = m = P) is all of S_P: it is left as P S_P = rho . grad and the
                    // 1/P goes into the Horner steps below, so rho_i / P is never formed
                    constexpr int qd = (q == P) ? 1 : q;
                    if constexpr (fr_qfirst_S(P, m) == q) S[m] = vmul(rd[0][qd], Gt[0]);
                    else S[m] = vfma(rd[0][qd], Gt[0], S[m]);
                    S[m] = vfma(rd[1][qd], Gt[1], S[m]);
                    S[m] = vfma(rd[2][qd], Gt[2], S[m]);
                    if constexpr (fr_qfirst_G(P, m) == q) { G[m][0] = Gt[0]; G[m][1] = Gt[1]; G[m][2] = Gt[2]; }
                    else { G[m][0] = vadd(G[m][0], Gt[0]); G[m][1] = vadd(G[m][1], Gt[1]); G[m][2] = vadd(G[m][2], Gt[2]); }
                }
            }
        });
    });
    // pot = -(1/s) sum_m h_m S_m ;  acc_i = (1/s^2) [ sum_m h_m G_m,i - rho_i q sum_m (2m+1) h_m S_m ],  h_m = h0 q^m.
    // With Pq(q) = sum_m S_m q^m the last sum is h0 (Pq + 2 q Pq'), so value and derivative come from one Horner pass
    // in q, and sum_m h_m G_m,i = h0 q^2 Horner(G_P,i .. G_2,i): 5P + 9 packed instructions instead of 7P + 7.
    // (for P >= 3, S[P] holds P S_P: its two uses, the first step of each recurrence, multiply by q / P instead of q)
    constexpr bool TOPEUL = P >= 3;
    const T qs = TOPEUL ? vmul(qi, vdup<T>(1.0f / (float)P)) : qi;
    T pq = S[P], dq = S[P];
    static_for<1, P + 1>([&](auto K) {
        constexpr int m = P - decltype(K)::value;                 // P-1 .. 0
        if constexpr (m == P - 2) dq = vfma(dq, qs, pq);
        else if constexpr (m < P - 2) dq = vfma(dq, qi, pq);
        if constexpr (m == P - 1) pq = vfma(pq, qs, S[m]);
        else pq = vfma(pq, qi, S[m]);
    });
    const T tt = vfma(vmul(dq, qi), vdup<T>(2.0f), pq);
    T gh[3] = {G[P][0], G[P][1], G[P][2]};
    static_for<1, (DIP ? P : P - 1)>([&](auto K) {
        constexpr int m = P - decltype(K)::value;                 // P-1 .. 2 (.. 1 with a dipole: G_1 = the dipole itself)
        gh[0] = vfma(gh[0], qi, G[m][0]); gh[1] = vfma(gh[1], qi, G[m][1]); gh[2] = vfma(gh[2], qi, G[m][2]);
    });
    const T u = vmul(vmul(qi, vmul(h0, vdup<T>(hB.y))), tt);       // -h0 q (Pq + 2 q Pq') / s^2
    const T k1 = vmul(qi, vmul(h0, vdup<T>(hB.w)));                // h0 q / s^2
    const T k2 = DIP ? k1 : vmul(k1, qi);                          // h0 q^2 / s^2 when the gradient sums start at m = 2
    ax = vfma(gh[0], k2, ax); ay = vfma(gh[1], k2, ay); az = vfma(gh[2], k2, az);
    ax = vfma(rho[0], u, ax); ay = vfma(rho[1], u, ay); az = vfma(rho[2], u, az);
    if constexpr (POT) pot = vfma(vmul(pq, h0), vdup<T>(hB.z), pot);
}

// ---- F2 kernel ------------------------------------------------------------------------------------------
// Per warp: tiles of up to NCELL listed cells.  The force rows of a tile are brought into shared memory as they
// are, with cp.async (LDGSTS, 16 B): the lane that holds a cell's list entry copies that cell's row, so there is
// no index arithmetic (LPC = 32 / NCELL lanes share a row when rows are long).  (A cp.async.bulk per row was
// tried: UBLKCP takes uniform registers, so 32 different rows become a 32-trip serial loop, 18 % of all
// instructions under ncu.)  The NEXT tile's rows are in flight while the current tile is evaluated and the
// list entries one tile further ahead sit in a register, so no global-memory latency is exposed between tiles.
// When a tile has arrived, one lane per cell rewrites the row's 8-float header in place (centre of mass relative
// to the sink group's cell centre, image shift absorbed exactly, times -1/s; 1/s, eps^2/s^2, -1/s^2, -1/s, 1/s^2) and the sub-groups
// run the body over alternate cells.
// One task (warp) per block: tasks differ in length by more than 10x (list length, sub-group count), and a
// multi-warp block holds its registers and shared memory until its longest warp ends.
#define FW 1
#define M64_MINB 12          // resident warps per SM of the fp64-monopole variants at p <= 4 (164 registers; at 16 they spill: C3 19.05 vs 18.78 ms)
// MODE 0: isolated (fp32, no dipole block); 1: periodic without background subtraction (monopoles in fp64, see the kernel);
// 2: periodic with background subtraction (reading O4b: fp32 throughout, rows carry a dipole block)
template <int P, int MODE> struct m2p_cfg {
    static constexpr bool M64 = MODE == 1, DIP = MODE == 2;
    static constexpr int NCELL = (P <= 4) ? 32 : (P <= 6 ? 16 : 8);   // cells per tile
    static constexpr int LPC = 32 / NCELL;                             // lanes that share the copy of one row
    static constexpr int FROW = fr_rowlen(P, DIP);
    static constexpr int NCH = FROW / 4;                               // 16-byte chunks per row
    static constexpr size_t BUF_BYTES = (size_t)NCELL * FROW * sizeof(float);
    static constexpr size_t M64_BYTES = M64 ? (size_t)NCELL * 4 * sizeof(double) : 0;   // com' xyz and mass of a tile's cells
    static constexpr size_t WARP_BYTES = 2 * BUF_BYTES + M64_BYTES;    // two row buffers + fp64 monopoles
};

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int P, bool POT, int MODE>
__global__ void __launch_bounds__(FW * 32, (P <= 4 ? (MODE == 1 ? M64_MINB : 16) : 1)) k_m2p(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap, int periodic,
                                                 float box, float eps2, const float *__restrict__ frows,
                                                 const float4 *__restrict__ spos, const uint32_t *__restrict__ gfirst,
                                                 const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ gcell,
                                                 const uint32_t *__restrict__ list, const uint64_t *__restrict__ off,
                                                 uint64_t base, const uint32_t *__restrict__ len,
                                                 float4 *__restrict__ sacc, float4 *__restrict__ sacc_lo)
{
    using C = m2p_cfg<P, MODE>;
    constexpr bool M64 = C::M64, DIP = C::DIP;
    constexpr int NCELL = C::NCELL, LPC = C::LPC, FROW = C::FROW, NCH = C::NCH;
    constexpr uint32_t CELL_MASK = (1u << DSK_CELL_BITS) - 1u;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const warp_task t = make_task(t0, t1, FW, taskmap, gfirst, gcount);
    if (!t.valid) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *wbase = smem_raw + (size_t)warp * C::WARP_BYTES;
    double *mono = reinterpret_cast<double *>(wbase + 2 * C::BUF_BYTES);   // [NCELL][4], M64 only
    const float *grow = frows + (size_t)gcell[t.g] * FROW;
    const float cgx = grow[0], cgy = grow[1], cgz = grow[2];
    const float4 ma = spos[t.sa], mb = spos[t.sb];
    const uint32_t n = len[t.g];
    const uint32_t *lst = list + (off[t.g] - base);
    // running sums as two-float (hi, lo) pairs, continued from the P2P kernel (sub-group 0 carries them);
    // each tile is summed from zero in plain fp32 and folded in with TwoSum, so no addition ever rounds at
    // the size of the total
    sink_acc A;
    acc_load(A, t, sacc, sacc_lo);
    const f2 X = f2_make(ma.x - cgx, mb.x - cgx), Y = f2_make(ma.y - cgy, mb.y - cgy), Z = f2_make(ma.z - cgz, mb.z - cgz);
    // cells per tile: a multiple of the number of sub-groups, so that they finish together
    const uint32_t tc = (uint32_t)(t.S >= NCELL ? NCELL : (NCELL / t.S) * t.S);
    const int mycell = lane / LPC, mypart = lane - mycell * LPC;     // the row (and share of it) this lane copies

    // issue the copies of one tile: entry e = list entry of cell `mycell` of the tile
    auto fetch = [&](uint32_t e, int ncell, int b) {
        if (mycell < ncell) {
            const float4 *src = reinterpret_cast<const float4 *>(frows + (size_t)(e & CELL_MASK) * FROW);
            float4 *dst = reinterpret_cast<float4 *>(wbase + (size_t)b * C::BUF_BYTES) + (size_t)mycell * NCH;
#pragma unroll
            for (int ch = mypart; ch < NCH; ch += LPC) cp_async16(dst + ch, src + ch);
        }
        cp_async_commit();
    };
    uint32_t e_cur = (mycell < (int)tc && (uint32_t)mycell < n) ? lst[mycell] : 0u;
    fetch(e_cur, (int)min(tc, n), 0);
    uint32_t e_nxt = (mycell < (int)tc && tc + mycell < n) ? lst[tc + mycell] : 0u;

    uint32_t it = 0;
    for (uint32_t b0 = 0; b0 < n; b0 += tc, it++) {
        const int ntc = (int)min(tc, n - b0);
        const int b = (int)(it & 1u);
        float *rows = reinterpret_cast<float *>(wbase + (size_t)b * C::BUF_BYTES);
        cp_async_wait_all();
        __syncwarp();
        // ---- header in place ----
        if (mycell < ntc && mypart == 0) {
            float *r = rows + (size_t)mycell * FROW;
            const float4 h0 = *reinterpret_cast<const float4 *>(r);
            const float4 h1 = *reinterpret_cast<const float4 *>(r + 4);
            float shx = 0.0f, shy = 0.0f, shz = 0.0f;
            if (periodic) {
                const int img = (int)(e_cur >> DSK_CELL_BITS), side = 2 * DSK_WS + 1;
                shz = (float)(img % side - DSK_WS) * box;
                shy = (float)((img / side) % side - DSK_WS) * box;
                shx = (float)(img / (side * side) - DSK_WS) * box;
            }
            const float sinv = h0.w;
            const float nsinv = -sinv, sinv2 = sinv * sinv;
            *reinterpret_cast<float4 *>(r) = make_float4((((h0.x - cgx) + shx) + h1.x) * nsinv, (((h0.y - cgy) + shy) + h1.y) * nsinv,
                                                         (((h0.z - cgz) + shz) + h1.z) * nsinv, sinv);
            *reinterpret_cast<float4 *>(r + 4) = make_float4(eps2 * sinv2, -sinv2, nsinv, sinv2);
            if constexpr (M64) {
                // the monopole of this cell is evaluated in fp64 below: centre of mass in double (the two
                // differences are exact), mass out of the fp32 row
                double *m4 = mono + 4 * mycell;
                m4[0] = ((double)(h0.x - cgx) + (double)shx) + (double)h1.x;
                m4[1] = ((double)(h0.y - cgy) + (double)shy) + (double)h1.y;
                m4[2] = ((double)(h0.z - cgz) + (double)shz) + (double)h1.z;
                m4[3] = (double)r[8];
                r[8] = 0.0f;
            }
        }
        __syncwarp();
        // ---- next tile on its way while this one is evaluated ----
        e_cur = e_nxt;
        if (b0 + tc < n) {
            fetch(e_cur, (int)min(tc, n - b0 - tc), b ^ 1);
            const uint32_t b2 = b0 + 2u * tc;
            e_nxt = (mycell < (int)tc && b2 + mycell < n) ? lst[b2 + mycell] : 0u;
        }
        if (t.active) {
            f2 pot = f2_dup(0.0f), ax = f2_dup(0.0f), ay = f2_dup(0.0f), az = f2_dup(0.0f);
            if constexpr (M64) {
                // Monopoles in fp64.  In a periodic, nearly uniform box the image block's monopole terms are
                // O(M/L^2) each and cancel to a net force hundreds of times smaller, so their fp32 rounding
                // (1e-7 of each term) alone exceeds the 1e-4 per-particle gate (measured on C3: p99.9 = 6e-4).
                // The fp64 monopole of a cell rides in the same loop trip as its fp32 body: the chain difference ->
                // r2 -> MUFU seed (1e-7) -> one Newton step (1.5e-14) -> products is ~150 cycles long and hides under the
                // ~150 independent packed fp32 instructions of the same warp (other pipes).  As a pass of its own,
                // one chain at a time: C3 19.9 ms, C4 641; four chains: 19.2, 602; in the body's loop: 18.8, 596.
                const double e2d = (double)eps2;
                const double xs0 = (double)ma.x - (double)cgx, ys0 = (double)ma.y - (double)cgy, zs0 = (double)ma.z - (double)cgz;
                const double xs1 = (double)mb.x - (double)cgx, ys1 = (double)mb.y - (double)cgy, zs1 = (double)mb.z - (double)cgz;
                double s0[4] = {0.0, 0.0, 0.0, 0.0}, s1[4] = {0.0, 0.0, 0.0, 0.0};
                auto mono1 = [&](const double2 c01, const double2 c23, double xs, double ys, double zs, double *sm) {
                    const double dx = c01.x - xs, dy = c01.y - ys, dz = c23.x - zs;
                    const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, e2d)));
                    const double y0 = (double)rsqrtf((float)r2);
                    const double ri = y0 * fma(-0.5 * r2, y0 * y0, 1.5);
                    const double mri = c23.y * ri, mri3 = mri * ri * ri;
                    sm[0] = fma(dx, mri3, sm[0]); sm[1] = fma(dy, mri3, sm[1]); sm[2] = fma(dz, mri3, sm[2]);
                    if (POT) sm[3] -= mri;
                };
                for (int k = t.sub; k < ntc; k += t.S) {
                    const double2 c01 = *reinterpret_cast<const double2 *>(mono + 4 * k);
                    const double2 c23 = *reinterpret_cast<const double2 *>(mono + 4 * k + 2);
                    mono1(c01, c23, xs0, ys0, zs0, s0);
                    mono1(c01, c23, xs1, ys1, zs1, s1);
                    m2p_body<P, f2, POT, DIP>(X, Y, Z, rows + (size_t)k * FROW, pot, ax, ay, az);
                }
                acc_add_double(A, 0, 0, s0[0]); acc_add_double(A, 0, 1, s0[1]); acc_add_double(A, 0, 2, s0[2]);
                acc_add_double(A, 1, 0, s1[0]); acc_add_double(A, 1, 1, s1[1]); acc_add_double(A, 1, 2, s1[2]);
                if (POT) { acc_add_double(A, 0, 3, s0[3]); acc_add_double(A, 1, 3, s1[3]); }
            } else {
                for (int k = t.sub; k < ntc; k += t.S) m2p_body<P, f2, POT, DIP>(X, Y, Z, rows + (size_t)k * FROW, pot, ax, ay, az);
            }
            acc_fold(A, ax, ay, az, pot, POT);
        }
        __syncwarp();
    }
    task_store(t, A, reinterpret_cast<double *>(wbase), sacc, sacc_lo);
}

// ---- longest task first ----------------------------------------------------------------------------------
// Task lengths differ by more than 10x (list length / sub-groups) and the longest run for milliseconds, so in
// list order the kernel ends with a few SMs busy (ncu: SMs active 90 % of the elapsed cycles, 10.6 of 16 warp
// slots occupied on average).  A one-pass counting sort by descending cost fixes the order; within a bin the
// order is arbitrary, which cannot change any result (a task owns its sinks).
#define TASK_BINS 1024
__device__ __forceinline__ uint32_t task_cost_bin(uint32_t m, const uint32_t *__restrict__ gcount,
                                                  const uint32_t *__restrict__ len, int shift)
{
    const uint32_t g = m >> 2;
    uint32_t soff, ns;
    dsk_task_range(gcount[g], m & 3u, soff, ns);
    const uint32_t w = (ns + 1) >> 1, S = 32u / w;
    const uint32_t cost = (len[g] + S - 1) / S;                      // body executions per lane
    return TASK_BINS - 1u - min((uint32_t)TASK_BINS - 1u, cost >> shift);
}
__global__ void __launch_bounds__(256) k_task_hist(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap,
                                                   const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ len,
                                                   int shift, uint32_t *__restrict__ hist)
{
    const uint32_t t = t0 + blockIdx.x * 256 + threadIdx.x;
    // neighbouring tasks cost about the same: one atomic per distinct bin and warp, not per task
    const uint32_t bin = t < t1 ? task_cost_bin(taskmap[t], gcount, len, shift) : 0xffffffffu;
    const uint32_t peers = __match_any_sync(0xffffffffu, bin), lane = threadIdx.x & 31u;
    if (t < t1 && (peers & ((1u << lane) - 1u)) == 0u) atomicAdd(&hist[bin], (uint32_t)__popc(peers));
}
__global__ void __launch_bounds__(TASK_BINS) k_task_scan(uint32_t *__restrict__ hist)
{
    __shared__ uint32_t s[TASK_BINS];
    const int i = threadIdx.x;
    const uint32_t v = hist[i];
    s[i] = v;
    __syncthreads();
    for (int o = 1; o < TASK_BINS; o <<= 1) {
        const uint32_t y = i >= o ? s[i - o] : 0u;
        __syncthreads();
        s[i] += y;
        __syncthreads();
    }
    hist[i] = s[i] - v;
}
__global__ void __launch_bounds__(256) k_task_scatter(uint32_t t0, uint32_t t1, const uint32_t *__restrict__ taskmap,
                                                      const uint32_t *__restrict__ gcount, const uint32_t *__restrict__ len,
                                                      int shift, uint32_t *__restrict__ hist, uint32_t *__restrict__ sorted)
{
    const uint32_t t = t0 + blockIdx.x * 256 + threadIdx.x;
    const uint32_t m = t < t1 ? taskmap[t] : 0u;
    const uint32_t bin = t < t1 ? task_cost_bin(m, gcount, len, shift) : 0xffffffffu;
    const uint32_t peers = __match_any_sync(0xffffffffu, bin), lane = threadIdx.x & 31u;
    const uint32_t before = __popc(peers & ((1u << lane) - 1u));
    uint32_t at = 0;
    if (t < t1 && before == 0u) at = atomicAdd(&hist[bin], (uint32_t)__popc(peers));      // the first lane of each bin reserves for all
    at = __shfl_sync(0xffffffffu, at, __ffs((int)peers) - 1);
    if (t < t1) sorted[t0 + at + before] = m;
}

// g_task_sorted[t0, t1) = the tasks of g_task[t0, t1) by descending (len[group] >> shift) / sub-groups
int dsk_order_tasks(dsk_ctx *c, uint32_t t0, uint32_t t1, const uint32_t *len, int shift)
{
#ifdef DSK_NO_TASK_ORDER        // tuning experiments only: list (Morton) order
    DSK_CUDA(cudaMemcpyAsync(c->g_task_sorted + t0, c->g_task + t0, sizeof(uint32_t) * (size_t)(t1 - t0), cudaMemcpyDeviceToDevice, c->stream));
    return DSK_OK;
#endif
    const unsigned nb = (t1 - t0 + 255) / 256;
    DSK_CUDA(cudaMemsetAsync(c->task_hist, 0, sizeof(uint32_t) * TASK_BINS, c->stream));
    k_task_hist<<<nb, 256, 0, c->stream>>>(t0, t1, c->g_task, c->gcount, len, shift, c->task_hist);
    k_task_scan<<<1, TASK_BINS, 0, c->stream>>>(c->task_hist);
    k_task_scatter<<<nb, 256, 0, c->stream>>>(t0, t1, c->g_task, c->gcount, len, shift, c->task_hist, c->g_task_sorted);
    DSK_COUNT(c, 3);
    return cudaGetLastError() == cudaSuccess ? DSK_OK : DSK_ECUDA;
}

template <int P, bool POT, int MODE>
static int launch_m2p_v(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base)
{
    using C = m2p_cfg<P, MODE>;
    static bool attr_flags[DSK_MAXDEV];
    bool *attr_done = dsk_device_flag(attr_flags);
    const size_t smem = FW * C::WARP_BYTES;
    if (!*attr_done) {
        DSK_CUDA(cudaFuncSetAttribute(k_m2p<P, POT, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        DSK_CUDA(cudaFuncSetAttribute(k_m2p<P, POT, MODE>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        *attr_done = true;
    }
    const float e2 = c->soft_kind == 1 ? 0.0f : c->eps * c->eps;      // K1 (O6b): the accepted cells lie beyond the kernel's support, Newtonian expansion
    const unsigned grid = (t1 - t0 + FW - 1) / FW;
    k_m2p<P, POT, MODE><<<grid, FW * 32, smem, c->stream>>>(t0, t1, c->g_task_sorted, c->periodic, c->box, e2, c->frows, c->spos,
                                                            c->gfirst, c->gcount, c->gcell, c->list_m2p, c->g_m2p_off, base,
                                                            c->g_m2p_len, c->sacc, c->sacc_lo);
    return DSK_OK;
}

template <int P>
static int launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot)
{
    int e = dsk_order_tasks(c, t0, t1, c->g_m2p_len, 3);
    if (e) return e;
    // the rows' layout (dipole block or not) was fixed when they were made: the kernel must match it
    if (c->frow_dip) return want_pot ? launch_m2p_v<P, true, 2>(c, t0, t1, base) : launch_m2p_v<P, false, 2>(c, t0, t1, base);
    // periodic without background subtraction: monopoles in fp64 (see the kernel)
    if (c->periodic) return want_pot ? launch_m2p_v<P, true, 1>(c, t0, t1, base) : launch_m2p_v<P, false, 1>(c, t0, t1, base);
    return want_pot ? launch_m2p_v<P, true, 0>(c, t0, t1, base) : launch_m2p_v<P, false, 0>(c, t0, t1, base);
}

int dsk_launch_m2p(dsk_ctx *c, uint32_t t0, uint32_t t1, uint64_t base, int want_pot)
{
    if (t1 <= t0) return DSK_OK;
    switch (c->p) {
    case 2: return launch_m2p<2>(c, t0, t1, base, want_pot);
    case 3: return launch_m2p<3>(c, t0, t1, base, want_pot);
    case 4: return launch_m2p<4>(c, t0, t1, base, want_pot);
    case 5: return launch_m2p<5>(c, t0, t1, base, want_pot);
    case 6: return launch_m2p<6>(c, t0, t1, base, want_pot);
    case 8: return launch_m2p<8>(c, t0, t1, base, want_pot);
    default: return DSK_EINVAL;
    }
}
