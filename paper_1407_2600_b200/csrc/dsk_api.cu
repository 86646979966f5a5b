// dsk_api.cu — the C ABI of include/dsk.h: context, workspace carving, orchestration of the phases
// K S T G U W F1 F2 F3 X I on the caller's stream, status read-back.  No device allocation after
// dsk_bind_workspace; one small D2H read + stream synchronise at the end of each compute call.
#include "dsk_internal.cuh"
#include <math.h>
#include <new>
#include <string.h>

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// carve (or just measure, when base == nullptr) the workspace
static size_t carve(dsk_ctx *c, char *base)
{
    size_t o = 0;
    const size_t n = (size_t)c->N;
    auto take = [&](size_t bytes) -> char * {
        char *p = base ? base + o : nullptr;
        o += align_up(bytes);
        return p;
    };
    c->ntile = (int)((n + DSK_SORT_TILE - 1) / DSK_SORT_TILE);
    // measured <= 0.06 cells and <= 0.05 groups per particle (NLEAF 64-112, NCRIT 64-192) on every config; a pathological
    // input (deep chains of near-coincident clumps) that needs more ends in DSK_ECELLOVERFLOW, not in a fault
    c->ncell_cap = (int64_t)(n / 4 + 4096);
    if (c->ncell_cap > (1ll << DSK_CELL_BITS)) c->ncell_cap = 1ll << DSK_CELL_BITS;
    c->ngroup_cap = (int64_t)(n / 4 + 1024);
    const size_t nc = (size_t)c->ncell_cap, ng = (size_t)c->ngroup_cap;
    c->dstate = (dsk_devstate *)take(sizeof(dsk_devstate));
    c->key_a = (uint64_t *)take(8 * n);
    c->key_b = (uint64_t *)take(8 * n);
    c->idx_a = (uint32_t *)take(4 * n);
    c->idx_b = (uint32_t *)take(4 * n);
    c->sort_hist = (uint32_t *)take(4 * (n <= (size_t)DSK_SORT_ONESWEEP_NMAX ? 8 * 256 + 64 + (size_t)8 * 256 * c->ntile : 256 * (size_t)c->ntile));
    c->scan_tmp = (uint32_t *)take(4 * 4096);
    c->spos = (float4 *)take(16 * n);
    c->sacc = (float4 *)take(16 * n);
    c->sacc_lo = (float4 *)take(16 * n);
    c->hotkey = (uint64_t *)take(8 * nc);
    c->cell = (dsk_cellrec *)take(16 * nc);
    c->parent = (uint32_t *)take(4 * nc);
    c->nchild_tmp = (uint32_t *)take(4 * nc);
    c->cbounds = (uint32_t *)take(32 * nc);
    c->whdr = (float4 *)take(16 * nc);
    c->wmac = (float4 *)take(32 * nc);     // MAC record + cell record per cell
    c->rows = (float *)take(4 * (size_t)dsk_rowlen(c->p_cap) * nc);
    // background subtraction (periodic): cells of level <= l_b have a second, subtracted force row behind the ncell plain ones
    c->bg_level = dsk_bg_level(c->N);
    c->ntop_cap = 0;
    if (c->periodic) {
        int64_t full = 0;
        for (int l = 0; l <= c->bg_level; l++) full += (int64_t)1 << (3 * l);
        c->ntop_cap = full < c->ncell_cap ? full : c->ncell_cap;
    }
    const size_t nt = (size_t)c->ntop_cap;
    c->frows = (float *)take(4 * (size_t)dsk_frow_len(c->p_cap, c->periodic) * (nc + nt));
    c->topgeo = (int4 *)take(16 * nt);
    c->mass64 = (double *)take(8 * nt);
    c->kbg = (float *)take(4 * nt);
    c->rows_bg = (float *)take(4 * (size_t)dsk_rowlen(c->p_cap) * nt);
    c->g_left_len = (uint32_t *)take(4 * (c->periodic ? ng : 0));
    c->g_left_off = (uint64_t *)take(8 * (c->periodic ? ng + 1 : 0));
    // third list: cubes kept outside the windows.  Usually < 1 per group, a few for groups next to a halo: N/2 records
    // give the one-pass walk ~20 per group (a group that needs more sends the evaluation to the two-pass form)
    c->list_left_cap = c->periodic ? n / 2 + (1u << 16) : 0;
    c->list_left = (uint4 *)take(16 * c->list_left_cap);
    c->pg_key = (uint64_t *)take(8 * ng);
    c->pg_m2p = (uint32_t *)take(4 * ng);
    c->pg_p2p = (uint32_t *)take(4 * ng);
    c->pg_left = (uint32_t *)take(4 * ng);
    c->frtab_beg = (uint32_t *)take(4 * DSK_FRTAB_BEG);
    c->frtab_ent = (void *)take(8 * DSK_FRTAB_ENT);
    c->gmark = (uint32_t *)take(4 * n);
    c->gscan = (uint32_t *)take(4 * n);
    c->gfirst = (uint32_t *)take(4 * ng);
    c->gcount = (uint32_t *)take(4 * ng);
    c->gcell = (uint32_t *)take(4 * ng);
    c->gbox = (float4 *)take(32 * ng);
    c->g_m2p_len = (uint32_t *)take(4 * ng);
    c->g_p2p_len = (uint32_t *)take(4 * ng);
    c->g_p2p_src = (uint32_t *)take(4 * ng);
    c->g_taskoff = (uint32_t *)take(4 * (ng + 1));
    c->gact = (uint8_t *)take(ng);
    c->g_task = (uint32_t *)take(16 * ng);
    c->g_task_sorted = (uint32_t *)take(16 * ng);
    c->task_hist = (uint32_t *)take(4 * 1024);
    c->g_m2p_off = (uint64_t *)take(8 * (ng + 1));
    c->g_p2p_off = (uint64_t *)take(8 * (ng + 1));
    // interaction lists: 256 / 32 entries per particle cover theta >= 0.3 in one batch on the paper-like
    // workloads; anything longer (or very large N) runs in batches of groups (force.cu)
    c->list_m2p_cap = n * 256 + (1u << 20);
    c->list_p2p_cap = n * 32 + (1u << 18);
    const size_t cap_entries = (size_t)3 << 30;                    // 12 GiB of u32 per list at most
    if (c->list_m2p_cap > cap_entries) c->list_m2p_cap = cap_entries;
    if (c->list_p2p_cap > cap_entries / 4) c->list_p2p_cap = cap_entries / 4;
    c->list_m2p = (uint32_t *)take(4 * c->list_m2p_cap);
    c->list_p2p = (uint32_t *)take(4 * c->list_p2p_cap);
    c->kdk_acc = (float *)take(12 * n);
    c->kdk_active = (uint8_t *)take(n);
    c->far_partial = (double *)take(8 * DSK_NFAR * 1024);
    c->far_M = (double *)take(8 * DSK_NFAR);
    c->far_T_dev = (double *)take(8 * DSK_NFAR);
    c->far_lambda = (double *)take(8 * DSK_NFAR);
    return o;
}

static int check_params(float eps, float theta, int p)
{
    if (!(eps > 0.0f) || !isfinite(eps)) return DSK_EINVAL;
    if (!(theta > 0.0f && theta <= 1.0f)) return DSK_EINVAL;
    if (p != 2 && p != 3 && p != 4 && p != 5 && p != 6 && p != 8) return DSK_EINVAL;
    return DSK_OK;
}

extern "C" int dsk_create(dsk_ctx **out, int64_t N, float box, int periodic, float eps, float theta, int p)
{
    if (!out) return DSK_EINVAL;
    *out = nullptr;
    if (N <= 0 || N > 0xfffffff0ll || !(box > 0.0f) || !isfinite(box)) return DSK_EINVAL;
    if (check_params(eps, theta, p)) return DSK_EINVAL;
    dsk_ctx *c = new (std::nothrow) dsk_ctx;
    if (!c) return DSK_ECUDA;
    memset(c, 0, sizeof(*c));
    c->N = N; c->box = box; c->periodic = periodic ? 1 : 0; c->eps = eps; c->theta = theta; c->p = p;
    c->moments_p = -1; c->p_cap = p; c->frow_tab_p = -1; c->frow_tab_dip = -1;
    c->bg = c->periodic;                         // background subtraction is the default in periodic boxes (dsk_set_background)
    c->omega_m = 1.0; c->omega_l = 0.0;
    c->onepass_bad_theta = -1.0f;
    c->ws_bytes = 0;
    carve(c, nullptr);
    c->img_ws = DSK_WS_DEFAULT;
    if (c->periodic) dsk_lattice_tensors((double)box, c->img_ws, c->far_T);
    c->stats.n = N;
    *out = c;
    return DSK_OK;
}

extern "C" int dsk_destroy(dsk_ctx *c)
{
    if (!c) return DSK_EINVAL;
    if (c->hstate) {
        cudaFreeHost(c->hstate);
        for (int i = 0; i < 20; i++) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    }
    delete c;
    return DSK_OK;
}

extern "C" size_t dsk_workspace_bytes(const dsk_ctx *c)
{
    if (!c) return 0;
    dsk_ctx tmp = *c;
    return carve(&tmp, nullptr);
}

extern "C" int dsk_bind_workspace(dsk_ctx *c, void *dev_ptr, size_t bytes)
{
    if (!c) return DSK_EINVAL;
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255)) return DSK_ENOWORKSPACE;
    if (bytes < dsk_workspace_bytes(c)) return DSK_ENOWORKSPACE;
    int dev = 0;
    DSK_CUDA(cudaGetDevice(&dev));
    DSK_CUDA(cudaDeviceGetAttribute(&c->nsm, cudaDevAttrMultiProcessorCount, dev));
    if (!c->hstate) {
        DSK_CUDA(cudaMallocHost((void **)&c->hstate, 4096));
        memset(c->hstate, 0, 4096);
        for (int i = 0; i < 20; i++) DSK_CUDA(cudaEventCreate(&c->ev[i]));
    }
    c->ws = (char *)dev_ptr;
    c->ws_bytes = bytes;
    carve(c, c->ws);
    c->have_tree = 0; c->moments_p = -1; c->lists_valid = 0; c->pg_valid = 0; c->kdk_have_acc = 0; c->frow_tab_p = -1; c->frow_tab_dip = -1;
    if (c->periodic)
        DSK_CUDA(cudaMemcpyAsync(c->far_T_dev, c->far_T, sizeof(double) * DSK_NFAR, cudaMemcpyHostToDevice, c->stream));
    DSK_CUDA(cudaMemsetAsync(c->dstate, 0, sizeof(dsk_devstate), c->stream));
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return DSK_OK;
}

extern "C" int dsk_set_stream(dsk_ctx *c, void *stream)
{
    if (!c) return DSK_EINVAL;
    c->stream = (cudaStream_t)stream;
    return DSK_OK;
}

extern "C" int dsk_set_params(dsk_ctx *c, float eps, float theta, int p)
{
    if (!c) return DSK_EINVAL;
    if (check_params(eps, theta, p)) return DSK_EINVAL;
    if (p > c->p_cap) return DSK_ENOWORKSPACE;        // rows were sized for dsk_create's p
    if (eps != c->eps || theta != c->theta || p != c->p) c->pg_valid = 0;      // other lists: no prediction from the old ones (walk.cu)
    c->eps = eps; c->theta = theta; c->p = p;
    return DSK_OK;
}

static int status_to_error(uint32_t st)
{
    if (st & ST_NONFINITE) return DSK_ENONFINITE;
    if (st & ST_OUTOFBOX) return DSK_EOUTOFBOX;
    if (st & ST_CELLOVF) return DSK_ECELLOVERFLOW;
    if (st & (ST_STACKOVF | ST_LISTOVF)) return DSK_ELISTOVERFLOW;
    return DSK_OK;
}

static int read_state(dsk_ctx *c)
{
    DSK_CUDA(cudaMemcpyAsync(c->hstate, c->dstate, sizeof(dsk_devstate), cudaMemcpyDeviceToHost, c->stream));
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    DSK_CUDA(cudaGetLastError());
    return status_to_error(c->hstate->status);
}

static float ev_ms(cudaEvent_t a, cudaEvent_t b)
{
    float ms = 0.0f;
    if (cudaEventElapsedTime(&ms, a, b) != cudaSuccess) { cudaGetLastError(); return 0.0f; }
    return ms;
}

extern "C" int dsk_build_tree(dsk_ctx *c, const float *pos, const float *mass)
{
    if (!c || !pos || !mass) return DSK_EINVAL;
    if (!c->ws) return DSK_ENOWORKSPACE;
    c->have_tree = 0; c->moments_p = -1; c->lists_valid = 0;
    c->onepass_bad_theta = -1.0f;          // a new tree gets a new one-pass attempt (an old overflow says nothing about it)
    c->stats.n_launch = 0;
    DSK_CUDA(cudaMemsetAsync(c->dstate, 0, sizeof(dsk_devstate), c->stream));
    int e = dsk_run_keysort(c, pos, mass);
    if (e) return e;
    e = dsk_run_build(c);
    if (e) return e;
    e = read_state(c);                       // ncell, ngroup, level starts, status
    if (e) return e;
    c->stats.ncell = c->hstate->ncell; c->stats.ngroup = c->hstate->ngroup;
    c->stats.nlevel = c->hstate->nlevel; c->stats.nleaf_cells = c->hstate->nleaf_cells;
    c->have_tree = 1;
    e = dsk_run_upward(c);
    if (e) return e;
    c->pending_build_ms = 3;                 // phase times are read at the next synchronisation anyway due (end of dsk_accel, dsk_get_stats)
    return DSK_OK;
}

// the stream is synchronised: read the event times that earlier calls left pending
static void finish_ms(dsk_ctx *c)
{
    if (c->pending_build_ms & 1) {
        c->stats.ms_key = ev_ms(c->ev[0], c->ev[1]);
        c->stats.ms_sort = ev_ms(c->ev[1], c->ev[2]);
        c->stats.ms_build = ev_ms(c->ev[2], c->ev[3]);
        c->stats.ms_group = ev_ms(c->ev[3], c->ev[4]);
    }
    if (c->pending_build_ms & 2) c->stats.ms_upward = ev_ms(c->ev[5], c->ev[6]);
    if (c->pending_force_ms) {
        if (c->pending_force_ms == 2) c->stats.ms_walk = ev_ms(c->ev[7], c->ev[8]);
        c->stats.ms_p2p = ev_ms(c->ev[8], c->ev[9]);
        c->stats.ms_m2p = ev_ms(c->ev[9], c->ev[10]);
    }
    c->pending_build_ms = c->pending_force_ms = 0;
}

// shard_rank >= 0: evaluate only the contiguous run of sink groups that the work-weighted cut gives this rank (dsk_accel_shard)
static int accel_impl(dsk_ctx *c, const uint8_t *active, float *acc, float *pot, int shard_rank = -1, int shard_n = 1,
                      int64_t *shard_lo = nullptr, int64_t *shard_hi = nullptr)
{
    if (!c || !acc) return DSK_EINVAL;
    if (!c->ws) return DSK_ENOWORKSPACE;
    if (!c->have_tree) return DSK_ENOTREE;
    int e;
    uint32_t r_lo = 0, r_hi = 0xffffffffu;
    if (c->moments_p != c->p) {
        e = dsk_run_upward(c);
        if (e) return e;
        c->pending_build_ms |= 2;
    }
    c->gact_cur = nullptr;
    if (active) {                                   // lists of an active subset are never reused
        e = dsk_run_group_active(c, active);
        if (e) return e;
        c->gact_cur = c->gact;
        c->lists_valid = 0;
    }
    if (shard_rank >= 0) {
        static const uint32_t fm[7] = {78, 136, 252, 423, 682, 1040, 1536};         // flop per M2P interaction at p = 2 .. 8 (accounting.py)
        uint32_t cut[1025];
        e = dsk_run_shard(c, shard_rank, shard_n, fm[c->p - 2], 19u, cut);
        if (e) return e;
        const uint32_t g_lo = cut[shard_rank], g_hi = cut[shard_rank + 1], ng = c->hstate->ngroup;
        if (shard_lo) *shard_lo = g_lo;
        if (shard_hi) *shard_hi = g_hi;
        // the shard's sorted ranks [first rank of g_lo, first rank of g_hi)
        uint32_t ends[2] = {0, (uint32_t)c->N};
        if (g_lo < ng) DSK_CUDA(cudaMemcpyAsync(&ends[0], c->gfirst + g_lo, 4, cudaMemcpyDeviceToHost, c->stream));
        else ends[0] = (uint32_t)c->N;
        if (g_hi < ng) DSK_CUDA(cudaMemcpyAsync(&ends[1], c->gfirst + g_hi, 4, cudaMemcpyDeviceToHost, c->stream));
        DSK_CUDA(cudaStreamSynchronize(c->stream));
        r_lo = ends[0]; r_hi = ends[1];
        c->gact_cur = c->gact;
        c->lists_valid = 0;
    }
    if (!(c->lists_valid && c->lists_theta == c->theta)) {
        e = dsk_run_walk(c);
        if (e) { c->gact_cur = nullptr; return e; }
    }
    e = dsk_run_force(c, pot != nullptr);
    if (e == DSK_RETRY_WALK) {                       // a list outgrew the slot predicted from the previous evaluation: COUNT + FILL after all
        c->pg_valid = 0; c->lists_valid = 0;        // (P2P stores, M2P adds to it: starting over needs no clearing)
        c->pg_retries++;
        c->pg_backoff = c->pg_backoff >= 7 ? 15 : 2 * c->pg_backoff + 1;      // a tree that changes this fast: predict less often
        c->pg_wait = c->pg_backoff;
        e = dsk_run_walk(c);
        if (e) { c->gact_cur = nullptr; return e; }
        e = dsk_run_force(c, pot != nullptr);
    }
    c->gact_cur = nullptr;
    if (active || shard_rank >= 0) c->lists_valid = 0;
    if (e) return e;
    cudaEventRecord(c->ev[12], c->stream);
    if (c->periodic) {
        e = dsk_run_farfield(c);
        if (e) return e;
        if (c->bg) {                                 // the exact background of the windows (background.cu)
            e = dsk_run_bg_window(c, pot != nullptr);
            if (e) return e;
        }
    }
    cudaEventRecord(c->ev[13], c->stream);
    e = dsk_run_scatter(c, acc, pot, active, r_lo, r_hi);
    if (e) return e;
    cudaEventRecord(c->ev[14], c->stream);
    e = read_state(c);                   // the call's closing synchronisation: every event of this and of the build before it has completed
    finish_ms(c);
    c->stats.ms_far = ev_ms(c->ev[12], c->ev[13]);
    c->stats.ms_scatter = ev_ms(c->ev[13], c->ev[14]);
    c->stats.n_p2p = (int64_t)c->hstate->n_p2p; c->stats.n_m2p = (int64_t)c->hstate->n_m2p;
    c->stats.list_m2p = (int64_t)c->hstate->tot_m2p_list; c->stats.list_p2p = (int64_t)c->hstate->tot_p2p_list;
    c->stats.list_bg = (int64_t)c->hstate->tot_left_list;
    return e;
}

extern "C" int dsk_accel(dsk_ctx *c, const float *pos, const float *mass, float *acc, float *pot)
{
    (void)pos; (void)mass;
    return accel_impl(c, nullptr, acc, pot);
}

extern "C" int dsk_accel_active(dsk_ctx *c, const float *pos, const float *mass, const uint8_t *active, float *acc,
                                float *pot)
{
    (void)pos; (void)mass;
    if (!active) return DSK_EINVAL;
    return accel_impl(c, active, acc, pot);
}

extern "C" int dsk_accel_shard(dsk_ctx *c, int rank, int nranks, float *acc, float *pot, int64_t *first_group, int64_t *end_group)
{
    if (!c || nranks < 1 || nranks > 1023 || rank < 0 || rank >= nranks) return DSK_EINVAL;
    return accel_impl(c, nullptr, acc, pot, rank, nranks, first_group, end_group);
}

// Leapfrog factors (O9 / O9b): H0^2 = (8 pi/3) M_tot / (box^3 Omega_m),
// K(a1,a2) = int da / (a^2 H), D(a1,a2) = int da / (a^3 H).  Einstein-de Sitter in closed form, any other
// Friedmann background by 16-point Gauss-Legendre on each (short) interval, fp64 on the host.
static double gl16(double a1, double a2, int apow, double om, double ol)
{
    static const double x[8] = {0.0950125098376374401853193, 0.2816035507792589132304605, 0.4580167776572273863424194,
                                0.6178762444026437484466718, 0.7554044083550030338951012, 0.8656312023878317438804679,
                                0.9445750230732325760779884, 0.9894009349916499325961542};
    static const double w[8] = {0.1894506104550684962853967, 0.1826034150449235888667637, 0.1691565193950025381893121,
                                0.1495959888165767320815017, 0.1246289712555338720524763, 0.0951585116824927848099251,
                                0.0622535239386478928628438, 0.0271524594117540948517806};
    const double ok = 1.0 - om - ol, c = 0.5 * (a1 + a2), h = 0.5 * (a2 - a1);
    double sum = 0.0;
    for (int i = 0; i < 8; i++)
        for (int sgn = -1; sgn <= 1; sgn += 2) {
            const double a = c + sgn * h * x[i];
            sum += w[i] / (pow(a, (double)apow) * sqrt(om / (a * a * a) + ok / (a * a) + ol));
        }
    return sum * h;
}

static void kdk_factors(const dsk_ctx *c, double mtot, double a, double da, double *k1, double *d, double *k2)
{
    if (!c->periodic) { *k1 = 0.5 * da; *d = da; *k2 = 0.5 * da; return; }
    const double PI = 3.14159265358979323846;
    const double H0 = sqrt(8.0 * PI / 3.0 * mtot / ((double)c->box * c->box * c->box) / c->omega_m);
    const double am = a + 0.5 * da, a1 = a + da;
    if (c->omega_m == 1.0 && c->omega_l == 0.0) {
        *k1 = 2.0 / H0 * (sqrt(am) - sqrt(a));
        *k2 = 2.0 / H0 * (sqrt(a1) - sqrt(am));
        *d = 2.0 / H0 * (1.0 / sqrt(a) - 1.0 / sqrt(a1));
        return;
    }
    *k1 = gl16(a, am, 2, c->omega_m, c->omega_l) / H0;
    *k2 = gl16(am, a1, 2, c->omega_m, c->omega_l) / H0;
    *d = gl16(a, a1, 3, c->omega_m, c->omega_l) / H0;
}

// K(a1, a2) = int dt/a, D(a1, a2) = int dt/a^2 over an arbitrary interval (isolated: a2 - a1)
static double kick_factor(const dsk_ctx *c, double mtot, double a1, double a2)
{
    double k1, d, k2;
    kdk_factors(c, mtot, a1, 2.0 * (a2 - a1), &k1, &d, &k2);
    return k1;
}
static double drift_factor(const dsk_ctx *c, double mtot, double a1, double a2)
{
    double k1, d, k2;
    kdk_factors(c, mtot, a1, a2 - a1, &k1, &d, &k2);
    return d;
}

extern "C" int dsk_set_cosmology(dsk_ctx *c, double omega_m, double omega_lambda)
{
    if (!c) return DSK_EINVAL;
    if (!(omega_m > 0.0) || !isfinite(omega_m) || !isfinite(omega_lambda)) return DSK_EINVAL;
    c->omega_m = omega_m; c->omega_l = omega_lambda;
    return DSK_OK;
}

extern "C" int dsk_set_softening(dsk_ctx *c, int kind, float length)
{
    if (!c || (kind != 0 && kind != 1) || !(length > 0.0f) || !isfinite(length)) return DSK_EINVAL;
    c->soft_kind = kind; c->eps = length;
    c->lists_valid = 0; c->pg_valid = 0; c->kdk_have_acc = 0;          // the K1 walk keeps cells out of the kernel's support: other lists
    return DSK_OK;
}

extern "C" int dsk_set_mac(dsk_ctx *c, int kind, float tol)
{
    if (!c || (kind != 0 && kind != 1)) return DSK_EINVAL;
    if (kind == 1 && (!(tol > 0.0f) || !isfinite(tol))) return DSK_EINVAL;
    c->mac_kind = kind; c->mac_tol = kind == 1 ? tol : 0.0f;
    c->lists_valid = 0; c->pg_valid = 0; c->kdk_have_acc = 0;
    return DSK_OK;
}

extern "C" int dsk_set_image_block(dsk_ctx *c, int ws)
{
    if (!c || !c->periodic || ws < 1 || ws > DSK_WS) return DSK_EINVAL;
    if (ws == c->img_ws) return DSK_OK;
    c->img_ws = ws;
    dsk_lattice_tensors((double)c->box, ws, c->far_T);         // the far field starts where the block ends
    if (c->ws_bytes) {
        DSK_CUDA(cudaMemcpyAsync(c->far_T_dev, c->far_T, sizeof(double) * DSK_NFAR, cudaMemcpyHostToDevice, c->stream));
        DSK_CUDA(cudaStreamSynchronize(c->stream));
    }
    c->lists_valid = 0; c->pg_valid = 0; c->kdk_have_acc = 0;
    return DSK_OK;
}

extern "C" int dsk_get_image_block(dsk_ctx *c, int *ws)
{
    if (!c || !ws) return DSK_EINVAL;
    *ws = c->periodic ? c->img_ws : 0;
    return DSK_OK;
}

extern "C" int dsk_set_background(dsk_ctx *c, int on)
{
    if (!c) return DSK_EINVAL;
    if (on && !c->periodic) return DSK_EINVAL;
    if ((on != 0) != (c->bg != 0)) { c->moments_p = -1; c->lists_valid = 0; c->pg_valid = 0; c->kdk_have_acc = 0; }   // rows and lists depend on it
    if (c->bg_closed != (on == 2)) c->kdk_have_acc = 0;
    c->bg = on ? 1 : 0;
    c->bg_closed = on == 2;
    return DSK_OK;
}

extern "C" int dsk_get_background(dsk_ctx *c, int *on, int *level, int *halfwidth, int64_t *ntop, double *rhobar)
{
    if (!c) return DSK_EINVAL;
    if (on) *on = c->bg;
    if (level) *level = c->bg_level;
    if (halfwidth) *halfwidth = dsk_bg_halfwidth(c->theta, c->bg_level, c->img_ws);
    if (ntop) *ntop = c->bg && c->have_tree ? (int64_t)c->ntop : 0;
    if (rhobar) {
        *rhobar = 0.0;
        if (c->bg && c->have_tree && c->moments_p == c->p) {
            double m = 0.0;
            DSK_CUDA(cudaMemcpyAsync(&m, c->mass64, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            DSK_CUDA(cudaStreamSynchronize(c->stream));
            *rhobar = m / ((double)c->box * c->box * c->box);
        }
    }
    return DSK_OK;
}

extern "C" int dsk_get_bg_moments(dsk_ctx *c, float *moments)
{
    if (!c || !moments || !c->bg) return DSK_EINVAL;
    if (!c->have_tree) return DSK_ENOTREE;
    if (c->moments_p != c->p) {
        int e = dsk_run_upward(c);
        if (e) return e;
    }
    return dsk_run_get_bg_moments(c, moments);
}

extern "C" int dsk_set_walk_mode(dsk_ctx *c, int mode)
{
    if (!c || mode < 0 || mode > 4) return DSK_EINVAL;
    c->walk_two_pass_only = mode;
    c->onepass_bad_theta = -1.0f;
    c->lists_valid = 0; c->pg_valid = 0;
    return DSK_OK;
}

extern "C" int dsk_set_walk_sharing(dsk_ctx *c, int groups)
{
    if (!c || groups < 0 || groups > 8) return DSK_EINVAL;
    c->walk_share = groups;
    c->lists_valid = 0; c->pg_valid = 0;
    return DSK_OK;
}

extern "C" int dsk_get_walk_info(dsk_ctx *c, int *predicted, int64_t *retries)
{
    if (!c) return DSK_EINVAL;
    if (predicted) *predicted = c->walk_predicted;
    if (retries) *retries = c->pg_retries;
    return DSK_OK;
}

extern "C" int dsk_kdk_reset(dsk_ctx *c)
{
    if (!c) return DSK_EINVAL;
    c->kdk_have_acc = 0;
    return DSK_OK;
}

// H^2 > 0 at both ends of the step (a closed model turns around; beyond that the factors are not defined)
static bool friedmann_ok(const dsk_ctx *c, double e0, double e1)
{
    const double ok = 1.0 - c->omega_m - c->omega_l;
    return c->omega_m / (e0 * e0 * e0) + ok / (e0 * e0) + c->omega_l > 0.0 &&
           c->omega_m / (e1 * e1 * e1) + ok / (e1 * e1) + c->omega_l > 0.0;
}

extern "C" int dsk_kdk_step(dsk_ctx *c, float *pos, float *vel, const float *mass, double a, double da)
{
    if (!c || !pos || !vel || !mass) return DSK_EINVAL;
    if (!c->ws) return DSK_ENOWORKSPACE;
    if (c->periodic && !(a > 0.0 && a + da > 0.0)) return DSK_EINVAL;
    if (c->periodic && !friedmann_ok(c, a, a + da)) return DSK_EINVAL;
    int e;
    if (!c->kdk_have_acc) {
        e = dsk_build_tree(c, pos, mass);
        if (e) return e;
        e = dsk_accel(c, pos, mass, c->kdk_acc, nullptr);
        if (e) return e;
        c->kdk_have_acc = 1;
    }
    // total mass = root monopole of the current tree (row 0 holds the root cell)
    float mroot = 0.0f;
    DSK_CUDA(cudaMemcpyAsync(&mroot, c->rows + 8, sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    double k1, d, k2;
    kdk_factors(c, (double)mroot, a, da, &k1, &d, &k2);
    cudaEventRecord(c->ev[15], c->stream);
    e = dsk_run_kick(c, vel, c->kdk_acc, (float)k1);
    if (e) return e;
    e = dsk_run_drift(c, pos, vel, (float)d);
    if (e) return e;
    cudaEventRecord(c->ev[16], c->stream);
    c->kdk_have_acc = 0;
    e = dsk_build_tree(c, pos, mass);
    if (e) return e;
    e = dsk_accel(c, pos, mass, c->kdk_acc, nullptr);
    if (e) return e;
    cudaEventRecord(c->ev[17], c->stream);
    e = dsk_run_kick(c, vel, c->kdk_acc, (float)k2);
    if (e) return e;
    cudaEventRecord(c->ev[18], c->stream);
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    c->stats.ms_kdk = ev_ms(c->ev[15], c->ev[16]) + ev_ms(c->ev[17], c->ev[18]);
    c->stats.n_launch += 2;                      // the first kick and the drift (build_tree reset the counter)
    c->kdk_have_acc = 1;
    return DSK_OK;
}


// One block step with hierarchical individual time steps (O9c).
extern "C" int dsk_kdk_block_step(dsk_ctx *c, float *pos, float *vel, const float *mass, uint8_t *rung, double a,
                                  double da, int rmax, float eta)
{
    if (!c || !pos || !vel || !mass || !rung) return DSK_EINVAL;
    if (!c->ws) return DSK_ENOWORKSPACE;
    if (rmax < 0 || rmax > DSK_RMAX || !(eta > 0.0f) || !(da > 0.0)) return DSK_EINVAL;
    if (c->periodic && !(a > 0.0)) return DSK_EINVAL;
    if (c->periodic && !friedmann_ok(c, a, a + da)) return DSK_EINVAL;
    int e;
    if (!c->kdk_have_acc) {
        e = dsk_build_tree(c, pos, mass);
        if (e) return e;
        e = dsk_accel(c, pos, mass, c->kdk_acc, nullptr);
        if (e) return e;
        c->kdk_have_acc = 1;
    }
    float mroot = 0.0f;
    DSK_CUDA(cudaMemcpyAsync(&mroot, c->rows + 8, sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    const double mtot = (double)mroot;
    const uint32_t nsub = 1u << rmax;
    const double h = da / (double)nsub;
    float kf[DSK_RMAX + 1];
    for (uint32_t s = 0; s < nsub; s++) {
        const double as = a + (double)s * h, at = a + (double)(s + 1) * h;
        for (int r = 0; r <= DSK_RMAX; r++) kf[r] = r <= rmax ? (float)kick_factor(c, mtot, as, as + (double)(nsub >> r) * h * 0.5) : 0.0f;
        e = dsk_run_kick_rung(c, vel, c->kdk_acc, rung, s, nsub, rmax, kf);
        if (e) return e;
        e = dsk_run_drift(c, pos, vel, (float)drift_factor(c, mtot, as, at));
        if (e) return e;
        c->kdk_have_acc = 0;
        e = dsk_run_rung_active(c, rung, s + 1, nsub, rmax, c->kdk_active);
        if (e) return e;
        e = dsk_build_tree(c, pos, mass);
        if (e) return e;
        e = dsk_accel_active(c, pos, mass, c->kdk_active, c->kdk_acc, nullptr);
        if (e) return e;
        for (int r = 0; r <= DSK_RMAX; r++) kf[r] = r <= rmax ? (float)kick_factor(c, mtot, at - (double)(nsub >> r) * h * 0.5, at) : 0.0f;
        e = dsk_run_kick_rung(c, vel, c->kdk_acc, rung, s + 1, nsub, rmax, kf);      // the same test: t % L == 0
        if (e) return e;
        e = dsk_run_rung_update(c, c->kdk_acc, c->kdk_active, rung, s + 1, nsub, rmax, (float)da, eta);
        if (e) return e;
    }
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    c->kdk_have_acc = 1;          // t = nsub ends every rung's step: kdk_acc holds the forces of all particles
    return DSK_OK;
}

// ---- introspection -------------------------------------------------------------------------------------
extern "C" int dsk_get_keys(dsk_ctx *c, uint64_t *sorted_keys, uint32_t *order)
{
    if (!c) return DSK_EINVAL;
    if (!c->have_tree) return DSK_ENOTREE;
    if (sorted_keys) DSK_CUDA(cudaMemcpyAsync(sorted_keys, c->key_a, 8 * (size_t)c->N, cudaMemcpyDeviceToDevice, c->stream));
    if (order) DSK_CUDA(cudaMemcpyAsync(order, c->idx_a, 4 * (size_t)c->N, cudaMemcpyDeviceToDevice, c->stream));
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return DSK_OK;
}

__global__ void k_unpack_cells(const dsk_cellrec *__restrict__ cell, uint32_t n, uint32_t *first, uint32_t *count,
                               uint8_t *nchild)
{
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    dsk_cellrec r = cell[i];
    if (first) first[i] = r.first;
    if (count) count[i] = r.count;
    if (nchild) nchild[i] = (uint8_t)(r.meta & 255u);
}

extern "C" int dsk_get_tree(dsk_ctx *c, int64_t *ncell, uint64_t *hotkey, uint32_t *first, uint32_t *count,
                            uint8_t *nchild)
{
    if (!c || !ncell) return DSK_EINVAL;
    if (!c->have_tree) return DSK_ENOTREE;
    const uint32_t n = c->hstate->ncell;
    *ncell = n;
    if (hotkey) DSK_CUDA(cudaMemcpyAsync(hotkey, c->hotkey, 8 * (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
    if (first || count || nchild) k_unpack_cells<<<(n + 255) / 256, 256, 0, c->stream>>>(c->cell, n, first, count, nchild);
    DSK_CUDA(cudaStreamSynchronize(c->stream));
    return DSK_OK;
}

static int get_moments_impl(dsk_ctx *c, float *com_mass, float *moments, int scaled)
{
    if (!c) return DSK_EINVAL;
    if (!c->have_tree) return DSK_ENOTREE;
    if (c->moments_p != c->p) {
        int e = dsk_run_upward(c);
        if (e) return e;
    }
    return dsk_run_get_moments(c, com_mass, moments, scaled);
}
extern "C" int dsk_get_moments(dsk_ctx *c, float *com_mass, float *moments) { return get_moments_impl(c, com_mass, moments, 0); }
extern "C" int dsk_get_moments_scaled(dsk_ctx *c, float *com_mass, float *moments) { return get_moments_impl(c, com_mass, moments, 1); }

__global__ void k_unpack_gbox(const float4 *__restrict__ gbox, uint32_t n, float *out)
{
    uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n) return;
    float4 lo = gbox[2 * (size_t)g], hi = gbox[2 * (size_t)g + 1];
    float *o = out + 6 * (size_t)g;
    o[0] = lo.x; o[1] = lo.y; o[2] = lo.z; o[3] = hi.x; o[4] = hi.y; o[5] = hi.z;
}

extern "C" int dsk_get_groups(dsk_ctx *c, int64_t *ngroup, uint32_t *first, uint32_t *count, float *bbox,
                              uint32_t *m2p_len, uint32_t *p2p_len)
{
    if (!c || !ngroup) return DSK_EINVAL;
    if (!c->have_tree) return DSK_ENOTREE;
    const uint32_t n = c->hstate->ngroup;
    *ngroup = n;
    cudaStream_t s = c->stream;
    if (first) DSK_CUDA(cudaMemcpyAsync(first, c->gfirst, 4 * (size_t)n, cudaMemcpyDeviceToDevice, s));
    if (count) DSK_CUDA(cudaMemcpyAsync(count, c->gcount, 4 * (size_t)n, cudaMemcpyDeviceToDevice, s));
    if (bbox) k_unpack_gbox<<<(n + 255) / 256, 256, 0, s>>>(c->gbox, n, bbox);
    if (m2p_len) DSK_CUDA(cudaMemcpyAsync(m2p_len, c->g_m2p_len, 4 * (size_t)n, cudaMemcpyDeviceToDevice, s));
    if (p2p_len) DSK_CUDA(cudaMemcpyAsync(p2p_len, c->g_p2p_len, 4 * (size_t)n, cudaMemcpyDeviceToDevice, s));
    DSK_CUDA(cudaStreamSynchronize(s));
    return DSK_OK;
}

extern "C" int dsk_get_stats(dsk_ctx *c, dsk_stats *out)
{
    if (!c || !out) return DSK_EINVAL;
    if (c->pending_build_ms || c->pending_force_ms) {
        DSK_CUDA(cudaStreamSynchronize(c->stream));
        finish_ms(c);
    }
    *out = c->stats;
    return DSK_OK;
}

extern "C" int dsk_get_param(const char *name, double *v)
{
    if (!name || !v) return DSK_EINVAL;
    if (!strcmp(name, "NLEAF")) *v = DSK_NLEAF;
    else if (!strcmp(name, "NCRIT")) *v = DSK_NCRIT;
    else if (!strcmp(name, "WS")) *v = DSK_WS_DEFAULT;
    else if (!strcmp(name, "WS_MAX")) *v = DSK_WS;
    else if (!strcmp(name, "KEY_LEVELS")) *v = DSK_KEY_LEVELS;
    else if (!strcmp(name, "FAR_ORDER")) *v = DSK_FAR_ORDER;
    else return DSK_EINVAL;
    return DSK_OK;
}

extern "C" int dsk_get_task_widths(int n, int widths[4])
{
    static constexpr dsk_parts_tab tab = dsk_make_parts_tab();
    if (!widths || n < 1 || n > DSK_NCRIT) return DSK_EINVAL;
    const uint32_t word = tab.w[(n + 1) / 2];
    for (int k = 0; k < 4; k++) widths[k] = (int)((word >> (8 * k)) & 255u);
    return DSK_OK;
}

extern "C" int dsk_get_lattice_tensors(dsk_ctx *c, double *T)
{
    if (!c || !T || !c->periodic) return DSK_EINVAL;
    memcpy(T, c->far_T, sizeof(double) * DSK_NFAR);
    return DSK_OK;
}

extern "C" const char *dsk_strerror(int e)
{
    switch (e) {
    case DSK_OK: return "ok";
    case DSK_EINVAL: return "invalid argument";
    case DSK_ENOWORKSPACE: return "workspace missing, too small or misaligned";
    case DSK_ENOTREE: return "no tree built";
    case DSK_EOUTOFBOX: return "position outside [0, box) in isolated mode";
    case DSK_ENONFINITE: return "non-finite position";
    case DSK_ELISTOVERFLOW: return "traversal stack or interaction list overflow";
    case DSK_ECUDA: return "CUDA error";
    case DSK_ECELLOVERFLOW: return "more tree cells or groups than the workspace holds";
    case DSK_ETOOLARGE: return "size beyond the fixed maximum of this no-allocation entry point (DSK_NOALLOC_NMAX)";
    default: return "unknown error";
    }
}
