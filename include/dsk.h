/* dsk.h — C ABI of libdsk: B200-native tree gravity, the force path of 2HOT
 * (arxiv 1407.2600 "Dark Sky Simulations: Early Data Release").
 *
 * The operation: the gravitational field of N bodies is evaluated in O(N log N)
 * by approximating distant groups of bodies with truncated (order-p) multipole expansions held in the
 * cells of an oct-tree.  Stages: a Morton key per particle -> sort along the
 * space-filling curve -> oct-tree whose topology the keys define -> multipole moments of every cell
 * (upward pass) -> per sink group a traversal under a multipole acceptance test that yields the list
 * of cells to take as multipoles and the list of leaves to take particle by particle -> evaluation
 * of those lists (m sources x n sinks blocks) -> periodic boundary conditions through a
 * p = 8 local expansion of the far images -> symplectic leapfrog update.
 * The exact definitions (key bit layout, tree rule, MAC, expansion, softening, periodic split) are
 * the readings O1..O9 in DESIGN.md; G = 1.
 *
 * Conventions
 *  - Every array argument is a DEVICE pointer owned by the caller (e.g. a torch tensor's data_ptr())
 *    unless it says "host".  Layout: pos/vel/acc are AoS float32 [N,3] (the paper's particle record is
 *    32-bit x,y,z,vx,vy,vz); mass/pot float32 [N].  Outputs are in CALLER order.
 *  - The library allocates no device memory for its working set: the caller lends one workspace of
 *    dsk_workspace_bytes() bytes (256-byte aligned) with dsk_bind_workspace(); it must stay valid and
 *    untouched until dsk_destroy().  (A 4 KiB pinned host page and a few events are owned by the ctx.)
 *  - All device work is enqueued on the bound CUDA stream (default: the legacy default stream).  Each
 *    call that can fail on the device ends with ONE small device->host read of a status/counter block
 *    and a stream synchronise; everything before it is asynchronous.
 *  - Return value: 0 = DSK_OK, negative = error (below).  No exceptions, no printing, no global state.
 *    Calls on one context are not thread-safe; different contexts are independent.
 *  - There is no CPU fallback: without a CUDA device every compute call returns DSK_ECUDA.
 *
 * Multi-index order of moment arrays (interface convention): n = (a,b,c), rank l = a+b+c,
 * index(n) = l(l+1)(l+2)/6 + (b+c)(b+c+1)/2 + c  (ranks ascending; a descending, then b descending),
 * N_p = (p+1)(p+2)(p+3)/6 entries.
 */
#ifndef DSK_H
#define DSK_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DSK_OK             0
#define DSK_EINVAL        -1   /* bad argument (N <= 0, p not in {2,4,6,8}, theta not in (0,1], ...)   */
#define DSK_ENOWORKSPACE  -2   /* no workspace bound, or it is too small / misaligned                  */
#define DSK_ENOTREE       -3   /* dsk_accel / getters before a successful dsk_build_tree               */
#define DSK_EOUTOFBOX     -4   /* isolated mode: a position outside [0, box)                           */
#define DSK_ENONFINITE    -5   /* NaN or Inf position                                                  */
#define DSK_ELISTOVERFLOW -6   /* traversal stack or interaction-list buffer exhausted                 */
#define DSK_ECUDA         -7   /* CUDA runtime error (no device, launch failure, ...)                  */
#define DSK_ECELLOVERFLOW -8   /* more tree cells than the workspace was sized for                     */
#define DSK_ETOOLARGE     -9   /* size beyond the fixed maximum of a no-allocation entry point         */

typedef struct dsk_ctx dsk_ctx;      /* opaque; created by dsk_create, released by dsk_destroy        */

/* Counters and timings of the last dsk_build_tree / dsk_accel / dsk_kdk_step (host struct).
 * Interactions are USEFUL ones: sum over groups of n_sink x n_listed (self pairs included in n_p2p).
 * ms_* are CUDA-event times on the bound stream of the last call that ran that phase. */
typedef struct dsk_stats {
    int64_t n, ncell, nleaf_cells, ngroup, nlevel;
    int64_t n_p2p;            /* particle-particle interactions                                        */
    int64_t n_m2p;            /* cell-particle interactions                                            */
    int64_t list_m2p;         /* total M2P list entries (cells) over all groups                        */
    int64_t list_p2p;         /* total P2P list entries (leaves) over all groups                       */
    int64_t nbatch;           /* list batches the evaluation was split in                              */
    int64_t n_launch;         /* kernels launched since the last dsk_build_tree began (inclusive)      */
    int64_t list_bg;          /* background subtraction: cubes kept outside the groups' windows        */
    float ms_key, ms_sort, ms_build, ms_upward, ms_group, ms_walk, ms_p2p, ms_m2p, ms_far, ms_scatter,
          ms_kdk;
} dsk_stats;

/* Create a context for N particles in the cube [0, box)^3.  PAPER.md:61-63; O1-O7.
 *   periodic : 0 isolated, 1 periodic (explicit (2 WS+1)^3 image block + order-8 far field)
 *   eps      : Plummer softening length (> 0);  theta : opening angle, 0 < theta <= 1
 *   p        : expansion order = highest multipole rank kept, one of 2, 3, 4, 5, 6, 8 (the even ones are BASELINE.json's sweep; 3 and
 *              5 sit between them in cost and error, and 3 is what the absolute-error rule wants at an RMS error of 1e-4)
 * Host-only work (the lattice tensors of the far field are computed here in fp64). */
int dsk_create(dsk_ctx **out, int64_t N, float box, int periodic, float eps, float theta, int p);
int dsk_destroy(dsk_ctx *ctx);

/* Bytes of device workspace this context needs (depends on N and on the order p given to dsk_create: the
 * moment rows are sized for that order, so dsk_set_params may lower p but not raise it). */
size_t dsk_workspace_bytes(const dsk_ctx *ctx);
/* Lend the workspace (device pointer, >= dsk_workspace_bytes(), 256-byte aligned). */
int dsk_bind_workspace(dsk_ctx *ctx, void *dev_ptr, size_t bytes);
/* cudaStream_t as void* (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
int dsk_set_stream(dsk_ctx *ctx, void *cuda_stream);
/* Change eps / theta / p without rebuilding the tree (moments are recomputed when p changes, lists
 * when theta changes) — the (theta, p) sweep of BASELINE.json configs[1].  p may not exceed the p given
 * to dsk_create (the workspace is sized for that order): DSK_ENOWORKSPACE otherwise. */
int dsk_set_params(dsk_ctx *ctx, float eps, float theta, int p);

/* Keys -> sort -> octree -> groups -> upward pass (order p) for these positions and masses.
 * PAPER.md:61 (keys, tree), :57/:75 (moments).  pos dev [N,3], mass dev [N]; not retained. */
int dsk_build_tree(dsk_ctx *ctx, const float *pos, const float *mass);

/* Walk + evaluate: acc dev [N,3], pot dev [N] or NULL, caller order.  pos and mass are IGNORED (they may be NULL):
 * the forces are those of the positions and masses given to the last dsk_build_tree, whose sorted copy is used.  A
 * caller who has moved particles since must call dsk_build_tree again (dsk_kdk_step does).
 * PAPER.md:69-75 (lists, P2P, multipole interactions), :63 (periodic far field). */
int dsk_accel(dsk_ctx *ctx, const float *pos, const float *mass, float *acc, float *pot);

/* The same for an ACTIVE SUBSET of sinks: the force evaluation a hierarchical (block) time-step scheme needs
 * ("adaptive symplectic integrator (Quinn et al. 1997)").  active dev uint8 [N],
 * caller order: active[i] != 0 marks particle i as a sink; every particle remains a source.  Only sink groups that
 * hold an active particle are walked and evaluated; acc/pot entries of inactive particles are left untouched. */
int dsk_accel_active(dsk_ctx *ctx, const float *pos, const float *mass, const uint8_t *active, float *acc, float *pot);

/* The same for ONE SHARD of the sink groups (the sorted list is cut into pieces weighted
 * by work).  Every rank of a multi-GPU job holds all particles and builds the same tree; rank `rank` of `nranks` (<= 1023)
 * evaluates the contiguous run of sink groups (Morton order) whose work, n_sinks x (M2P list length x flop per M2P + P2P sources
 * x flop per pair) from a counting walk of ALL groups, falls into its 1/nranks of the total; every particle stays a source.
 * The cut is a function of the tree, theta and the acceptance rule alone, so the ranks agree on it without communicating.
 * acc/pot entries of particles in other shards are left untouched: with acc zero-filled beforehand, a sum-reduction over the
 * ranks (ncclAllReduce) assembles the full result.  first_group / end_group (host, may be NULL) receive the run [first, end). */
int dsk_accel_shard(dsk_ctx *ctx, int rank, int nranks, float *acc, float *pot, int64_t *first_group, int64_t *end_group);

/* One kick-drift-kick step of the comoving leapfrog (O9), in place:
 * vel is the canonical momentum per unit mass a^2 dx/dt; periodic: Einstein-de Sitter factors from
 * the total mass in the box, positions wrapped to [0,box); isolated: Newtonian with dt = da.
 * The first call evaluates the force at pos; later calls reuse the force cached by the previous
 * step (call dsk_kdk_reset after changing pos/vel by hand).  One force evaluation per step. */
int dsk_kdk_step(dsk_ctx *ctx, float *pos, float *vel, const float *mass, double a, double da);
int dsk_kdk_reset(dsk_ctx *ctx);

/* Background subtraction in a periodic box ("a technique to subtract the uniform background density";
 * reading O4b of DESIGN.md): the sources become particles - rho_bar, rho_bar = M_tot / box^3.  Cells of level <= l_b that
 * the walk accepts outside the sink group's window (a cube of level-l_b cells reaching k = ceil(1/theta) cells beyond the
 * group's cell) carry the moments of that difference over their cube; the background of the window and of the few coarse
 * cubes that stick out of it is summed exactly (closed-form field of a homogeneous cuboid); the far field acts on the
 * neutral box.  ON BY DEFAULT in a periodic context; on = 0 restores plain particle moments with the neutralising
 * background in the far field alone (and fp64 monopoles).
 * The window's field is summed by the series of the cube's interior potential about its centre where the sinks sit well inside
 * the window (within 0.36 of its half-width: every group at or below level l_b), by the closed form elsewhere; on = 2
 * (diagnostic) uses the closed form everywhere - the results agree to the rounding of the fp32 accumulators.
 * DSK_EINVAL for on != 0 in an isolated context.  Changing it invalidates moments, lists and the cached KDK force. */
int dsk_set_background(dsk_ctx *ctx, int on);
/* Pair softening law.  kind 0 (default): Plummer, phi = -m (r^2 + eps^2)^(-1/2), length = eps (the same as dsk_set_params' eps).
 * kind 1: Dehnen's K1 compensating kernel of compact support h = length ("using a Dehnen K1 compensating smoothing kernel
 * (Dehnen 2001)"; reading O6b of DESIGN.md): the point mass is the density 105/(64 pi h^3)(1 - u)(5 - 9u), u = r^2/h^2 < 1 (unit mass,
 * zero second moment), the pair force is -m d/h^3 (175/16 - 147/8 u + 135/16 u^2) inside h and exactly Newtonian outside.  Cells are then
 * expanded with the Newtonian Green's function and accepted only if all their sources lie farther than h from the sink group.
 * dsk_set_params keeps the kind and changes the length.  DSK_EINVAL for another kind or length <= 0. */
int dsk_set_softening(dsk_ctx *ctx, int kind, float length);
/* Acceptance rule of the walk.  kind 0 (default): the opening angle of dsk_create / dsk_set_params, accept iff
 * d^2 > (s/theta + delta)^2.  kind 1: an ABSOLUTE ERROR BOUND per cell interaction ("We adjust the error tolerance
 * parameter to limit absolute errors ..."; reading O5b of DESIGN.md): accept iff d^2 > (s + delta)^2 and
 *     (p + 2) Q b^(p-1) / (d^(p+1) (d - b)^2) <= tol,
 * Q = sum m |y - z|^2 over the cell (plus rho_bar times the cube's for a background-subtracted copy), b = sqrt(3)/2 s + delta,
 * d the distance from the cell's expansion centre to the sink group's box; tol > 0 in units of acceleration (G = 1).
 * theta still sets the window of background subtraction.  DSK_EINVAL for another kind or tol <= 0 with kind 1. */
int dsk_set_mac(dsk_ctx *ctx, int kind, float tol);
/* Half-width WS of the block of periodic images that is summed explicitly by the tree, (2 WS + 1)^3 images; everything
 * beyond it is the order-8 far field (reading O7 of DESIGN.md: "WS is measured, not assumed").  ws = 1 or 2;
 * 1 is the default (dsk_get_param "WS"), 2 the largest the library supports ("WS_MAX").  With background subtraction the far
 * field sees a neutral box and ws = 1 floors the force error at ~2e-4 of the rms force on a near-lattice box and ~3e-6 on a
 * clustered one (WS = 2: 5e-6 and 5e-9), for 11-18 % fewer cell interactions; WITHOUT subtraction ws = 1 floors at 3e-3 to
 * 2e-2: a context that switches subtraction off should set ws = 2.
 * DSK_EINVAL in an isolated context or for another value.  Invalidates lists and the cached KDK force. */
int dsk_set_image_block(dsk_ctx *ctx, int ws);
int dsk_get_image_block(dsk_ctx *ctx, int *ws /* host; 0 in an isolated context */);
/* host pointers, each may be NULL: on / off, l_b, the window half-width k for the current theta, the number of cells of
 * level <= l_b in the current tree (0 when off or no tree) and rho_bar (0 unless the moments are up to date). */
int dsk_get_background(dsk_ctx *ctx, int *on, int *level, int *halfwidth, int64_t *ntop, double *rhobar);
/* the subtracted moments of those cells (canonical order: they are the first ntop cells) in units of the cell side,
 * M'_n / s^|n|, dev [ntop, N_p]; DSK_EINVAL when subtraction is off. */
int dsk_get_bg_moments(dsk_ctx *ctx, float *moments);

/* Diagnostic: mode 0 (default) lets the walk try its one-pass form (lists written into a fixed capacity per group,
 * fallback to COUNT + FILL when one does not fit); mode 1 always takes the two-pass form; mode 2 gives the one-pass
 * attempt capacities that overflow, so that every evaluation exercises the fallback; mode 3 takes the two-pass form and
 * pretends the list buffers hold 65536 / 8192 entries, so that even a small input is evaluated in batches of groups (the
 * path a 512^3 run takes).  Results are identical in modes 0-3.  Mode 4 pretends they hold 256 / 8 entries: a group whose
 * lists are longer cannot be evaluated and dsk_accel returns DSK_ELISTOVERFLOW (the context stays usable). */
int dsk_set_walk_mode(dsk_ctx *ctx, int mode);

/* The walk variant (second half; "bundle a set of m source cells which have interactions in
 * common with a set of n sink particles"): up to `groups` consecutive sink groups (neighbours along the Morton curve, and, with
 * background subtraction, of one window) are walked by one warp.  Against the union of their boxes it lists once, for all of them,
 * every cell the union accepts, opens once every cell all of them reject, and sets aside the cells they disagree on, which each
 * group then walks by itself.  Every group's lists hold exactly the entries a walk of its own would give, in another order, so the
 * forces differ by fp32 summation order only.  groups = 1: every group walks alone; 2..8: share; 0 (default): as many (<= 8) as
 * leave every SM 16 walks.  Sharded, batched and active-subset evaluations list a group's entries in the same order as a full one
 * (the sets are formed from the group indices, not from what is evaluated).  DSK_EINVAL outside 0..8. */
int dsk_set_walk_sharing(dsk_ctx *ctx, int groups);

/* How the last evaluation sized its lists (introspection; host pointers, either may be NULL).  When the lists do not fit a fixed
 * capacity per group (very large N: 512^3), an evaluation normally walks twice, COUNT then FILL.  From its second evaluation on the
 * context instead sizes every group's list slots from the lengths the groups of the same region of the Morton curve had in the
 * previous evaluation (plus a half) and walks once; a list that outgrows its slot makes the evaluation start over with COUNT + FILL
 * (same results, the time of one walk lost) and the context sit out a few evaluations before predicting again.
 * predicted: 1 if the last evaluation walked once into predicted slots and they held; retries: evaluations started over so far. */
int dsk_get_walk_info(dsk_ctx *ctx, int *predicted, int64_t *retries);

/* One BLOCK step of size da with hierarchical individual time steps (reading O9c of DESIGN.md; "adaptive
 * symplectic integrator (Quinn et al. 1997)").  rung dev uint8 [N], in/out: particle i takes steps of da / 2^rung[i],
 * 0 <= rung <= rmax <= 8 (a larger entry is read as rmax and written back clamped).  The block is cut into 2^rmax substeps; per substep: opening half kicks of the particles whose
 * step starts, drift of all, tree + forces of the particles whose step ends (dsk_accel_active), their closing half kicks,
 * and their new rung from step_i = eta sqrt(eps / |acc_i|), rung = ceil(log2(da / step_i)) (decided in fp32; finer at
 * once, coarser one level at a time and only when synchronised).  rmax = 0 is dsk_kdk_step.  Same state, cached force
 * and factors as dsk_kdk_step. */
int dsk_kdk_block_step(dsk_ctx *ctx, float *pos, float *vel, const float *mass, uint8_t *rung, double a, double da,
                       int rmax, float eta);

/* Background cosmology of the periodic leapfrog (the paper's runs use
 * Omega_m = 0.295, Omega_Lambda = 0.705).  H(a) = H0 sqrt(Omega_m a^-3 + (1 - Omega_m - Omega_Lambda) a^-2 + Omega_Lambda),
 * H0^2 = (8 pi/3) M_tot / (box^3 Omega_m); kick = int da/(a^2 H), drift = int da/(a^3 H), integrated on the host in
 * fp64.  Default (1, 0) = Einstein-de Sitter.  omega_m > 0 and H^2 > 0 on the steps taken; DSK_EINVAL otherwise. */
int dsk_set_cosmology(dsk_ctx *ctx, double omega_m, double omega_lambda);

/* ---- introspection (parity tests, reporting) ---------------------------------------------------- */
/* sorted keys and the permutation: sorted_keys[r] = key(order[r]); dev [N] each (either may be NULL). */
int dsk_get_keys(dsk_ctx *ctx, uint64_t *sorted_keys, uint32_t *order);
/* tree topology in canonical (ascending hotkey) order; *ncell is always written (host pointer); the
 * arrays are dev [ncell] and may be NULL. */
int dsk_get_tree(dsk_ctx *ctx, int64_t *ncell, uint64_t *hotkey, uint32_t *first, uint32_t *count,
                 uint8_t *nchild);
/* per cell (canonical order): com_mass dev [ncell,4] = (com x,y,z, mass); moments dev [ncell,N_p] =
 * raw (unscaled) Cartesian moments M_n = sum m (y - com)^n of the current order p.  Either may be NULL. */
int dsk_get_moments(dsk_ctx *ctx, float *com_mass, float *moments);
/* the same with the moments in units of the cell side s = box 2^-level: M_n / s^|n| (what the library stores: at p = 8
 * the raw moments of a level >= 15 cell, ~ m s^8, are below the fp32 range, SURVEY.md section 7 hard part 2). */
int dsk_get_moments_scaled(dsk_ctx *ctx, float *com_mass, float *moments);
/* sink groups in Morton order: *ngroup host; first/count dev [ngroup], bbox dev [ngroup,6] (min, max);
 * m2p_len/p2p_len dev [ngroup] = list lengths of the last walk (cells / leaves).  Arrays may be NULL. */
int dsk_get_groups(dsk_ctx *ctx, int64_t *ngroup, uint32_t *first, uint32_t *count, float *bbox,
                   uint32_t *m2p_len, uint32_t *p2p_len);
int dsk_get_stats(dsk_ctx *ctx, dsk_stats *out /* host */);
/* library constants: "NLEAF", "NCRIT", "WS" (default image-block half-width), "WS_MAX", "KEY_LEVELS", "FAR_ORDER"; host pointer. */
int dsk_get_param(const char *name, double *value);
/* How the force kernels cut a sink group of n (1..NCRIT) sinks into warp tasks: widths[k] =
 * sink lanes (two sinks each) of task k, 0 for unused tasks; the widths sum to ceil(n/2), each <= 32.  Host pointer;
 * DSK_EINVAL outside 1..NCRIT.  Introspection for tests and for the bench's accounting; no device work. */
int dsk_get_task_widths(int n, int widths[4]);
/* far-field lattice tensors T_n (|n| <= 8, 165 doubles, host) of this context; periodic only. */
int dsk_get_lattice_tensors(dsk_ctx *ctx, double *T /* host [165] */);
/* FP32 issue-rate probe: the measured denominator of the force kernels' roofline (the force path of
 * PAPER.md:73-75 is FP32 FMA work).  Runs a pure FMA kernel on the current device (default stream, its own few MB of
 * device memory) and writes to HOST pointers: TFLOP/s (FMA = 2 flop per lane), cycles per warp instruction per SM
 * sub-partition, and the SM clock in MHz the kernel ran at.  variant 0: packed fma.rn.f32x2 with three register operands;
 * 1: packed, one operand a scalar broadcast to both halves (the form the force kernels feed sources in); 2: scalar FFMA
 * with three distinct registers; 3 and 4: packed and scalar with the two source operands repeated from one instruction to
 * the next (operand-reuse cache; 0-2 are register-bandwidth bound); 5 and 6: the M2P body's pattern, a new scalar coefficient
 * every instruction / every second instruction.  DSK_EINVAL for another variant or a NULL pointer,
 * DSK_ECUDA without a device. */
int dsk_probe_fp32_peak(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz);
/* the same, plus TFLOP/s as implied by the SMs' own cycle counters and clock (cross-check of the event timing) */
int dsk_probe_fp32_peak_ex(int variant, double *tflops, double *cycles_per_inst_smsp, double *sm_mhz, double *tflops_by_cycles);

/* Steps K and S with NO allocation and no context ("assign a Key to each particle, based on Morton ordering";
 * the sort along the curve), for callers that can neither call cudaMalloc nor lend a workspace (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid allocation).  The same kernels as dsk_build_tree's key and sort
 * phases; their scratch (second key / index buffer, tile histograms, scan sums, status word) is a fixed file-scope device
 * array of 12.6 MiB that every GPU which loads the library holds until the process exits.
 *   pos dev [N][3] fp32, N <= DSK_NOALLOC_NMAX; box, periodic as in dsk_create;
 *   sorted_keys dev [N] uint64 (out), order dev [N] uint32 (out): sorted_keys[r] = key(order[r]), equal keys in input order —
 *   bit for bit what dsk_get_keys returns after dsk_build_tree on the same positions;  cuda_stream: cudaStream_t as void*,
 *   NULL = default stream; the work is enqueued there on the CURRENT device, and the call returns after one 4-byte read-back
 *   and a stream synchronise.
 * Calls no cudaMalloc / cudaFree and no allocating library routine.  Every call on a device shares the one array, which keeps
 * the last call's contents (what must start at zero is cleared at the start of each call): calls that OVERLAP on the same
 * GPU (two streams, two host threads) race on it and give wrong orders — serialise them.
 * Errors: DSK_ETOOLARGE for N > DSK_NOALLOC_NMAX (nothing is launched); DSK_EINVAL for N <= 0, a NULL pointer or a bad box;
 * DSK_EOUTOFBOX / DSK_ENONFINITE as dsk_build_tree (outputs then undefined); DSK_ECUDA. */
#define DSK_NOALLOC_NMAX 1048576
int dsk_sort_keys_noalloc(const float *pos, int64_t N, float box, int periodic, uint64_t *sorted_keys, uint32_t *order,
                          void *cuda_stream);
const char *dsk_strerror(int err);

#ifdef __cplusplus
}
#endif
#endif
