/*
 * gothic.h -- C ABI of the B200-native GOTHIC hot path (Miki & Umemura, arxiv 1610.07279).
 *
 * What the library computes: Plummer-softened gravitational accelerations and potentials (eq. 1)
 * of the currently ACTIVE i-particles of a block time step, approximated by an oct-tree
 * walk over monopole pseudo j-particles under a multipole acceptance criterion (eq. 2 / eq. 5,
 * PAPER.md:68-89), plus the tree build (App. A) and block-step bookkeeping that feed it.
 *
 * Conventions
 *   - G = 1.  Positions, masses, outputs are FP32.
 *   - Unless a parameter says HOST, every array pointer is a DEVICE pointer owned by the caller; the library
 *     never frees or reallocates caller memory.  `stream` is a cudaStream_t passed as void* (NULL = default
 *     stream).  Calls enqueue work on `stream` and return without synchronising unless stated.
 *   - "sorted order" s: position in the space-filling-curve order produced by gothic_build_tree;
 *     perm[s] = original index of the particle at sorted position s.
 *   - Return value: 0 = GOTHIC_OK, negative = error.  Nothing throws or aborts.  On error outputs are
 *     unspecified.  An asynchronous capacity overflow (node pool, traversal stack) sets a device flag that
 *     gothic_get_tree_view / gothic_check report as GOTHIC_ERR_CAPACITY.
 *   - One context per stream; a context is not thread-safe.
 *   - There is no CPU fallback: without a CUDA device every compute call returns GOTHIC_ERR_CUDA.
 */
#ifndef GOTHIC_B200_H
#define GOTHIC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gothic_ctx gothic_ctx; /* opaque: owns keys, permutation, sorted positions, nodes, scratch */

enum {
    GOTHIC_OK = 0,
    GOTHIC_ERR_ARG = -1,           /* bad argument (NULL, n = 0, n > n_max, eps <= 0, ...) */
    GOTHIC_ERR_STATE = -2,         /* walk / update before a successful build */
    GOTHIC_ERR_CAPACITY = -3,      /* node pool or traversal stack overflow */
    GOTHIC_ERR_CUDA = -4,          /* CUDA runtime error (see gothic_last_cuda_error) */
    GOTHIC_ERR_UNIMPLEMENTED = -5,
    GOTHIC_ERR_TOO_LARGE = -6      /* gothic_active_list_static: n above GOTHIC_STATIC_ACTIVE_MAX_N */
};

enum { GOTHIC_KEY_PEANO_HILBERT = 0, GOTHIC_KEY_MORTON = 1 };   /* PAPER.md:54 / PAPER.md:564 */
enum { GOTHIC_BALL_GEO = 0, GOTHIC_BALL_EBS = 1, GOTHIC_BALL_COM = 2, GOTHIC_BALL_CMP = 3, GOTHIC_BALL_SEB = 4 };   /* enclosing ball of an i-group, App. B PAPER.md:568 items 3, 2, 4, 5, 1 */
enum { GOTHIC_MAC_ACCELERATION = 0, GOTHIC_MAC_OPENING_ANGLE = 1, GOTHIC_MAC_MULTIPOLE = 2 }; /* eq. 5 PAPER.md:85-89 / eq. 2 PAPER.md:68-72 / eq. 3-4 */

/* Allocates a context for up to n_max particles (n_max <= 2^30: the sort's look-back words carry 30-bit prefixes).
 *   node_max      node pool capacity; 0 -> 2*n_max (+64).  Must be < 2^28.
 *   group_size    G: number of consecutive sorted indices that share one traversal (PAPER.md:103-109,
 *                 "T_sub"; R3): 8, 16 or 32; 0 -> 32.  With G < 32 the spare lanes of the warp split
 *                 each i-particle's interaction list (ij-parallelisation, S = 32/G).
 *   scratch_bytes extra scratch for the traversal stacks; 0 -> automatic.
 * Synchronous (allocates device memory). */
int gothic_create(gothic_ctx **out, uint32_t n_max, uint32_t node_max, int group_size, size_t scratch_bytes);
void gothic_destroy(gothic_ctx *ctx);
const char *gothic_strerror(int code);       /* static strings */
const char *gothic_last_cuda_error(gothic_ctx *ctx); /* text of the last CUDA error seen by this context */

/* Tree build, PAPER.md:52-62 + App. A (steps B1-B6 of DESIGN.md):
 * root box -> 63-bit Peano-Hilbert (Listing 1) or Morton (Listing 3) keys -> stable radix sort of (key, index)
 * -> positions gathered into sorted order -> canonical oct-tree (breadth-first node ids, children contiguous)
 * -> pseudo j-particle moments m_J, r_J, b_J.
 *   pos_m   float4[n] (x, y, z, m), ORIGINAL order, device.
 *   n_leaf  a cell with more than n_leaf particles is subdivided (1..64; 0 -> 16).
 * Synchronises `stream` once (reads back the node count and per-level offsets). */
int gothic_build_tree(gothic_ctx *ctx, const float *pos_m, uint32_t n, int key_kind, int n_leaf, void *stream);

/* Pseudo j-particle moments only, on the existing topology (the paper recomputes them every step).
 *   pos_m_sorted  float4[n] in SORTED order, device; NULL -> keep the positions stored at build time.
 * Asynchronous. */
int gothic_update_moments(gothic_ctx *ctx, const float *pos_m_sorted, void *stream);

/* Gravity walk for the active i-particles, PAPER.md:95-132 (steps W1-W6 of DESIGN.md).
 * All index spaces are SORTED order.
 *   active        ascending sorted indices of the active particles, device; NULL -> all n particles.
 *   n_active      number of entries of `active` (ignored if active == NULL).
 *   n_active_dev  optional device uint32 that overrides n_active (lets set_timesteps feed the walk
 *                 without a host round trip); NULL -> use n_active.
 *   eps           Plummer softening length, > 0.
 *   mac_kind      GOTHIC_MAC_ACCELERATION: accept J iff d >= (m_J b_J^2 / (mac_param |a_old|))^(1/4)  (eq. 5)
 *                 GOTHIC_MAC_OPENING_ANGLE: accept J iff b_J / d <= mac_param                         (eq. 2)
 *                 GOTHIC_MAC_MULTIPOLE:     accept J iff d >= b_J/2 + sqrt(b_J^2/4 + sqrt(3 B_2 / mac_param)) (eq. 3-4), evaluated
 *                                           as d >= b_J and mac_param (d (d - b_J))^2 >= 3 B_2 (R16)
 *                 d measured from the surface of the group's enclosing ball (eq. 6-7; the ball is chosen
 *                 with gothic_set_ball).
 *   r_crit        critical separation of PAPER.md:122-126 (R13): a group's member list (ascending) whose
 *                 enclosing ball has b_I > r_crit is cut into its first ceil(k/2) members and the rest, recursively,
 *                 until b_I <= r_crit or one member is left; every piece walks the tree on its own.  INFINITY = never
 *                 split; 0 = every particle alone.  Must not be NaN or negative.  (The paper auto-tunes this number
 *                 from timings; here it is the caller's.  With INFINITY the few groups that straddle a jump of the
 *                 space-filling curve walk almost the whole tree and hold the last warps for milliseconds: pass a finite
 *                 value, e.g. a few per cent of the system's size.)
 *   aold          float[n] |a_old| per particle, sorted order; required iff mac_kind == ACCELERATION.
 *   acc_pot       float4[n] sorted order; ONLY active entries are written: (ax, ay, az, Phi).
 *   amag_out      optional float[n]: |a| of the new acceleration for active entries (may alias aold).
 *   n_interactions optional device counter, incremented by sum over walked pieces (#members x list length)
 *                 (counted in a separate run; pass NULL in timed runs).
 * Asynchronous. */
int gothic_walk_tree(gothic_ctx *ctx, const uint32_t *active, uint32_t n_active, const uint32_t *n_active_dev,
                     float eps, int mac_kind, float mac_param, float r_crit, const float *aold,
                     float *acc_pot, float *amag_out, unsigned long long *n_interactions, void *stream);

/* Block time steps (criterion from BASELINE.json configs[2], R6):
 * dt_i = eta sqrt(eps / |a_i|) floored to a power of two; level 0 = finest level present, clamped to
 * max_levels - 1; a particle is active at `substep` (1-based within the cycle) iff level <= ctz(substep).
 *   acc_pot       float4[n] accelerations, device; NULL -> keep `level` as is and only emit the active list.
 *   level         uint8[n] in/out.
 *   active        uint32[n] out: ascending indices of the active particles.
 *   n_active_dev  uint32 out (device).
 *   emin_nlev_dev int32[2] out (device): {exponent of the finest dt, number of levels}; written only when
 *                 acc_pot != NULL.  May be NULL.
 * Asynchronous. */
int gothic_set_timesteps(gothic_ctx *ctx, const float *acc_pot, uint32_t n, float eps, float eta, int max_levels,
                         uint32_t substep, uint8_t *level, uint32_t *active, uint32_t *n_active_dev,
                         int32_t *emin_nlev_dev, void *stream);

/* Read-only device views for parity tests; valid until the next build.  Synchronises `stream`. */
typedef struct {
    uint32_t n, n_nodes, n_levels_tree, group_size;
    float box[4];                 /* xmin, ymin, zmin, side */
    const uint64_t *key;          /* [n] sorted keys */
    const uint32_t *perm;         /* [n] */
    const float *pos_m_sorted;    /* float4[n] */
    const uint32_t *node_head, *node_num, *node_child; /* [n_nodes]; child = 0xFFFFFFFF for a leaf */
    const uint8_t *node_level, *node_nchild;           /* [n_nodes] */
    const uint32_t *level_ofs;    /* [23] device: id of the first node of each level */
    const float *node_com;        /* float4[n_nodes]: r_J, m_J */
    const float *node_b;          /* [n_nodes]: b_J */
    const float *node_b2;         /* [n_nodes]: B_2 = sum_j m_j |r_j - r_J|^2 (eq. 4) */
} gothic_tree_view;
int gothic_get_tree_view(gothic_ctx *ctx, gothic_tree_view *out, void *stream);

/* Synchronises `stream` and returns GOTHIC_ERR_CAPACITY / GOTHIC_ERR_CUDA if an asynchronous error was
 * flagged since the last check, else GOTHIC_OK.  The traversal-stack flag of a walk is sticky: it survives later
 * builds and walks until a check reads (and clears) it, so one check after a whole cycle validates every walk in it. */
int gothic_check(gothic_ctx *ctx, void *stream);

/* End-to-end convenience with HOST buffers (bench.py "e2e"): H2D copy of pos_m (and aold), build, one walk of
 * all particles, D2H copy of acc_pot in SORTED order and of perm.  Synchronises.
 *   pos_m_host float4[n] HOST; aold_host float[n] HOST in ORIGINAL order (NULL allowed for opening-angle MAC);
 *   acc_pot_host float4[n] HOST out (sorted order); perm_host uint32[n] HOST out (may be NULL). */
int gothic_gravity_host(gothic_ctx *ctx, const float *pos_m_host, uint32_t n, int key_kind, int n_leaf,
                        float eps, int mac_kind, float mac_param, float r_crit, const float *aold_host,
                        float *acc_pot_host, uint32_t *perm_host, void *stream);

/* One full block-step cycle end to end with HOST buffers (bench.py "e2e"; the paper's per-step loop PAPER.md:179-187
 * with static positions): H2D copy of pos_m and of the previous accelerations, tree build, block levels from the
 * previous accelerations (gothic_set_timesteps), then for substep = 1 .. 2^(n_levels-1): active list, pseudo-j moments
 * (recomputed every step), walk of the active particles with the acceleration MAC (eq. 5) using the
 * running |a| as |a_old|; finally D2H copy of the accelerations.  The last substep has every particle active, so
 * acc_pot_host is complete.  Synchronises (one small read-back of n_levels, one at the end).
 *   pos_m_host    float4[n] HOST (pinned for full speed), ORIGINAL order.
 *   acc_prev_host float4[n] HOST, ORIGINAL order: accelerations of the previous step (levels and |a_old|, R6/R7).
 *   acc_pot_host  float4[n] HOST out, ORIGINAL order.   level_host  uint8[n] HOST out, ORIGINAL order (may be NULL).
 *   info_host     int32[4] HOST out: {exponent of finest dt, n_levels, n_substeps, 0} (may be NULL).
 *   n_interactions_host  optional HOST out: interactions summed over the cycle (enables the device counter;
 *                        pass NULL in timed runs). */
int gothic_block_cycle_host(gothic_ctx *ctx, const float *pos_m_host, const float *acc_prev_host, uint32_t n, int key_kind,
                            int n_leaf, float eps, float eta, int max_levels, float delta_acc, float r_crit, float *acc_pot_host,
                            uint8_t *level_host, int32_t *info_host, unsigned long long *n_interactions_host, void *stream);

/* Enclosing ball of the pseudo i-particle used by the following walks (App. B): GOTHIC_BALL_GEO (default;
 * centre of the members' bounding cuboid), GOTHIC_BALL_EBS (Ritter's efficient bounding sphere; R17), GOTHIC_BALL_COM
 * (centre of mass of the members), GOTHIC_BALL_CMP (the smaller of GEO and COM) or GOTHIC_BALL_SEB (the smallest enclosing ball, by Welzl's
 * move-to-front recursion in single precision, R19; the costliest generator, PAPER.md:568 Table B.4).  In all of them the
 * radius is the exact maximum distance of the members from the centre.  Also decides the r_crit splitting (R13). */
int gothic_set_ball(gothic_ctx *ctx, int ball_kind);

/* Orbit integration under block time steps, section 2.7 (second-order predictor-corrector; NEXT row f1).
 * Every particle carries (r, v, a) at its own last corrected time t_last, an integer count of dt_unit = 2^e_min (the finest
 * step, {e_min, n_levels} from gothic_set_timesteps).  All arrays share ONE index space of the caller's choice (normally
 * the sorted order of the last build).  Single precision, one fused multiply-add per component (R15).
 *
 * gothic_predict: eq. 15-16 for ALL n j-particles: dt = (t_now - t_last[j]) dt_unit, v' = v + (dt/2) a, r' = r + dt v'.
 *   pos_m float4[n], vel float4[n] (vx,vy,vz,unused), acc_pot float4[n], t_last uint32[n]: in;  pos_pred float4[n]: out
 *   (x,y,z predicted, mass copied).  t_now >= every t_last.  Asynchronous; 68 B per particle. */
int gothic_predict(gothic_ctx *ctx, const float *pos_m, const float *vel, const float *acc_pot, const uint32_t *t_last,
                   uint32_t t_now, float dt_unit, uint32_t n, float *pos_pred, void *stream);

/* gothic_correct: eq. 17 for the ACTIVE i-particles (ascending indices as produced by gothic_set_timesteps):
 * v <- (v + (dt/2) a_old) + (dt/2) a_new, r <- pos_pred, a <- acc_new, t_last <- t_now; other particles untouched.
 *   active uint32[n_active] (NULL -> all n); n_active_dev optional device count overriding n_active.
 *   pos_pred, acc_new float4[n]: in (acc_new = output of gothic_walk_tree for this substep; must not alias acc_pot).
 *   pos_m, vel, acc_pot float4[n], t_last uint32[n]: in/out.
 *   level uint8[n] in/out, or NULL for no level migration.  With level: the level the new acceleration asks for is
 *   clamp(floor(log2(eta sqrt(eps/|a_new|))) - e_min, 0, max_levels-1) (same arithmetic as gothic_set_timesteps, R6);
 *   a particle moves to any FINER level at once and ONE level coarser only when t_now is a multiple of that coarser
 *   step (reading R15; the paper does not describe the migration).  Asynchronous. */
int gothic_correct(gothic_ctx *ctx, const uint32_t *active, uint32_t n_active, const uint32_t *n_active_dev, uint32_t n,
                   const float *pos_pred, const float *acc_new, uint32_t t_now, float dt_unit, float *pos_m, float *vel,
                   float *acc_pot, uint32_t *t_last, uint8_t *level, float eps, float eta, int e_min, int max_levels,
                   void *stream);

/* Live block time stepping: the paper's per-step loop with MOVING particles, state kept on the
 * device by the library in tree order.  One gothic_live_step is one block step: t_now += 1 (in units of dt_unit = 2^e_min),
 *   predict ALL particles to t_now (eq. 15-16) -> tree: rebuild from the predicted positions (and re-order the state by the new
 *   permutation), or keep the links and only recompute the pseudo-j moments from the predicted positions ->
 *   active list of the substep (level <= ctz(t_now)) -> walk of the active particles with the acceleration MAC (eq. 5,
 *   |a_old| = the particle's last |a|) -> correct the active particles (eq. 17) with level migration (reading R15).
 * When t_now reaches n_substeps = 2^(n_levels-1) every particle is synchronised: the levels are taken afresh from the new
 * accelerations (gothic_set_timesteps' arithmetic), t_now and every t_last return to 0, and one 8-byte read-back of
 * {e_min, n_levels} synchronises the stream (once per cycle).  A rebuild step synchronises once as well (gothic_build_tree reads back
 * the node count).  Everything else is asynchronous.
 *
 * gothic_live_init: pos_m float4[n], vel float4[n] (vx, vy, vz, unused) in ORIGINAL order; builds the tree, bootstraps the
 *   accelerations with an opening-angle walk (eq. 2, theta_boot; R7), takes the first levels.  Synchronises.
 * gothic_live_step: rebuild != 0 rebuilds the tree in this step.  n_interactions (device, optional) accumulates P:331's count.
 * gothic_live_get: device pointers of the current state (tree order; orig[s] = original index of row s) and the clock.
 *   The pointers stay valid until the next rebuild step or gothic_live_init; rows change with every step.
 * Errors: GOTHIC_ERR_ARG for bad arguments; GOTHIC_ERR_STATE before a successful gothic_live_init, after any other build on this
 *   context (gothic_build_tree, gothic_gravity_host, gothic_block_cycle_host: the rows no longer belong to the tree, even for the same
 *   n), and after a gothic_live_step that failed (its rows may be half-way through the step; the clock t_now and `steps` advance only
 *   when every stage of a step has been launched): call gothic_live_init again. */
typedef struct gothic_live_state {
    uint32_t n;
    uint32_t t_now;               /* substep index within the cycle, 0 .. n_substeps */
    uint32_t n_substeps;          /* 2^(n_levels-1) */
    int32_t e_min;                /* dt_unit = 2^e_min */
    int32_t n_levels;
    uint32_t steps_since_rebuild;
    unsigned long long steps;     /* block steps taken since gothic_live_init */
    const float *pos_m;           /* float4[n]: position at the row's own t_last, mass */
    const float *vel;             /* float4[n] */
    const float *acc_pot;         /* float4[n]: (ax, ay, az, Phi) at t_last */
    const float *amag;            /* float[n]: |a|, the next walk's |a_old| */
    const uint32_t *t_last;       /* uint32[n] */
    const uint8_t *level;         /* uint8[n] */
    const uint32_t *orig;         /* uint32[n] */
    const uint32_t *active;       /* uint32[n_active]: active rows of the last step (ascending) */
    const uint32_t *n_active;     /* device count of `active` */
} gothic_live_state;
int gothic_live_init(gothic_ctx *ctx, const float *pos_m, const float *vel, uint32_t n, int key_kind, int n_leaf, float eps,
                     float eta, int max_levels, float theta_boot, void *stream);
int gothic_live_step(gothic_ctx *ctx, float delta_acc, float r_crit, int rebuild, unsigned long long *n_interactions, void *stream);
int gothic_live_get(gothic_ctx *ctx, gothic_live_state *out);

/* Device times of the LAST gothic_live_step, for a caller that tunes the rebuild interval from timings as the paper does
 * (eq. 8-12: t_make against the growth of t_walk).  Every step records three CUDA events on its stream; this call
 * waits for the last of them (it synchronises with that step's walk, nothing else) and returns
 *   ms_host[0]  HOST out: the tree stage: predict + rebuild + state re-ordering on a rebuild step, predict + moments refresh otherwise;
 *   ms_host[1]  HOST out: active list + walk;
 *   n_active_host  HOST out, may be NULL: the step's number of active particles (a 4-byte read-back).
 * A step whose active list came back at the end of a cycle is timed like any other (the cycle's level pass is not in either figure).
 * Errors: GOTHIC_ERR_STATE before the first successful step of a live run. */
int gothic_live_timing(gothic_ctx *ctx, float *ms_host, uint32_t *n_active_host);

/* Active list of one substep for callers that must not allocate device memory.
 *
 * Who this is for.  Every other compute call needs a gothic_ctx, and gothic_create sizes and cudaMallocs its buffers.  That does
 * not suit a host program that took the GPU's memory for itself at start-up -- an N-body code whose particle arrays are sized to
 * fill the HBM, or a framework that keeps all device memory in its own pool -- because a later cudaMalloc there fails or takes
 * memory the program has promised elsewhere; nor a stepping loop that cannot afford the device-wide synchronisation that
 * cudaMalloc / cudaFree imply.  Such a caller still has to turn its block levels into the ascending active list of a substep
 * (T2 of DESIGN.md; level <= ctz(substep)), and this call does exactly that with the same three kernels as
 * gothic_set_timesteps(acc_pot = NULL), bit for bit the same output, without a context: it calls no cudaMalloc, cudaFree or
 * any library routine that allocates.
 *
 * Where the scratch lives.  The per-tile counts of the ordered compaction (one uint32 per 2048 particles) sit in a file-scope
 * `static __device__` array of GOTHIC_STATIC_ACTIVE_MAX_N / 2048 words = 128 KiB inside the library image; every GPU that loads
 * libgothic_b200.so holds those 128 KiB until the process exits, whether or not this call is ever made.
 *   level         uint8[n] device, in: block level of every particle.
 *   n             1 .. GOTHIC_STATIC_ACTIVE_MAX_N; a larger n returns GOTHIC_ERR_TOO_LARGE and launches nothing.
 *   substep       1-based substep of the cycle (> 0).
 *   active        uint32[n] device, out: ascending indices i with level[i] <= ctz(substep); entries past the count are untouched.
 *   n_active_dev  uint32 device, out: the count.
 * Errors: GOTHIC_ERR_ARG (NULL pointer, n = 0, substep = 0, device ordinal above 63), GOTHIC_ERR_TOO_LARGE, GOTHIC_ERR_CUDA
 * (no device, or a launch failed; cudaGetLastError has the reason).  Asynchronous on `stream` of the CURRENT device.
 *
 * First call on a device.  The first call made with a given device current looks up that device's address of the array
 * (cudaGetSymbolAddress, which may also make the runtime load the library's kernels there) and remembers it; make that call
 * before the stream is put into capture.  Later calls on that device do no set-up.
 *
 * Sharing.  All calls on one device use the same array, and it keeps what the last call left in it.  Nothing in it has to start
 * at zero (the count pass of a call writes every word that the call's scan then reads), so no clearing is done.  Two calls whose
 * kernels can overlap on the GPU -- different streams without an ordering between them, or two host threads -- race on the
 * array and produce garbage: serialise them (same stream, or an event). */
#define GOTHIC_STATIC_ACTIVE_MAX_N (1u << 26)
int gothic_active_list_static(const uint8_t *level, uint32_t n, uint32_t substep, uint32_t *active, uint32_t *n_active_dev,
                              void *stream);

/* Number of kernels this library has launched through this context (bench.py "gpu_launches"). */
unsigned long long gothic_launch_count(gothic_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* GOTHIC_B200_H */
