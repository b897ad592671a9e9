/* bh.h -- C ABI of the B200-native Barnes-Hut force pipeline (arxiv/paper_1106_1900, "Bonsai").
 *
 * One step of the paper's method (PAPER.md = /root/reference/PAPER.md, "L<n>" = line n):
 *   S0 domain box (L374)            S1 60-bit Morton keys (L374-392)      S2 stable key radix sort (L59, L352, L362)
 *   S3 reorder by the sort (L174)   S4 sparse octree, <= nleaf per leaf (L63-65, Fig.1-2)
 *   S5 groups, <= ncrit (L75)       S6 monopole + quadrupole moments in fp64, boxes (L109-115, L127, L266)
 *   S7 group walk, MAC d > l/theta + delta (L83-87, Eq.1)          S8 softened p-p / p-c forces + potentials (L85, L97)
 *   S9 shared-step leapfrog (L105)
 * Every step runs in hand-written sm_100a CUDA kernels inside this library; there is no CPU fallback.
 *
 * Conventions
 *   - Units: N-body units, G = 1 (L238).  Arithmetic: fp32 except the moments (fp64), as in the paper (L154, L170).
 *   - Particle layout: pos_mass = float[n][4] (x, y, z, m); vel = float[n][4] (vx, vy, vz, unused);
 *     acc_pot = float[n][4] (ax, ay, az, phi); id = uint32[n] (caller identity).
 *   - The library keeps the particle state inside the caller-provided WORKSPACE, in key-sorted order
 *     (bh_tree_build re-sorts it; `id` follows the particles).  bh_set_particles / bh_get_particles copy in / out;
 *     bh_bind_particles borrows the caller's device arrays as that state instead (no copy).
 *   - Memory: the library never allocates device memory.  `d_workspace` is device memory owned by the caller
 *     (e.g. a torch tensor) and must stay alive until bh_destroy.  Host objects are owned by the ctx.
 *   - Streams: `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  bh_tree_build,
 *     bh_compute_forces and bh_leapfrog_step only enqueue work: no host synchronisation, no host<->device copies,
 *     so they can be captured into a CUDA graph.  One ctx = one stream at a time; not thread-safe.
 *   - Errors: every call returns BH_OK (0) or a negative bh_status; nothing throws or exits.  Errors that only the
 *     device can see (non-finite input, capacity overflow) are recorded in a device status word and reported by
 *     bh_sync_status.
 */
#ifndef BH_B200_H
#define BH_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum bh_status {
    BH_OK = 0,
    BH_ERR_INVALID_ARG = -1, /* null pointer, n <= 0, n > n_max, theta <= 0 or non-finite, eps < 0, non-finite dt, bad config */
    BH_ERR_WORKSPACE = -2,   /* workspace too small or not device memory */
    BH_ERR_STATE = -3,       /* forces before build, step before forces, build before particles */
    BH_ERR_CUDA = -4,        /* a CUDA runtime call failed (bh_last_cuda_error gives the code); also the deferred status when a
                              * bounded device-side wait (grid barrier of the front end, look-back of a sort pass) ran out:
                              * the kernels then finish without writing out of bounds, but the build is not valid */
    BH_ERR_NONFINITE = -5,   /* deferred: NaN/Inf position or mass <= 0 seen by S0 (A27) */
    BH_ERR_CAPACITY = -6,    /* deferred: more cells than max_cells */
    BH_ERR_TOO_LARGE = -7    /* bh_domain_box_static only: n is above BH_DOMAIN_STATIC_MAX_N, the built-in scratch cannot hold it */
} bh_status;

/* Tunables.  Zero-initialise and override; 0 means "default". */
typedef struct bh_config {
    int32_t nleaf;     /* max particles per leaf, 1..64; default 16 (L63) */
    int32_t ncrit;     /* max particles per group, 1..64; default 64 (L75) */
    int64_t max_cells; /* cell capacity; default = the hard bound n_max + 20*(n_max/(nleaf+1)) + 1 */
    int64_t list_entries; /* capacity of the interaction-list buffer (S7 -> S8), 4-byte entries; default
                           * clamp(320 * n_max, 2^22, 2^30).  Bounds memory only: groups whose lists do not fit are walked and
                           * evaluated by the fused kernel, with identical counts and forces within rounding. */
    int32_t walk_mode; /* 0 (default): list walk + list evaluation, fused kernel for what does not fit; 1: fused kernel only */
    int32_t walk_waves; /* 0 (default): as few waves of groups as the list buffer allows (normally 1), one after the other;
                         * k > 1: at least k waves, run as a pipeline (list walk of wave w + 1 beside the evaluation of
                         * wave w on internal streams); 0..255 */
    int32_t front_mode; /* 0 (default): S0-S3 in one cooperative launch whenever every sort tile is resident at once
                         * (n <= 8192 x SMs, 1.2 M on B200), with the short sort (radix passes over the leading key bits only,
                         * then every run of equal leading bits finished in place; the full sort is redone on the device if a
                         * run is too long: bh_stats.sort_retries); 1: always one launch per step and sort pass (any n);
                         * 2: the cooperative launch with all 8 radix passes.  The result is the same stable order in all three */
    int32_t walk_private; /* 0 (default): the eight groups of a block share the common part of their walks (cells every one of
                           * them accepts / opens, decided once against the union of their boxes; exact, see walk_lists.cu);
                           * 1: every group walks from the root on its own.  Counts are identical; the order of the list
                           * entries, and with it the last bits of the fp32 sums, differs between the two */
} bh_config;

typedef struct bh_ctx bh_ctx;

/* What a step produced.  Filled by bh_sync_status (which synchronises the stream). */
typedef struct bh_stats {
    int32_t status;        /* deferred device status: BH_OK, BH_ERR_NONFINITE, BH_ERR_CAPACITY, BH_ERR_CUDA (a bounded device-side
                            * wait ran out) or BH_ERR_STATE (block time-steps: the 32-bit tick counter is about to end) */
    int32_t n_levels;      /* deepest occupied level + 1 */
    int64_t n;             /* particles */
    int64_t n_cells;       /* tree cells (S4) */
    int64_t n_groups;      /* groups (S5) */
    int64_t sum_pc;        /* particle-cell interactions evaluated by the last bh_compute_forces: sum_g n_g * n_pc[g] */
    int64_t sum_pp;        /* particle-particle interactions: sum_g n_g * n_pp[g] (includes the self term) */
    int64_t sum_mac;       /* MAC evaluations (Eq.1) in the last walk */
    int64_t launches;      /* kernels launched by this ctx since bh_create */
    float   lo[3];         /* S0: domain corner */
    float   hi[3];         /* S0: per-axis maximum */
    int32_t domain_exp;    /* S0: cube side = 2^domain_exp */
    int32_t sort_retries;  /* S2: times since bh_create the short sort (leading key bits + fix-up) had to be redone in full */
    int32_t sort_passes;   /* S2: radix passes of the last build's first sort (8: the full sort; fewer: the short sort) */
    int32_t reserved;
} bh_stats;

/* Device pointers into the workspace, valid until the next bh_tree_build / bh_set_particles (particle arrays) or
 * bh_destroy.  All arrays are in the canonical numbering of DESIGN.md: cells level-major, ascending first particle
 * within a level (A10); groups in particle order.  Filled by bh_export_tree, which enqueues one conversion kernel on
 * `stream` (the caller synchronises before reading).  n_cells / n_groups come from bh_sync_status. */
typedef struct bh_tree_view {
    const float*    pos_mass;      /* float[n][4], sorted */
    const float*    vel;           /* float[n][4], sorted */
    const float*    acc_pot;       /* float[n][4], sorted; valid after bh_compute_forces */
    const uint32_t* id;            /* uint32[n] */
    const uint64_t* key;           /* uint64[n], sorted Morton keys (S1, S2) */
    const uint32_t* perm;          /* uint32[n]: position BEFORE this build of the j-th sorted particle (S2) */
    const uint32_t* level_offset;  /* uint32[22]: cells of level L are [level_offset[L], level_offset[L+1]) */
    const int32_t*  cell_level;    /* int32[C] */
    const uint64_t* cell_prefix;   /* uint64[C]: key >> (60 - 3 level) */
    const uint32_t* cell_pbegin;   /* uint32[C]: first particle */
    const uint32_t* cell_pcount;   /* uint32[C] */
    const int32_t*  cell_child_begin; /* int32[C]: first child, -1 for a leaf */
    const int32_t*  cell_nchild;   /* int32[C]: 0 for a leaf */
    const int32_t*  cell_parent;   /* int32[C]: -1 for the root */
    const double*   cell_mom64;    /* double[C][10]: M, com xyz, Qxx, Qyy, Qzz, Qxy, Qxz, Qyz (S6, fp64) */
    const float*    cell_box;      /* float[C][6]: min xyz, max xyz (S6) */
    const float*    cell_mom32;    /* float[C][10]: the fp32 roundings used by the walk; valid after bh_compute_forces */
    const float*    cell_r2open;   /* float[C]: (l/theta + delta)^2 (Eq.1); valid after bh_compute_forces */
    const float*    cell_trec;     /* float[C][4]: what a MAC test of the walk reads: (com xyz as fp32, r2open); valid after bh_compute_forces */
    const float*    cell_erec;     /* float[C][12]: what an accepted cell costs the force loop (S8): (com xyz, M) (-3Qxx, -3Qyy, -3Qzz, -3Qxy)
                                    * (-3Qxz, -3Qyz, -T/2, -3T/2), T = Qxx + Qyy + Qzz, every entry one fp32 operation on the fp32 roundings */
    const uint32_t* group_begin;   /* uint32[G+1]: first particle of each group; group_begin[G] = n (S5) */
    const uint32_t* group_cell;    /* uint32[G]: the cell a group comes from */
    const uint32_t* group_npc;     /* uint32[G]: accepted cells per group (S7); valid after bh_compute_forces */
    const uint32_t* group_npp;     /* uint32[G]: particles of opened leaves per group (S7) */
} bh_tree_view;

/* Bytes of device workspace needed for up to n_max particles (host-only, pure).  0 on a bad argument. */
size_t bh_workspace_bytes(int64_t n_max, const bh_config* cfg);

/* Create a context on the device that owns `d_workspace` (256-byte aligned device memory, `bytes` long).
 * cfg may be NULL (defaults).  The device is taken from the pointer. */
int bh_create(bh_ctx** out, int64_t n_max, const bh_config* cfg, void* d_workspace, size_t bytes);
int bh_destroy(bh_ctx* ctx);

/* Copy n particles into the workspace (cudaMemcpyAsync on `stream`; pointers may be host or device memory, host
 * memory should be pinned for the copy to be asynchronous).  vel may be NULL (zeros); id may be NULL (0..n-1).
 * Invalidates tree and forces.  The velocity and id copies run on an internal stream beside S0-S2 of the next
 * bh_tree_build (which only need positions) and are joined by an event before anything reads them; under stream
 * capture every copy stays on `stream`.  All source buffers must stay valid until the work enqueued on `stream` by the
 * next bh_tree_build / bh_get_particles (or a synchronisation after it) has completed. */
int bh_set_particles(bh_ctx* ctx, int64_t n, const float* pos_mass, const float* vel, const uint32_t* id, void* stream);

/* Borrow the caller's DEVICE arrays as the simulation state instead of copying it in (section 1 and PAPER.md:264
 * section 5: the particles live on the GPU and no step moves them to the host or back).
 * d_pos_mass, d_vel, d_acc_pot: float[n][4], 16-byte aligned; d_id: uint32[n]; all on the context's device, n <= n_max.
 * Nothing is copied, zeroed or enqueued: the four arrays take the place of the workspace's first set of particle arrays
 * and of its acc_pot array, and every later call reads and writes them directly on the stream it is given (the caller orders
 * its own accesses against those streams).  Invalidates tree and forces, like bh_set_particles; acc_pot is not read before
 * the first force evaluation has written it.  The arrays are borrowed until bh_set_particles (which goes back to the
 * workspace's own arrays), another bh_bind_particles or bh_destroy.
 * Where the state is afterwards.  acc_pot: always the caller's array, rows in the current key-sorted order.  Positions,
 * velocities and ids: S3 gathers them from one set of arrays into the other (caller's -> workspace's, workspace's -> caller's),
 * so after an EVEN number of builds since the binding (bh_tree_build, and the one inside every bh_leapfrog_step,
 * bh_step_graph_launch and bh_block_step with rebuild) the caller's arrays hold the current sorted state, and after an odd
 * number the workspace does (bh_export_tree gives the pointers either way).  bh_land_particles makes the caller's arrays
 * current in that case with one device-to-device copy of 36 bytes per particle (nothing is enqueued when they already are);
 * tree, forces and block state stay valid.  A run that steps in pairs never copies a particle. */
int bh_bind_particles(bh_ctx* ctx, int64_t n, float* d_pos_mass, float* d_vel, float* d_acc_pot, uint32_t* d_id);
int bh_land_particles(bh_ctx* ctx, void* stream);

/* Copy the current (key-sorted) state out; any pointer may be NULL; host or device destinations.  BH_ERR_STATE when
 * acc_pot is asked for between a bh_tree_build (which re-sorts the particles) and the next evaluation that puts every row
 * in the new order (bh_compute_forces, bh_leapfrog_step, bh_step_graph_launch, bh_block_step with a rebuild): the stored
 * accelerations would be in the previous order.  bh_compute_forces_active alone does not lift this: it writes the rows of
 * the walked groups only. */
int bh_get_particles(bh_ctx* ctx, float* pos_mass, float* vel, float* acc_pot, uint32_t* id, void* stream);

/* S0-S6: domain, keys, sort, reorder, octree, groups, fp64 moments and boxes (L55-65, L107-115).  theta-independent.
 * S2 produces THE stable ascending order of the 60-bit keys (L362).  How: radix passes over the leading key bits only, every
 * run of keys with equal leading bits finished in place, and the full 8-pass sort redone ON THE DEVICE when a run is too long
 * for that (no host round trip; bh_stats.sort_passes / sort_retries say what happened; bh_config.front_mode = 2 sorts all 60
 * bits in the first place).  The number of leading bits is a guess from n (one-launch front end) or from the depth of the
 * previous tree on this context (any n): it changes the time, never the result.  A grid barrier or look-back that exceeds its
 * spin limit (a device fault) sets the deferred status BH_ERR_CUDA and lets the kernel finish with an unspecified order. */
int bh_tree_build(bh_ctx* ctx, void* stream);

/* S7-S8 on the current tree: opening radii for `theta` (Eq.1), group walk, p-p and p-c forces + potentials
 * with Plummer softening `eps` (L85, L97).  Needs bh_tree_build.  eps = 0 with coincident particles is undefined. */
int bh_compute_forces(bh_ctx* ctx, float theta, float eps, void* stream);

/* Block time-steps (L105 "... or on a subset of particles in case of the block-time step regime"; L264-266).  The paper
 * gives two device-side ingredients and leaves the step criterion open (not part of this library, A23):
 *
 * bh_refresh_moments: S6 again on the EXISTING cells and groups after the particles moved (bh_kick_drift): "it is
 *   sufficient to only recompute the multipole moments of tree-cells that have updated child particles" (L266) -- here of
 *   all cells, in one launch; the tight boxes follow the particles, so the cell size l grows as L266 describes.  Needs a
 *   topology from an earlier bh_tree_build on this particle set; afterwards bh_compute_forces(_active) may be called.
 * bh_compute_forces_active: S7 + S8 for the groups that hold at least one ACTIVE particle only ("the tree-traverse time is
 *   reduced by a factor N_groups / N_active", L264).  d_active: uint8[n] DEVICE pointer in the current (key-sorted)
 *   particle order, non-zero = active; borrowed for the duration of the enqueued work.  Particles of other groups keep
 *   their acc_pot; group_npc / group_npp of other groups read 0; sum_pc / sum_pp count the walked groups only. */
int bh_refresh_moments(bh_ctx* ctx, void* stream);
int bh_compute_forces_active(bh_ctx* ctx, float theta, float eps, const uint8_t* d_active, void* stream);

/* bh_refresh_moments restricted to "the multipole moments of tree-cells that have updated child particles" (L266): only
 * the leaves that hold an active particle and their ancestors are recomputed (d_active as above); every other cell keeps
 * the moments, box and records it holds, which are still exact if only active particles moved. */
int bh_refresh_moments_active(bh_ctx* ctx, const uint8_t* d_active, void* stream);

/* The block time-step scheme itself (L45, L101 "time-step calculation ... on the GPU", L105, L264-266; reading A29).
 * Every particle i holds (x_i, v_i, a_i) at its own time t_i = tick_i * dt_max / 2^max_rung and steps by
 * dt_i = dt_max / 2^rung_i, rung_i = the smallest r in [0, max_rung] with dt_max / 2^r <= eta * sqrt(len_scale / |a_i|)
 * that keeps t_i a multiple of dt_i.
 * bh_block_init: needs valid forces (bh_compute_forces); all particles at tick 0, rungs from the criterion.
 * bh_block_step: one system step to t_next = min_i (t_i + dt_i).  The ACTIVE particles (t_i + dt_i = t_next) are predicted
 *   (x += v dt + a dt^2 / 2), the moments of the cells above them refreshed on the existing cells (rebuild = 0; L266) or the
 *   tree rebuilt from the current positions (rebuild != 0: S0-S6, the block state follows the sort), the groups that hold
 *   them walked (L264), their velocities corrected (v += (a_old + a_new) dt / 2) and their next step chosen.  Inactive
 *   particles are not touched.  Only enqueues work.
 * bh_block_state: synchronises and reports (any pointer may be NULL; host or device destinations, key-sorted order):
 *   tick, rung, the active flags of the last step, the held accelerations (float[n][4]).  interactions_now /
 *   interactions_first = the list lengths of the groups walked in the last step, now and when each group was first walked
 *   on the current cells: their ratio is the decline L266 speaks of ("the tree-cell size increases, which causes more
 *   cells to be opened"); the caller rebuilds when it has grown too far.
 * Time is counted in 32-bit ticks of dt_max / 2^max_rung: a run can cover 2^(32 - max_rung) dt_max (4096 dt_max at max_rung = 20).
 *   When the system time comes within two dt_max of that end, the deferred status (bh_sync_status) of the step becomes
 *   BH_ERR_STATE; that step and the next are still exact.  Start over with bh_block_init (ticks restart at 0).
 * acc_pot (bh_get_particles) after a block step: the new acceleration for the active particles; for the others either the one
 *   held by the scheme (after a step with rebuild != 0) or a newer by-product of a walk of their group.  The scheme's own
 *   accelerations are acc_held of bh_block_state. */
typedef struct bh_block_config {
    float len_scale;    /* length in the criterion (e.g. the softening eps), > 0 */
    float eta;          /* accuracy parameter, > 0 */
    float dt_max;       /* longest step, > 0 */
    int32_t max_rung;   /* shortest step = dt_max / 2^max_rung; 0..20 */
} bh_block_config;
typedef struct bh_block_stats {
    int64_t steps;                 /* block steps since bh_block_init */
    int64_t steps_since_rebuild;
    int64_t now_tick;              /* system time in ticks of dt_max / 2^max_rung */
    int64_t n_active;              /* particles moved by the last step */
    int64_t interactions_now;      /* sum over the groups walked in the last step of (n_pc + n_pp) */
    int64_t interactions_first;    /* the same groups when each was first walked on the current cells */
} bh_block_stats;
int bh_block_init(bh_ctx* ctx, const bh_block_config* cfg, void* stream);
int bh_block_step(bh_ctx* ctx, float theta, float eps, int rebuild, void* stream);
int bh_block_state(bh_ctx* ctx, bh_block_stats* out, uint32_t* tick, uint8_t* rung, uint8_t* active, float* acc_held, void* stream);

/* Which multipole acceptance criterion S7 uses from the next bh_compute_forces on (the tree need not be rebuilt).
 *   BH_MAC_EQ1 (default): Eq.1 (L125): d > l / theta + delta, d = distance between the group's box and the cell's centre of
 *     mass, l = longest side of the cell's tight box, delta = |centre of mass - box centre|.
 *   BH_MAC_MIN_DISTANCE: the minimum-distance MAC the paper also implemented (L129, [31]; A28): d > l / theta with
 *     d = distance between the group's box and the cell's tight BOX.  Opens more cells: smaller error, more interactions. */
enum { BH_MAC_EQ1 = 0, BH_MAC_MIN_DISTANCE = 1 };
int bh_set_mac(bh_ctx* ctx, int mac);

/* S9 around S0-S8 (L105): v += a dt/2; x += v dt; tree_build; compute_forces; v += a dt/2.  Needs valid forces. */
int bh_leapfrog_step(bh_ctx* ctx, float theta, float eps, float dt, void* stream);

/* The same step as ONE graph launch.  bh_step_graph_build captures bh_leapfrog_step(theta, eps, dt) on `stream` into CUDA
 * graphs owned by the ctx (nothing runs; the particle arrays ping-pong between two buffer sets, so the step is captured once
 * for either parity) and bh_step_graph_launch replays the one that matches the current state: the result is that of
 * bh_leapfrog_step bit for bit, without the per-kernel launch gaps (~12 launches per step).  Needs valid forces, like
 * bh_leapfrog_step.  The graphs stay valid until bh_set_particles with another n, bh_set_mac or bh_destroy; the list-walk
 * geometry (waves) is the one chosen at capture.  Stage timing (bh_set_stage_timing) enabled at capture time is recorded
 * by the replays as well.  Returns BH_ERR_STATE without forces or without a captured step. */
int bh_step_graph_build(bh_ctx* ctx, float theta, float eps, float dt, void* stream);
int bh_step_graph_launch(bh_ctx* ctx, void* stream);

/* S9 on its own (L105), the kick-drift form of the same leapfrog: v += a * dt_kick; x += v * dt_drift, with the
 * accelerations of the last bh_compute_forces.  Invalidates tree and forces (the particles moved) -- unless dt_drift is
 * exactly 0: a pure kick leaves positions, tree and forces as they are (x = fmaf(v, 0, x) = x). */
int bh_kick_drift(bh_ctx* ctx, float dt_kick, float dt_drift, void* stream);

/* Synchronise `stream`, then report the deferred device status and the counters.  Returns the deferred status. */
int bh_sync_status(bh_ctx* ctx, void* stream, bh_stats* out);

/* Fill `out` with device pointers to the canonical tree arrays (see bh_tree_view). */
int bh_export_tree(bh_ctx* ctx, bh_tree_view* out, void* stream);

/* Per-stage device times of the last bh_tree_build + bh_compute_forces, in ms, when enabled (adds event records; a step
 * captured by bh_step_graph_build while timing is enabled records them on every replay).  Order: bbox, keys, sort,
 * reorder, cells, groups, moments, record, walk, lists, eval.  The stages are timed in the groups they are launched in:
 * with the one-launch front end (front_mode 0, n <= 1.2 M) "sort" is the whole of S0-S3 (k_front) and bbox, keys, reorder
 * read ~0; "cells" = k_bounds + k_scan_rows, "groups" = k_emit (cells and groups are emitted together); "moments" = S6
 * including the fp32 walk records when theta is known at build time ("record" then reads ~0; otherwise it is
 * k_cell_record); walk = S7 + S8 (list walk, evaluation, fallback kernel), lists = k_walk_lists alone, eval =
 * k_walk_eval alone; the last two are 0 when the walk ran as a pipeline of several waves (the kernels overlap: see
 * bh_get_walk_timeline).  Synchronises. */
int bh_set_stage_timing(bh_ctx* ctx, int enable);
int bh_get_stage_ms(bh_ctx* ctx, float ms[11]);

/* Device timeline of the last bh_compute_forces (profiling aid; synchronises `stream`).  The walk runs as a pipeline
 * over waves of groups (S7 list walk of wave w + 1 beside the S8 evaluation of wave w); for wave w,
 * ns[4w .. 4w+3] = %globaltimer nanoseconds of {first list block start, last list block end, first evaluation block
 * start, last evaluation block end}.  Returns the number of waves written (<= capacity_waves), or a negative status. */
int bh_get_walk_timeline(bh_ctx* ctx, void* stream, int64_t* ns, int capacity_waves);

/* The accuracy reference of PAPER.md:196-200 (Eq.2: |a_tree - a_direct| / |a_direct|): softened O(N^2) direct summation
 * in binary64 from the fp32 inputs, on the GPU (the paper uses a double-precision GPU direct code for the same purpose).
 * d_pos_mass: float[n][4] DEVICE pointer (x, y, z, m); targets are particles [t0, t1); d_acc_pot: double[n][4] DEVICE
 * pointer, rows t0..t1-1 receive (ax, ay, az, phi), other rows are not touched.  phi_i = -sum_{j != i} m_j / rho_ij,
 * a_i = sum_{j != i} m_j (x_j - x_i) / rho_ij^3, rho^2 = |x_j - x_i|^2 + eps^2.  Needs no ctx; only enqueues work on
 * `stream`; both pointers are borrowed.  Not on the per-step path.  Returns BH_OK, BH_ERR_INVALID_ARG or BH_ERR_CUDA. */
int bh_direct_forces(const float* d_pos_mass, int64_t n, float eps, int64_t t0, int64_t t1, double* d_acc_pot, void* stream);

/* S0 on its own, WITHOUT a workspace and without any allocation: the domain box of n particles (per-axis minimum and
 * maximum, exact), the cube side 2^domain_exp that bh_tree_build would use for them (the smallest power of two strictly above
 * the largest extent, Appendix B "the domain"; O1) and the input check of S0 (finite positions, finite
 * mass > 0; A27).  The result is bit for bit what bh_tree_build + bh_sync_status report in bh_stats.lo / hi /
 * domain_exp for the same particles.
 *
 * For callers that cannot allocate device memory and so cannot create a bh_ctx (which needs a workspace): code living inside
 * an application whose allocator already owns the whole GPU, processes held to a fixed device-memory budget where a cudaMalloc
 * mid-run can fail, and time-step loops that must not call cudaMalloc / cudaFree because those stall every stream of the
 * device.  This call makes no cudaMalloc, cudaFree or other allocating call.  Its intermediates (one partial box per 4096
 * particles and a counter) sit in a 256 KiB array that is part of the library image, resident on every GPU that runs this
 * library's kernels until the process ends; its fixed size is the reason for the limit:
 *     n <= BH_DOMAIN_STATIC_MAX_N (2^25 = 33 554 432 particles; also returned by bh_domain_box_static_max_n).
 * A larger n is refused with BH_ERR_TOO_LARGE before anything is enqueued -- split the input and merge the boxes, or use a ctx.
 *
 * d_pos_mass: float[n][4] DEVICE pointer (x, y, z, m), borrowed.  d_out: DEVICE pointer to one bh_domain_box (32 bytes) on the
 * same device, written by the kernel: the caller copies it to the host (or reads it from a kernel of its own) after the work
 * on `stream` has completed.  out->status is BH_OK or BH_ERR_NONFINITE (then lo / hi are the box of the finite coordinates
 * and domain_exp is still a usable exponent).  Only enqueues work on `stream` (one 256-byte memset + one kernel); no host
 * synchronisation.  The device is taken from the pointers; the caller's current device is restored on return.
 *
 * First call on each device: looks up the device address of the built-in array (cudaGetSymbolAddress, which may make the
 * driver load the library's kernels on that device).  Make this first call during set-up, outside any stream capture.
 *
 * Sharing: every call on a device uses the same array, which still holds the previous call's contents; the call clears the
 * one word that must start at zero itself.  Calls whose GPU work may OVERLAP on one device (two streams, two host threads)
 * race on that array and return garbage: issue them on one stream, or order them with events.  Calls on different devices
 * are independent.  Thread-safe on the host side.
 * Returns BH_OK, BH_ERR_INVALID_ARG (null / host pointers, pointers on different devices, n < 1), BH_ERR_TOO_LARGE, BH_ERR_CUDA. */
#define BH_DOMAIN_STATIC_MAX_N 33554432
typedef struct bh_domain_box {
    float   lo[3];        /* per-axis minimum = corner of the key grid */
    float   hi[3];        /* per-axis maximum */
    int32_t domain_exp;   /* cube side = 2^domain_exp */
    int32_t status;       /* BH_OK or BH_ERR_NONFINITE */
} bh_domain_box;
int bh_domain_box_static(const float* d_pos_mass, int64_t n, bh_domain_box* d_out, void* stream);
int64_t bh_domain_box_static_max_n(void);

/* FP32 issue-rate probes ("a register-resident FFMA-chain probe"); a measurement aid, not on the
 * per-step path.  Runs one kernel on every SM of the current device (512 threads per block: four warps per scheduler,
 * the occupancy of the evaluation kernel) on the legacy default stream, synchronises, and returns the achieved rate.
 *   kind 0: scalar fma, three distinct 32-bit register operands        1: packed fma.rn.f32x2, three distinct 64-bit operands
 *   kind 2: packed, one operand shared by consecutive instructions     3: packed, a 32-bit scalar broadcast to both halves
 *   kind 4: the particle-cell body of S8 on entries in shared memory   5: the particle-particle body
 * *tflops: 2 flop per multiply-add lane (kinds 0-3); kinds 4, 5 in the 20 / 64 flop convention of DESIGN.md (A25), with
 * the flops the code really executes (56 per particle-cell interaction) in *tflops_executed (may be NULL).
 * d_scratch: device memory, at least 4 * (SMs * 512 + 4096) bytes, borrowed.  No ctx needed. */
int bh_probe_fp32(int kind, void* d_scratch, size_t scratch_bytes, double* tflops, double* tflops_executed);

int bh_last_cuda_error(const bh_ctx* ctx);
const char* bh_status_string(int status);

#ifdef __cplusplus
}
#endif
#endif /* BH_B200_H */
