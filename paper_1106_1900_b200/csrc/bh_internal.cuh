// bh_internal.cuh -- shared declarations of the CUDA library (not part of the C ABI).
// Product code: never includes or links anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/bh.h"

namespace bh {

constexpr int kMaxLevel = 20;
constexpr int kKeyBits = 20;           // per axis
constexpr int kLevels = kMaxLevel + 1; // levels 0..20
constexpr uint32_t kNone = 0xFFFFFFFFu;
constexpr uint32_t kSkip = 0xFFFFFFFEu;   // g_pcoff of a group that is not active in this walk (>= kSkip: nothing to evaluate)

// ---- sort geometry (S2)
constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kSortPasses = 8;                 // 8 x 8 bits covers the 60-bit key
constexpr int kSortThreads = 512;    // 512 x 8 keys: 64 registers per thread, 48 warps per SM (256 x 16: 128 registers, 16 warps)
constexpr int kSortItemsPerThread = 4096 / kSortThreads;
constexpr int kSortTile = kSortThreads * kSortItemsPerThread;   // 4096 keys per block

// ---- tree geometry (S4, S5): one boundary per thread
constexpr int kTreeTile = 1024;
constexpr int kHaloMax = 64;           // nleaf, ncrit <= 64
constexpr int kTreeRows = kLevels + 1; // per-tile counts of starts: cells of level 0..20, then groups
constexpr int kFrontTileCap = 1024;    // most sort tiles k_front can ever have resident (bounds its digit-count matrix)
constexpr int kFrontGroupCap = kFrontTileCap / 16;   // groups of 16 tiles
constexpr int kMomBlockCap = 160;      // most blocks of k_moments (one per SM; bounds the shared memory of k_moments_span)

// ---- walk (S7, S8): waves of groups whose interaction lists share the list buffer
constexpr int kMaxWaves = 255;

// Device-resident scalars (one struct, copied to the host by bh_sync_status).
struct DevScalars {
    uint32_t bb_min[3];      // order-preserving encodings of the per-axis minima / maxima (S0)
    uint32_t bb_max[3];
    int32_t status;          // deferred bh_status
    int32_t dom_e;           // cube side = 2^dom_e
    float lo[3];
    float hi[3];
    uint32_t level_offset[kLevels + 1];
    uint32_t n_cells;
    uint32_t n_groups;
    uint32_t n_levels;
    uint32_t walk_next;      // dynamic group counter of the walk
    unsigned long long sum_pc;
    unsigned long long sum_pp;
    unsigned long long sum_mac;
    // block time-steps (blockstep.cu)
    uint32_t tick_next[2];   // next system time, per step parity (the idle slot is reset to ~0)
    uint32_t n_active;       // particles moved by the last block step
    unsigned long long deg_now, deg_base;   // interactions of the groups walked in the last block step / when each was first walked on this tree
    uint32_t sort_skip;      // stage_sort: trailing (low) digits this build's first sort leaves to the fix-up (0: all 8 passes); set by k_reset_build
    uint32_t sort_redo;      // stage_sort: the fix-up met a run it could not finish: the full sort follows
    uint32_t sort_retries;   // full re-sorts since bh_create: the short sort of k_front / stage_sort met a run of equal leading key bits it could not finish
};

// Walk control block (device): wave boundaries in groups, work counters, the groups deferred to the fused kernel.
struct WalkCtl {
    uint32_t wave_g[kMaxWaves + 1];
    uint32_t list_next[kMaxWaves + 1];
    uint32_t eval_next[kMaxWaves + 1];
    uint32_t arena_next[kMaxWaves + 1];   // list-region cursor of each wave (chunks handed to walking warps)
    uint32_t n_deferred;
    uint32_t fused_next;
    // %globaltimer (ns) of the first block start / last block end of every list walk [0] and evaluation [1] (bh_get_walk_timeline)
    unsigned long long t_start[2][kMaxWaves + 1];
    unsigned long long t_end[2][kMaxWaves + 1];
};

__device__ __forceinline__ uint32_t ld_relaxed_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// ---- grid barriers of the cooperative kernels (front.cu, keys_sort.cu): counters in the workspace, bounded spins
constexpr uint32_t kBarSpinLimit = 1u << 24;
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// All blocks of the (cooperative) grid meet here.  bar[0] counts the arrivals of every barrier but the last (barrier k is
// passed at k x blocks arrivals); the last barrier of the launch counts on bar[1], which only ever grows (`b0` = its value
// when this block started, read before any block can arrive there), so that block 0 can put bar[0] back to zero for the
// next launch once everybody is known to have left it.
__device__ __forceinline__ void grid_barrier(uint32_t* bar, uint32_t target, DevScalars* sc) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();                                   // release what this block wrote
        atomicAdd(bar, 1u);
        uint32_t spins = 0;
        while (ld_acquire_u32(bar) < target)
            if (++spins > kBarSpinLimit) { atomicMin(&sc->status, (int)BH_ERR_CUDA); break; }   // never hang the device
        __threadfence();
    }
    __syncthreads();
}
// `closing`: the counter of the closing barriers (bar[1]), passed at `arrivals` arrivals since this block started; `used`: the
// counter of the barriers before it, which block 0 puts back to zero.
__device__ __forceinline__ void grid_barrier_last(uint32_t* closing, uint32_t b0, uint32_t arrivals, uint32_t* used, DevScalars* sc) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(closing, 1u);
        uint32_t spins = 0;
        while (ld_acquire_u32(closing) - b0 < arrivals)
            if (++spins > kBarSpinLimit) { atomicMin(&sc->status, (int)BH_ERR_CUDA); break; }
        if (blockIdx.x == 0) atomicExch(used, 0u);
        __threadfence();
    }
    __syncthreads();
}

typedef float4* float4_ptr;

// Pointers into the caller's workspace.
struct Ws {
    DevScalars* sc;
    float4* pos[2];
    float4* vel[2];
    uint32_t* idb[2];
    float4* acc;
    uint64_t* key[2];
    uint32_t* val[2];
    uint8_t* fl;          // [n+1] first level at which boundary i starts a new run (0..21)
    uint8_t* dep;         // [n]   level of the leaf holding particle i
    uint8_t* gl;          // [n]   level of the cell of the group that starts at particle i (0xFF: no group starts here)
    uint8_t* gflag;       // [n]   per GROUP: 1 if the group takes part in an active-subset walk (bh_compute_forces_active)
    uint32_t* g_begin;    // [n+1]
    uint32_t* g_cell;     // [n]
    uint32_t* g_npc;      // [n]
    uint32_t* g_npp;      // [n]
    uint32_t* sort_ghist;  // [kSortPasses][kRadix] keys per digit value, all passes (counted by k_keys)
    uint32_t* sort_ticket; // [2][kSortPasses] tile tickets                       (contiguous with sort_ghist and sort_status: one
    uint32_t* sort_status; // [2][kSortPasses][sortTiles][kRadix] look-back words  memset); [1]: the full re-sort after a failed short sort
    uint32_t* tile_cnt;   // [kTreeRows][treeTiles] starts per tile; after k_bounds: exclusive scan of every row over the tiles
    uint32_t* row_total;  // [kTreeRows] cells per level, groups
    uint32_t* mom_span;   // [kLevels][momentBlocks] cell of each level that straddles the end of a block's particle range (kNone: none)
    float* front_part;    // [sortTiles][8] per-tile box of k_front
    uint32_t* front_matrix; // [frontTiles][kRadix] per-tile digit counts of the current pass
    uint32_t* front_gsum;   // [kSortPasses][kFrontGroupCap][kRadix] digit counts per pass and group of 16 tiles (zero between launches)
    uint32_t* front_ctl;    // control words that are zero between launches: front_bar[5], then [5..6] the grid barrier of k_sort_passes
    uint32_t* front_bar;    // [5] grid barriers of k_front and its retry flag (front.cu: FrontArgs::bar)
    uint8_t* c_dirty;     // [max_cells] partial refresh (block time-steps): the cell has an active particle below it
    uint4* c_topo;        // [max_cells] (first particle, end particle, first child, end child); children (0, 0) for a leaf
    uint32_t* c_parent;
    double* mom64;        // [max_cells][10]
    float* box;           // [max_cells][6]
    float4* trec;         // [max_cells] walk record: (com, r2open)
    uint2* tlink;         // [max_cells] walk record: (first child | first particle, count | leaf << 31)
    float4* erec;         // [max_cells][3] evaluation record: (com, M) (Qm_xx, Qm_yy, Qm_zz, Qm_xy) (Qm_xz, Qm_yz, -T/2, -3T/2), Qm = -3 Q
    WalkCtl* ctl;
    // block time-steps: held accelerations, time of the last update (ticks of dt_max / 2^R), rung, active flags; [2]: ping-pong for a rebuild
    float4* accb[2];
    uint32_t* tick[2];
    uint8_t* rung[2];
    uint8_t* bactive[2];
    uint32_t* g_base;     // [n] per group: interactions when it was first walked on this tree (0: not yet)
    uint32_t* lists;      // [list_entries] interaction lists: cell indices / particle indices
    uint32_t* g_pcoff;    // [n] first entry of the group's cell list (kNone: deferred to the fused kernel)
    uint32_t* g_ppoff;    // [n] first entry of the group's particle list
    uint32_t* g_lpp;      // [n] length of the particle list (g_npp minus the group's own particles)
    uint32_t* deferred;   // [n] groups whose lists did not fit
    // export (canonical arrays of bh_tree_view)
    int32_t* e_level;
    uint64_t* e_prefix;
    uint32_t* e_pbegin;
    uint32_t* e_pcount;
    int32_t* e_cbegin;
    int32_t* e_nchild;
    int32_t* e_parent;
    float* e_mom32;
    float* e_r2open;
};

}  // namespace bh

struct bh_ctx {
    int device;
    int sm_count;
    int64_t n_max;
    int64_t n;
    int64_t max_cells;
    int32_t nleaf, ncrit;
    int cur;               // which of pos[2]/vel[2]/idb[2] holds the live state
    int sorted;            // which of key[2]/val[2] holds the sorted keys / perm
    bool have_particles, have_topology, have_tree, have_forces;   // topology: cells + groups; tree: topology + current moments
    bool bound;            // bh_bind_particles: ws.pos[0] / vel[0] / idb[0] / acc are the CALLER's arrays (home_*: the workspace's own)
    bh::float4_ptr home_pos0, home_vel0, home_acc;
    uint32_t* home_id0;
    bool acc_in_order;     // ws.acc is in the order of the current particle arrays (false between a re-sort and the next full forces)
    const uint8_t* active;   // per-particle flags of bh_compute_forces_active during that call (nullptr: every group)
    int64_t launches;
    int last_cuda;
    float theta_last;
    int64_t list_entries;
    int walk_mode;
    int walk_waves;
    int walk_share;        // 1: the groups of a block of eight share the common part of their walks (walk_lists.cu)
    int mac_kind;          // 0: Eq.1, 1: minimum distance (bh_set_mac)
    bh::Ws ws;
    int64_t sort_tiles, tree_tiles;
    int sort_grid;             // resident blocks of k_sort_passes (cooperative launch)
    int64_t front_max_tiles;   // sort tiles that are resident at once in a cooperative launch of k_front (0: not available)
    bool front_enabled;        // bh_config.front_mode != 1
    bool front_full;           // bh_config.front_mode == 2: k_front always sorts with all 8 passes
    // block time-steps
    bool block_on;             // bh_block_init done on this particle set
    int bcur;                  // which of accb / tick / rung / bactive is live
    float blk_len, blk_eta, blk_dt_max;
    int blk_R;
    int64_t blk_steps;         // block steps since bh_block_init (parity of tick_next)
    int64_t blk_since_rebuild; // block steps on the current cells
    bool rec_valid;            // trec / tlink / erec hold the current tree for (rec_theta, rec_mac)
    float rec_theta;
    int rec_mac;
    bool timing;
    bool capturing;        // inside bh_step_graph_build
    cudaGraphExec_t step_graph[2];   // bh_leapfrog_step captured for either parity of the particle ping-pong buffers (api.cu)
    bool step_graph_valid;
    float graph_theta, graph_eps, graph_dt;
    int64_t graph_launches;          // kernels in one captured step
    bool graph_split_timed;          // walk_split_timed as the captured step leaves it
    cudaEvent_t ev[13];     // [0..10] stage boundaries; [11], [12]: after the list walk / the evaluation of a one-wave walk
    bool copies_pending;    // bh_set_particles left copies on s_lists; ev_join marks their end (api.cu: join_copies)
    bool walk_split_timed;  // the last walk was one wave: ev[11], ev[12] are valid
    // walk pipeline (walk.cu): the list walk of wave w + 1 runs beside the evaluation of wave w on internal streams
    cudaStream_t s_lists, s_eval2;
    cudaEvent_t ev_fork, ev_join, ev_lists[bh::kMaxWaves + 1], ev_eval[bh::kMaxWaves + 1];
};

namespace bh {

#define BH_CUDA(ctx, call)                                   \
    do {                                                     \
        cudaError_t _e = (call);                             \
        if (_e != cudaSuccess) {                             \
            (ctx)->last_cuda = (int)_e;                      \
            return BH_ERR_CUDA;                              \
        }                                                    \
    } while (0)

#define BH_LAUNCH(ctx, kernel, grid, block, smem, stream, ...)              \
    do {                                                                    \
        kernel<<<(grid), (block), (smem), (stream)>>>(__VA_ARGS__);         \
        (ctx)->launches += 1;                                               \
        cudaError_t _e = cudaPeekAtLastError();                             \
        if (_e != cudaSuccess) {                                            \
            (ctx)->last_cuda = (int)_e;                                     \
            return BH_ERR_CUDA;                                             \
        }                                                                   \
    } while (0)

static inline int64_t div_up(int64_t a, int64_t b) { return (a + b - 1) / b; }
// words of sort bookkeeping (digit histograms, tickets, look-back status words for the first sort and for a re-sort)
static inline size_t sort_words(int64_t tiles) { return (size_t)kSortPasses * kRadix + 2 * (size_t)kSortPasses + 2 * (size_t)kSortPasses * kRadix * (size_t)tiles; }

// Stage-boundary event k on stream s.  While the step is being captured into a graph (bh_step_graph_build) the record
// becomes an external event node, so the stage times of a replayed graph can be read like those of plain launches.
static inline void stage_mark(bh_ctx* c, int k, cudaStream_t s) {
    if (c->capturing) cudaEventRecordWithFlags(c->ev[k], s, cudaEventRecordExternal);
    else cudaEventRecord(c->ev[k], s);
}

// stage entry points (each only enqueues kernels on `s`)
int front_init(bh_ctx* c);
int moments_init(bh_ctx* c);
bool front_fits(const bh_ctx* c);
int stage_front(bh_ctx* c, bool fuse_reorder, cudaStream_t s);   // S0-S2 (+ S3) in one cooperative launch (front.cu)
int stage_bbox_keys(bh_ctx* c, cudaStream_t s);       // S0, S1
int stage_sort(bh_ctx* c, cudaStream_t s);            // S2
int stage_reorder(bh_ctx* c, cudaStream_t s);         // S3
int stage_cells(bh_ctx* c, cudaStream_t s);           // S4 + S5
int stage_moments(bh_ctx* c, float theta, const uint8_t* d_active, cudaStream_t s);   // S6 (+ the fp32 records when theta > 0); d_active: only the cells above an active particle
int stage_cell_record(bh_ctx* c, float theta, cudaStream_t s);          // S6: fp32 walk record + r2open(theta) alone
int stage_walk(bh_ctx* c, float theta, float eps, cudaStream_t s);   // S7, S8
int stage_group_active(bh_ctx* c, const uint8_t* d_active, cudaStream_t s);   // groups with an active particle -> ws.gflag[g]
int walk_init(bh_ctx* c);
int sort_init(bh_ctx* c);
int walk_eval_init(bh_ctx* c);
int walk_lists_init(bh_ctx* c);
int walk_destroy(bh_ctx* c);
struct WalkListOut {       // what k_walk_lists writes
    DevScalars* sc;
    WalkCtl* ctl;
    // block time-steps: held accelerations, time of the last update (ticks of dt_max / 2^R), rung, active flags; [2]: ping-pong for a rebuild
    float4* accb[2];
    uint32_t* tick[2];
    uint8_t* rung[2];
    uint8_t* bactive[2];
    uint32_t* g_base;     // [n] per group: interactions when it was first walked on this tree (0: not yet)
    uint32_t *g_pcoff, *g_ppoff, *g_lpp, *g_npc, *g_npp, *deferred;
};
WalkListOut walk_list_out(bh_ctx* c);
int stage_walk_prepare(bh_ctx* c, int nwaves, uint32_t wave_particles, cudaStream_t s);
int stage_walk_lists(bh_ctx* c, int wave, int grid, uint32_t region_base, uint32_t region_entries, cudaStream_t s);   // S7
int stage_walk_eval(bh_ctx* c, int wave, float eps, int blocks_per_sm, bool by_class, cudaStream_t s);                           // S8
int stage_kick_drift(bh_ctx* c, float h, float dt, cudaStream_t s);  // S9
int stage_kick(bh_ctx* c, float h, cudaStream_t s);                  // S9
int stage_block_init(bh_ctx* c, cudaStream_t s);
int stage_block_predict(bh_ctx* c, cudaStream_t s);                   // next time, active set, predictor
int stage_block_permute(bh_ctx* c, cudaStream_t s);                   // after a rebuild: the block state follows the sort
int stage_block_correct(bh_ctx* c, cudaStream_t s);                   // corrector, new rungs, degradation sums
int stage_export(bh_ctx* c, cudaStream_t s);
int stage_iota(bh_ctx* c, uint32_t* dst, int64_t n, cudaStream_t s);

}  // namespace bh
