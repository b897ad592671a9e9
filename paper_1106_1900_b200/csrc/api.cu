// api.cu -- the C ABI of include/bh.h: argument checking, workspace carving, stage sequencing.
// No kernel arithmetic lives here; every step of the path is a kernel in the sibling translation units.
#include <cmath>
#include <cstring>
#include <new>

#include "bh_internal.cuh"

namespace bh {

struct Carver {
    unsigned char* base;
    size_t off;
    template <typename T>
    T* take(size_t count) {
        off = (off + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};

struct Geometry {
    int64_t n_max, max_cells, sort_tiles, tree_tiles, list_entries;
    int32_t nleaf, ncrit, walk_mode, walk_waves, front_mode, walk_private;
};

static bool make_geometry(int64_t n_max, const bh_config* cfg, Geometry* g) {
    if (n_max < 1 || n_max >= (int64_t)1 << 30) return false;   // counts must fit 30 bits (sort look-back words)
    g->n_max = n_max;
    g->nleaf = (cfg && cfg->nleaf) ? cfg->nleaf : 16;
    g->ncrit = (cfg && cfg->ncrit) ? cfg->ncrit : 64;
    if (g->nleaf < 1 || g->nleaf > kHaloMax || g->ncrit < 1 || g->ncrit > 64) return false;
    const int64_t bound = n_max + kMaxLevel * (n_max / (g->nleaf + 1)) + 1;
    g->max_cells = (cfg && cfg->max_cells > 0) ? cfg->max_cells : bound;
    if (g->max_cells > bound) g->max_cells = bound;
    if (g->max_cells < 1 || g->max_cells > ((int64_t)1 << 31) - 2) return false;
    g->list_entries = (cfg && cfg->list_entries > 0) ? cfg->list_entries
                                                     : std::min<int64_t>(std::max<int64_t>(320 * n_max, (int64_t)1 << 22), (int64_t)1 << 30);
    if (g->list_entries > ((int64_t)1 << 31)) return false;
    g->walk_mode = cfg ? cfg->walk_mode : 0;
    if (g->walk_mode < 0 || g->walk_mode > 1) return false;
    g->walk_waves = cfg ? cfg->walk_waves : 0;
    if (g->walk_waves < 0 || g->walk_waves > kMaxWaves) return false;
    g->walk_private = cfg ? cfg->walk_private : 0;
    if (g->walk_private < 0 || g->walk_private > 1) return false;
    g->front_mode = cfg ? cfg->front_mode : 0;
    if (g->front_mode < 0 || g->front_mode > 2) return false;
    g->sort_tiles = div_up(n_max, kSortTile);
    g->tree_tiles = div_up(n_max + 1, kTreeTile);
    return true;
}

static size_t carve(const Geometry& g, unsigned char* base, Ws* w) {
    Carver c{base, 0};
    Ws tmp;
    Ws& o = w ? *w : tmp;
    const size_t n = (size_t)g.n_max, C = (size_t)g.max_cells;
    o.sc = c.take<DevScalars>(1);
    for (int k = 0; k < 2; ++k) { o.pos[k] = c.take<float4>(n); o.vel[k] = c.take<float4>(n); o.idb[k] = c.take<uint32_t>(n); }
    o.acc = c.take<float4>(n);
    for (int k = 0; k < 2; ++k) { o.key[k] = c.take<uint64_t>(n); o.val[k] = c.take<uint32_t>(n); }
    // control words that must be zero between launches (one memset in bh_create): kept together
    o.front_gsum = c.take<uint32_t>((size_t)kSortPasses * kFrontGroupCap * kRadix + 8);
    o.front_ctl = o.front_gsum ? o.front_gsum + (size_t)kSortPasses * kFrontGroupCap * kRadix : nullptr;
    o.front_bar = o.front_ctl;
    o.front_part = c.take<float>(8 * (size_t)kFrontTileCap);
    o.front_matrix = c.take<uint32_t>((size_t)kRadix * (size_t)kFrontTileCap);
    o.fl = c.take<uint8_t>(n + 8);      // (k_bounds stores four boundaries per word: padded)
    o.dep = c.take<uint8_t>(n + 8);
    o.gl = c.take<uint8_t>(n + 8);
    o.gflag = c.take<uint8_t>(n);
    o.g_begin = c.take<uint32_t>(n + 1);
    o.g_cell = c.take<uint32_t>(n);
    o.g_npc = c.take<uint32_t>(n);
    o.g_npp = c.take<uint32_t>(n);
    o.sort_ghist = c.take<uint32_t>(sort_words(g.sort_tiles));
    o.sort_ticket = o.sort_ghist ? o.sort_ghist + kSortPasses * kRadix : nullptr;
    o.sort_status = o.sort_ghist ? o.sort_ticket + 2 * kSortPasses : nullptr;
    o.tile_cnt = c.take<uint32_t>((size_t)kTreeRows * g.tree_tiles);
    o.row_total = c.take<uint32_t>(kTreeRows);
    o.mom_span = c.take<uint32_t>((size_t)kLevels * kMomBlockCap);
    o.c_topo = c.take<uint4>(C);
    o.c_dirty = c.take<uint8_t>(C);
    o.c_parent = c.take<uint32_t>(C);
    o.mom64 = c.take<double>(10 * C);
    o.box = c.take<float>(6 * C);
    o.trec = c.take<float4>(C);
    o.tlink = c.take<uint2>(C);
    o.erec = c.take<float4>(3 * C);
    o.ctl = c.take<WalkCtl>(1);
    for (int k = 0; k < 2; ++k) { o.accb[k] = c.take<float4>(n); o.tick[k] = c.take<uint32_t>(n); o.rung[k] = c.take<uint8_t>(n); o.bactive[k] = c.take<uint8_t>(n); }
    o.g_base = c.take<uint32_t>(n);
    o.lists = c.take<uint32_t>((size_t)g.list_entries);
    o.g_pcoff = c.take<uint32_t>(n);
    o.g_ppoff = c.take<uint32_t>(n);
    o.g_lpp = c.take<uint32_t>(n);
    o.deferred = c.take<uint32_t>(n);
    o.e_level = c.take<int32_t>(C);
    o.e_prefix = c.take<uint64_t>(C);
    o.e_pbegin = c.take<uint32_t>(C);
    o.e_pcount = c.take<uint32_t>(C);
    o.e_cbegin = c.take<int32_t>(C);
    o.e_nchild = c.take<int32_t>(C);
    o.e_parent = c.take<int32_t>(C);
    o.e_mom32 = c.take<float>(10 * C);
    o.e_r2open = c.take<float>(C);
    return (c.off + 255) & ~(size_t)255;
}

}  // namespace bh

using namespace bh;

static void drop_step_graph(bh_ctx* c) {
    for (int k = 0; k < 2; ++k)
        if (c->step_graph[k]) { cudaGraphExecDestroy(c->step_graph[k]); c->step_graph[k] = nullptr; }
    c->step_graph_valid = false;
}

// Make `s` wait for the side-stream half of the last bh_set_particles (velocities, ids, zeroed accelerations).
static int join_copies(bh_ctx* c, cudaStream_t s) {
    if (!c->copies_pending) return BH_OK;
    BH_CUDA(c, cudaStreamWaitEvent(s, c->ev_join, 0));
    c->copies_pending = false;
    return BH_OK;
}

extern "C" {

size_t bh_workspace_bytes(int64_t n_max, const bh_config* cfg) {
    Geometry g;
    if (!make_geometry(n_max, cfg, &g)) return 0;
    return carve(g, nullptr, nullptr);
}

int bh_create(bh_ctx** out, int64_t n_max, const bh_config* cfg, void* d_workspace, size_t bytes) {
    if (!out || !d_workspace) return BH_ERR_INVALID_ARG;
    *out = nullptr;
    Geometry g;
    if (!make_geometry(n_max, cfg, &g)) return BH_ERR_INVALID_ARG;
    if (((uintptr_t)d_workspace & 255) != 0) return BH_ERR_WORKSPACE;
    if (carve(g, nullptr, nullptr) > bytes) return BH_ERR_WORKSPACE;
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, d_workspace) != cudaSuccess || attr.type != cudaMemoryTypeDevice) {
        (void)cudaGetLastError();
        return BH_ERR_WORKSPACE;
    }
    bh_ctx* c = new (std::nothrow) bh_ctx();
    if (!c) return BH_ERR_INVALID_ARG;
    std::memset(c, 0, sizeof(*c));
    c->device = attr.device;
    c->n_max = n_max;
    c->max_cells = g.max_cells;
    c->nleaf = g.nleaf;
    c->ncrit = g.ncrit;
    c->list_entries = g.list_entries;
    c->walk_mode = g.walk_mode;
    c->walk_waves = g.walk_waves;
    c->sort_tiles = g.sort_tiles;
    c->tree_tiles = g.tree_tiles;
    c->front_enabled = g.front_mode != 1;
    c->front_full = g.front_mode == 2;
    c->walk_share = g.walk_private ? 0 : 1;
    carve(g, static_cast<unsigned char*>(d_workspace), &c->ws);
    c->home_pos0 = c->ws.pos[0]; c->home_vel0 = c->ws.vel[0]; c->home_id0 = c->ws.idb[0]; c->home_acc = c->ws.acc;
    int rc = BH_OK;
    do {
        if (cudaSetDevice(c->device) != cudaSuccess) { rc = BH_ERR_CUDA; break; }
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess) { rc = BH_ERR_CUDA; break; }
        c->sm_count = sms;
        if (cudaMemset(c->ws.sc, 0, sizeof(DevScalars)) != cudaSuccess) { rc = BH_ERR_CUDA; break; }   // status = BH_OK before the first build
        if (cudaMemset(c->ws.front_gsum, 0, sizeof(uint32_t) * ((size_t)kSortPasses * kFrontGroupCap * kRadix + 8)) != cudaSuccess) { rc = BH_ERR_CUDA; break; }
        if (front_init(c) != BH_OK || moments_init(c) != BH_OK) { rc = BH_ERR_CUDA; break; }
        if (walk_init(c) != BH_OK || sort_init(c) != BH_OK) { rc = BH_ERR_CUDA; break; }
        for (int k = 0; k < 13; ++k)
            if (cudaEventCreate(&c->ev[k]) != cudaSuccess) { rc = BH_ERR_CUDA; break; }
    } while (0);
    if (rc != BH_OK) { walk_destroy(c); delete c; return rc; }
    *out = c;
    return BH_OK;
}

int bh_destroy(bh_ctx* c) {
    if (!c) return BH_ERR_INVALID_ARG;
    cudaSetDevice(c->device);
    for (int k = 0; k < 13; ++k)
        if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    drop_step_graph(c);
    walk_destroy(c);
    delete c;
    return BH_OK;
}

int bh_set_particles(bh_ctx* c, int64_t n, const float* pos_mass, const float* vel, const uint32_t* id, void* stream) {
    if (!c || !pos_mass || n < 1 || n > c->n_max) return BH_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    if (c->step_graph_valid && n != c->n) drop_step_graph(c);   // captured for the old particle count
    if (c->bound) {                                             // back to the workspace's own arrays: the caller's are released
        c->ws.pos[0] = c->home_pos0; c->ws.vel[0] = c->home_vel0; c->ws.idb[0] = c->home_id0; c->ws.acc = c->home_acc;
        c->bound = false;
        drop_step_graph(c);                                     // (the captured kernels hold the caller's pointers)
    }
    c->n = n;
    c->cur = 0;
    c->have_particles = c->have_topology = c->have_tree = c->have_forces = false;
    c->block_on = false;
    c->acc_in_order = true;                                   // zeroed below, in the callers' order
    BH_CUDA(c, cudaMemcpyAsync(c->ws.pos[0], pos_mass, sizeof(float4) * (size_t)n, cudaMemcpyDefault, s));
    // S0-S2 need the positions only: velocities, ids and the zeroed accelerations arrive on an internal stream beside them
    // and are joined (event) before the first stage that touches them (S3) or any call that reads them.  Not under
    // stream capture: there everything stays on the caller's stream.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(s, &cap) != cudaSuccess) { (void)cudaGetLastError(); cap = cudaStreamCaptureStatusActive; }
    cudaStream_t side = s;
    if (cap == cudaStreamCaptureStatusNone) {
        side = c->s_lists;
        BH_CUDA(c, cudaEventRecord(c->ev_fork, s));                // after whatever used the old arrays on the caller's stream
        BH_CUDA(c, cudaStreamWaitEvent(side, c->ev_fork, 0));
    }
    if (vel) BH_CUDA(c, cudaMemcpyAsync(c->ws.vel[0], vel, sizeof(float4) * (size_t)n, cudaMemcpyDefault, side));
    else BH_CUDA(c, cudaMemsetAsync(c->ws.vel[0], 0, sizeof(float4) * (size_t)n, side));
    if (id) BH_CUDA(c, cudaMemcpyAsync(c->ws.idb[0], id, sizeof(uint32_t) * (size_t)n, cudaMemcpyDefault, side));
    else { int rc = stage_iota(c, c->ws.idb[0], n, side); if (rc != BH_OK) return rc; }
    BH_CUDA(c, cudaMemsetAsync(c->ws.acc, 0, sizeof(float4) * (size_t)n, side));
    if (side != s) {
        BH_CUDA(c, cudaEventRecord(c->ev_join, side));
        c->copies_pending = true;
    }
    c->have_particles = true;
    return BH_OK;
}

int bh_bind_particles(bh_ctx* c, int64_t n, float* d_pos_mass, float* d_vel, float* d_acc_pot, uint32_t* d_id) {
    if (!c || !d_pos_mass || !d_vel || !d_acc_pot || !d_id || n < 1 || n > c->n_max) return BH_ERR_INVALID_ARG;
    const void* ptrs[4] = {d_pos_mass, d_vel, d_acc_pot, d_id};
    for (int k = 0; k < 4; ++k) {
        cudaPointerAttributes a;
        if (cudaPointerGetAttributes(&a, ptrs[k]) != cudaSuccess || a.type != cudaMemoryTypeDevice || a.device != c->device) {
            (void)cudaGetLastError();
            return BH_ERR_INVALID_ARG;
        }
        if (reinterpret_cast<uintptr_t>(ptrs[k]) % (k < 3 ? 16u : 4u)) return BH_ERR_INVALID_ARG;   // float4 rows are moved as 16-byte words
    }
    drop_step_graph(c);                                         // captured kernels hold the previous pointers
    c->ws.pos[0] = reinterpret_cast<float4*>(d_pos_mass);
    c->ws.vel[0] = reinterpret_cast<float4*>(d_vel);
    c->ws.acc = reinterpret_cast<float4*>(d_acc_pot);
    c->ws.idb[0] = d_id;
    c->bound = true;
    c->n = n;
    c->cur = 0;
    c->have_particles = true;
    c->have_topology = c->have_tree = c->have_forces = false;
    c->block_on = false;
    c->acc_in_order = true;                                     // the caller's acc_pot belongs to the caller's particles, row by row
    return BH_OK;
}

int bh_land_particles(bh_ctx* c, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->have_particles) return BH_ERR_STATE;
    if (c->cur == 0) return BH_OK;                              // already there
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    { int rcj = join_copies(c, s); if (rcj != BH_OK) return rcj; }
    const size_t n = (size_t)c->n;
    BH_CUDA(c, cudaMemcpyAsync(c->ws.pos[0], c->ws.pos[1], sizeof(float4) * n, cudaMemcpyDeviceToDevice, s));
    BH_CUDA(c, cudaMemcpyAsync(c->ws.vel[0], c->ws.vel[1], sizeof(float4) * n, cudaMemcpyDeviceToDevice, s));
    BH_CUDA(c, cudaMemcpyAsync(c->ws.idb[0], c->ws.idb[1], sizeof(uint32_t) * n, cudaMemcpyDeviceToDevice, s));
    c->cur = 0;                                                 // tree, forces and block state stay valid: same particles, same order
    return BH_OK;
}

int bh_get_particles(bh_ctx* c, float* pos_mass, float* vel, float* acc_pot, uint32_t* id, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->have_particles) return BH_ERR_STATE;
    if (acc_pot && !c->acc_in_order) return BH_ERR_STATE;    // the particles were re-sorted (bh_tree_build) after the last forces
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    { int rcj = join_copies(c, s); if (rcj != BH_OK) return rcj; }
    const size_t n = (size_t)c->n;
    if (pos_mass) BH_CUDA(c, cudaMemcpyAsync(pos_mass, c->ws.pos[c->cur], sizeof(float4) * n, cudaMemcpyDefault, s));
    if (vel) BH_CUDA(c, cudaMemcpyAsync(vel, c->ws.vel[c->cur], sizeof(float4) * n, cudaMemcpyDefault, s));
    if (acc_pot) BH_CUDA(c, cudaMemcpyAsync(acc_pot, c->ws.acc, sizeof(float4) * n, cudaMemcpyDefault, s));
    if (id) BH_CUDA(c, cudaMemcpyAsync(id, c->ws.idb[c->cur], sizeof(uint32_t) * n, cudaMemcpyDefault, s));
    return BH_OK;
}

int bh_tree_build(bh_ctx* c, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->have_particles) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    c->have_topology = c->have_tree = c->have_forces = false;
    c->acc_in_order = false;                                  // S3 permutes pos / vel / id; acc_pot follows at the next forces
    int rc;
    if (c->timing) stage_mark(c, 0, s);
    if (front_fits(c)) {
        // S0-S3 in one cooperative launch (front.cu); reported as "sort".  While velocities / ids of bh_set_particles are
        // still arriving on the side stream, S3 stays a launch of its own behind the join.
        const bool fuse = !c->copies_pending;
        if (c->timing) { stage_mark(c, 1, s); stage_mark(c, 2, s); }
        if ((rc = stage_front(c, fuse, s)) != BH_OK) return rc;
        if (c->timing) stage_mark(c, 3, s);
        if (!fuse) {
            if ((rc = join_copies(c, s)) != BH_OK) return rc;
            if ((rc = stage_reorder(c, s)) != BH_OK) return rc;
        }
    } else {
        if ((rc = stage_bbox_keys(c, s)) != BH_OK) return rc;      // records ev[1] between bbox and keys
        if (c->timing) stage_mark(c, 2, s);
        if ((rc = stage_sort(c, s)) != BH_OK) return rc;
        if (c->timing) stage_mark(c, 3, s);
        if ((rc = join_copies(c, s)) != BH_OK) return rc;          // S3 is the first stage that reads velocities and ids
        if ((rc = stage_reorder(c, s)) != BH_OK) return rc;
    }
    if (c->timing) stage_mark(c, 4, s);
    if ((rc = stage_cells(c, s)) != BH_OK) return rc;             // S4 + S5; records ev[5] between k_bounds and k_emit
    if (c->timing) stage_mark(c, 6, s);
    if ((rc = stage_moments(c, c->theta_last, nullptr, s)) != BH_OK) return rc;   // S6; with the fp32 records when theta is known
    if (c->timing) stage_mark(c, 7, s);
    c->have_topology = c->have_tree = true;
    return BH_OK;
}

int bh_refresh_moments(bh_ctx* c, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->have_topology) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    c->have_forces = false;
    int rc = stage_moments(c, c->theta_last, nullptr, s);
    if (rc != BH_OK) return rc;
    c->have_tree = true;
    return BH_OK;
}

static int compute_forces_impl(bh_ctx* c, float theta, float eps, const uint8_t* d_active, void* stream) {
    if (!c || !(theta > 0.0f) || !std::isfinite(theta) || !(eps >= 0.0f) || !std::isfinite(eps)) return BH_ERR_INVALID_ARG;
    if (!c->have_tree) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    int rc;
    if (d_active && (rc = stage_group_active(c, d_active, s)) != BH_OK) return rc;
    c->active = d_active;
    rc = stage_walk(c, theta, eps, s);      // records ev[8] (before the records), ev[9], ev[10] (around S7 + S8)
    c->active = nullptr;
    if (rc != BH_OK) return rc;
    c->theta_last = theta;
    c->have_forces = true;
    // A full walk writes every row of acc_pot in the current order.  An active-subset walk writes the rows of the walked
    // groups only: the others keep what they held, which is in order only if nothing re-sorted the particles since.
    if (!d_active) c->acc_in_order = true;
    return BH_OK;
}

int bh_compute_forces(bh_ctx* c, float theta, float eps, void* stream) { return compute_forces_impl(c, theta, eps, nullptr, stream); }

int bh_compute_forces_active(bh_ctx* c, float theta, float eps, const uint8_t* d_active, void* stream) {
    if (!d_active) return BH_ERR_INVALID_ARG;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, d_active) != cudaSuccess || a.type != cudaMemoryTypeDevice) { (void)cudaGetLastError(); return BH_ERR_INVALID_ARG; }
    return compute_forces_impl(c, theta, eps, d_active, stream);
}

int bh_refresh_moments_active(bh_ctx* c, const uint8_t* d_active, void* stream) {
    if (!c || !d_active) return BH_ERR_INVALID_ARG;
    if (!c->have_topology) return BH_ERR_STATE;
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, d_active) != cudaSuccess || a.type != cudaMemoryTypeDevice) { (void)cudaGetLastError(); return BH_ERR_INVALID_ARG; }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    c->have_forces = false;
    int rc = stage_moments(c, c->theta_last, d_active, s);
    if (rc != BH_OK) return rc;
    c->have_tree = true;
    return BH_OK;
}

int bh_block_init(bh_ctx* c, const bh_block_config* cfg, void* stream) {
    if (!c || !cfg || !(cfg->len_scale > 0.0f) || !std::isfinite(cfg->len_scale) || !(cfg->eta > 0.0f) || !std::isfinite(cfg->eta) ||
        !(cfg->dt_max > 0.0f) || !std::isfinite(cfg->dt_max) || cfg->max_rung < 0 || cfg->max_rung > 20)
        return BH_ERR_INVALID_ARG;
    if (!c->have_forces) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    c->blk_len = cfg->len_scale; c->blk_eta = cfg->eta; c->blk_dt_max = cfg->dt_max; c->blk_R = cfg->max_rung;
    c->blk_steps = 0;
    c->blk_since_rebuild = 0;
    int rc = stage_block_init(c, s);
    if (rc != BH_OK) return rc;
    c->block_on = true;
    return BH_OK;
}

int bh_block_step(bh_ctx* c, float theta, float eps, int rebuild, void* stream) {
    if (!c || !(theta > 0.0f) || !std::isfinite(theta) || !(eps >= 0.0f) || !std::isfinite(eps)) return BH_ERR_INVALID_ARG;
    if (!c->block_on || !c->have_topology || c->copies_pending) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    int rc;
    c->theta_last = theta;
    if ((rc = stage_block_predict(c, s)) != BH_OK) return rc;
    const uint8_t* act;
    if (rebuild) {
        // S0-S6 on the current positions (the active ones predicted); the block state then follows the sort
        if ((rc = bh_tree_build(c, stream)) != BH_OK) return rc;
        if ((rc = stage_block_permute(c, s)) != BH_OK) return rc;
        // acc_pot did not follow the sort.  Put the held accelerations (which did) there, so that the rows the walk below does
        // not write belong to the right particles: for those, acc_pot = the acceleration of the particle's last own update.
        BH_CUDA(c, cudaMemcpyAsync(c->ws.acc, c->ws.accb[c->bcur], sizeof(float4) * (size_t)c->n, cudaMemcpyDeviceToDevice, s));
        c->acc_in_order = true;
        c->blk_since_rebuild = 0;
        act = c->ws.bactive[c->bcur];
    } else {
        act = c->ws.bactive[c->bcur];
        c->have_forces = false;
        if ((rc = stage_moments(c, theta, act, s)) != BH_OK) return rc;       // only the cells above an active particle (L266)
        c->have_tree = true;
    }
    if ((rc = bh_compute_forces_active(c, theta, eps, act, stream)) != BH_OK) return rc;
    if ((rc = stage_block_correct(c, s)) != BH_OK) return rc;
    c->blk_steps += 1;
    c->blk_since_rebuild += 1;
    return BH_OK;
}

int bh_block_state(bh_ctx* c, bh_block_stats* out, uint32_t* tick, uint8_t* rung, uint8_t* active, float* acc_held, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->block_on) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    const size_t n = (size_t)c->n;
    const int b = c->bcur;
    if (tick) BH_CUDA(c, cudaMemcpyAsync(tick, c->ws.tick[b], sizeof(uint32_t) * n, cudaMemcpyDefault, s));
    if (rung) BH_CUDA(c, cudaMemcpyAsync(rung, c->ws.rung[b], n, cudaMemcpyDefault, s));
    if (active) BH_CUDA(c, cudaMemcpyAsync(active, c->ws.bactive[b], n, cudaMemcpyDefault, s));
    if (acc_held) BH_CUDA(c, cudaMemcpyAsync(acc_held, c->ws.accb[b], sizeof(float4) * n, cudaMemcpyDefault, s));
    DevScalars h;
    BH_CUDA(c, cudaMemcpyAsync(&h, c->ws.sc, sizeof(h), cudaMemcpyDeviceToHost, s));
    BH_CUDA(c, cudaStreamSynchronize(s));
    if (out) {
        std::memset(out, 0, sizeof(*out));
        out->steps = c->blk_steps;
        out->steps_since_rebuild = c->blk_since_rebuild;
        out->now_tick = c->blk_steps ? (int64_t)h.tick_next[(c->blk_steps - 1) & 1] : 0;
        out->n_active = (int64_t)h.n_active;
        out->interactions_now = (int64_t)h.deg_now;
        out->interactions_first = (int64_t)h.deg_base;
    }
    return BH_OK;
}

int bh_leapfrog_step(bh_ctx* c, float theta, float eps, float dt, void* stream) {
    if (!c || !std::isfinite(dt) || !(theta > 0.0f) || !std::isfinite(theta) || !(eps >= 0.0f) || !std::isfinite(eps))
        return BH_ERR_INVALID_ARG;
    if (!c->have_forces) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    const float h = 0.5f * dt;
    int rc;
    c->theta_last = theta;                                    // S6 writes the fp32 records for this theta in the same pass
    if ((rc = stage_kick_drift(c, h, dt, s)) != BH_OK) return rc;
    if ((rc = bh_tree_build(c, stream)) != BH_OK) return rc;
    if ((rc = bh_compute_forces(c, theta, eps, stream)) != BH_OK) return rc;
    if ((rc = stage_kick(c, h, s)) != BH_OK) return rc;
    return BH_OK;
}

int bh_step_graph_build(bh_ctx* c, float theta, float eps, float dt, void* stream) {
    if (!c || !std::isfinite(dt) || !(theta > 0.0f) || !std::isfinite(theta) || !(eps >= 0.0f) || !std::isfinite(eps))
        return BH_ERR_INVALID_ARG;
    if (!c->have_forces || c->copies_pending) return BH_ERR_STATE;
    (void)stream;                                             // nothing runs here; the capture uses an internal stream (the legacy
    cudaStream_t s = c->s_lists;                              // default stream cannot be captured) and the graph is replayed on the caller's
    BH_CUDA(c, cudaSetDevice(c->device));
    drop_step_graph(c);
    // The particle arrays ping-pong (S3 gathers from one set into the other), so a step is captured once for either
    // parity; capturing only records the launches, nothing runs, and after the second capture the host-side state is back
    // where it started.
    const int64_t launches0 = c->launches;
    // ... except for what describes the DEVICE: capturing bh_leapfrog_step walks through its bookkeeping (records written for
    // theta, accelerations in order, split walk timed) although no kernel ran.  Keep the truth and put it back afterwards.
    const bool rec_valid0 = c->rec_valid, acc_in_order0 = c->acc_in_order, split0 = c->walk_split_timed;
    const float rec_theta0 = c->rec_theta, theta_last0 = c->theta_last;
    const int rec_mac0 = c->rec_mac;
    int rc = BH_OK;
    for (int k = 0; k < 2 && rc == BH_OK; ++k) {
        const int parity = c->cur;
        cudaGraph_t g = nullptr;
        BH_CUDA(c, cudaStreamBeginCapture(s, cudaStreamCaptureModeRelaxed));
        c->capturing = true;
        rc = bh_leapfrog_step(c, theta, eps, dt, static_cast<void*>(s));
        c->capturing = false;
        const cudaError_t e = cudaStreamEndCapture(s, &g);
        if (rc == BH_OK && e != cudaSuccess) { c->last_cuda = (int)e; rc = BH_ERR_CUDA; }
        if (rc == BH_OK) {
            const cudaError_t e2 = cudaGraphInstantiate(&c->step_graph[parity], g, 0);
            if (e2 != cudaSuccess) { c->last_cuda = (int)e2; rc = BH_ERR_CUDA; }
        }
        if (g) cudaGraphDestroy(g);
    }
    c->graph_launches = (c->launches - launches0) / 2;
    c->launches = launches0;
    c->graph_split_timed = c->walk_split_timed;               // what a replay leaves behind (bh_step_graph_launch)
    c->rec_valid = rec_valid0; c->rec_theta = rec_theta0; c->rec_mac = rec_mac0;
    c->acc_in_order = acc_in_order0; c->walk_split_timed = split0; c->theta_last = theta_last0;
    if (rc != BH_OK) { (void)cudaGetLastError(); drop_step_graph(c); return rc; }
    c->graph_theta = theta; c->graph_eps = eps; c->graph_dt = dt;
    c->step_graph_valid = true;
    return BH_OK;
}

int bh_step_graph_launch(bh_ctx* c, void* stream) {
    if (!c) return BH_ERR_INVALID_ARG;
    if (!c->step_graph_valid || !c->have_forces || c->copies_pending) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    BH_CUDA(c, cudaGraphLaunch(c->step_graph[c->cur], s));
    // the host-side bookkeeping of bh_leapfrog_step
    c->cur ^= 1;
    c->theta_last = c->graph_theta;
    c->launches += c->graph_launches;
    c->rec_valid = true;                                      // S6 of the captured step wrote the fp32 records for its theta
    c->rec_theta = c->graph_theta;                            // (bh_set_mac drops the graphs, so mac_kind is the captured one)
    c->rec_mac = c->mac_kind;
    c->acc_in_order = true;                                   // a full walk
    c->walk_split_timed = c->graph_split_timed;
    c->have_topology = c->have_tree = c->have_forces = true;
    return BH_OK;
}

int bh_kick_drift(bh_ctx* c, float dt_kick, float dt_drift, void* stream) {
    if (!c || !std::isfinite(dt_kick) || !std::isfinite(dt_drift)) return BH_ERR_INVALID_ARG;
    if (!c->have_forces) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    int rc = stage_kick_drift(c, dt_kick, dt_drift, s);
    if (rc != BH_OK) return rc;
    if (dt_drift != 0.0f) c->have_tree = c->have_forces = false;   // the particles moved; the topology (cells, groups) stays: bh_refresh_moments can revive the tree
    return BH_OK;
}

int bh_sync_status(bh_ctx* c, void* stream, bh_stats* out) {
    if (!c) return BH_ERR_INVALID_ARG;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    DevScalars h;
    BH_CUDA(c, cudaMemcpyAsync(&h, c->ws.sc, sizeof(h), cudaMemcpyDeviceToHost, s));
    BH_CUDA(c, cudaStreamSynchronize(s));
    if (out) {
        std::memset(out, 0, sizeof(*out));
        out->status = h.status;
        out->n = c->n;
        out->launches = c->launches;
        out->sort_retries = (int32_t)h.sort_retries;
        out->sort_passes = (int32_t)(kSortPasses - h.sort_skip);
        if (c->have_tree) {
            out->n_levels = (int32_t)h.n_levels;
            out->n_cells = h.n_cells;
            out->n_groups = h.n_groups;
            for (int k = 0; k < 3; ++k) { out->lo[k] = h.lo[k]; out->hi[k] = h.hi[k]; }
            out->domain_exp = h.dom_e;
        }
        if (c->have_forces || c->theta_last > 0.0f) {
            out->sum_pc = (int64_t)h.sum_pc;
            out->sum_pp = (int64_t)h.sum_pp;
            out->sum_mac = (int64_t)h.sum_mac;
        }
    }
    return h.status;
}

int bh_export_tree(bh_ctx* c, bh_tree_view* v, void* stream) {
    if (!c || !v) return BH_ERR_INVALID_ARG;
    if (!c->have_tree) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    int rc = stage_export(c, s);
    if (rc != BH_OK) return rc;
    const Ws& w = c->ws;
    v->pos_mass = reinterpret_cast<const float*>(w.pos[c->cur]);
    v->vel = reinterpret_cast<const float*>(w.vel[c->cur]);
    v->acc_pot = reinterpret_cast<const float*>(w.acc);
    v->id = w.idb[c->cur];
    v->key = w.key[c->sorted];
    v->perm = w.val[c->sorted];
    v->level_offset = c->ws.sc->level_offset;
    v->cell_level = w.e_level;
    v->cell_prefix = w.e_prefix;
    v->cell_pbegin = w.e_pbegin;
    v->cell_pcount = w.e_pcount;
    v->cell_child_begin = w.e_cbegin;
    v->cell_nchild = w.e_nchild;
    v->cell_parent = w.e_parent;
    v->cell_mom64 = w.mom64;
    v->cell_box = w.box;
    v->cell_mom32 = w.e_mom32;
    v->cell_r2open = w.e_r2open;
    v->cell_trec = reinterpret_cast<const float*>(w.trec);
    v->cell_erec = reinterpret_cast<const float*>(w.erec);
    v->group_begin = w.g_begin;
    v->group_cell = w.g_cell;
    v->group_npc = w.g_npc;
    v->group_npp = w.g_npp;
    return BH_OK;
}

int bh_set_mac(bh_ctx* c, int mac) {
    if (!c || (mac != BH_MAC_EQ1 && mac != BH_MAC_MIN_DISTANCE)) return BH_ERR_INVALID_ARG;
    if (mac == c->mac_kind) return BH_OK;
    c->mac_kind = mac;
    c->have_forces = false;
    drop_step_graph(c);
    return BH_OK;
}

int bh_set_stage_timing(bh_ctx* c, int enable) {
    if (!c) return BH_ERR_INVALID_ARG;
    c->timing = enable != 0;
    return BH_OK;
}

int bh_get_stage_ms(bh_ctx* c, float ms[11]) {
    if (!c || !ms) return BH_ERR_INVALID_ARG;
    if (!c->timing || !c->have_forces) return BH_ERR_STATE;
    BH_CUDA(c, cudaSetDevice(c->device));
    BH_CUDA(c, cudaEventSynchronize(c->ev[10]));
    for (int k = 0; k < 7; ++k) BH_CUDA(c, cudaEventElapsedTime(&ms[k], c->ev[k], c->ev[k + 1]));
    BH_CUDA(c, cudaEventElapsedTime(&ms[7], c->ev[8], c->ev[9]));
    BH_CUDA(c, cudaEventElapsedTime(&ms[8], c->ev[9], c->ev[10]));
    ms[9] = ms[10] = 0.0f;
    if (c->walk_split_timed) {
        BH_CUDA(c, cudaEventElapsedTime(&ms[9], c->ev[9], c->ev[11]));
        BH_CUDA(c, cudaEventElapsedTime(&ms[10], c->ev[11], c->ev[12]));
    }
    return BH_OK;
}

int bh_get_walk_timeline(bh_ctx* c, void* stream, int64_t* ns, int capacity_waves) {
    if (!c || !ns || capacity_waves < 1) return BH_ERR_INVALID_ARG;
    if (!c->have_forces) return BH_ERR_STATE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    BH_CUDA(c, cudaSetDevice(c->device));
    static_assert(sizeof(unsigned long long) == sizeof(int64_t), "timeline words");
    WalkCtl* h = new (std::nothrow) WalkCtl;
    if (!h) return BH_ERR_INVALID_ARG;
    cudaError_t e = cudaMemcpyAsync(h, c->ws.ctl, sizeof(WalkCtl), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { delete h; c->last_cuda = (int)e; return BH_ERR_CUDA; }
    int w = 0;
    for (; w < capacity_waves && w < kMaxWaves && h->t_end[1][w] != 0ull; ++w) {
        ns[4 * w + 0] = (int64_t)h->t_start[0][w]; ns[4 * w + 1] = (int64_t)h->t_end[0][w];
        ns[4 * w + 2] = (int64_t)h->t_start[1][w]; ns[4 * w + 3] = (int64_t)h->t_end[1][w];
    }
    delete h;
    return w;
}

int bh_last_cuda_error(const bh_ctx* c) { return c ? c->last_cuda : 0; }

const char* bh_status_string(int status) {
    switch (status) {
        case BH_OK: return "ok";
        case BH_ERR_INVALID_ARG: return "invalid argument";
        case BH_ERR_WORKSPACE: return "workspace too small, misaligned or not device memory";
        case BH_ERR_STATE: return "call out of order (particles -> tree_build -> compute_forces -> leapfrog_step)";
        case BH_ERR_CUDA: return "CUDA runtime error";
        case BH_ERR_NONFINITE: return "non-finite position or mass <= 0 in the input";
        case BH_ERR_CAPACITY: return "tree needs more cells than max_cells";
        case BH_ERR_TOO_LARGE: return "n is above BH_DOMAIN_STATIC_MAX_N: the built-in scratch of bh_domain_box_static cannot hold it";
        default: return "unknown status";
    }
}

}  // extern "C"
