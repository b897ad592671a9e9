// walk_lists.cu -- S7: the group tree-walk with the MAC of Eq.1, writing the interaction lists.
//
// The paper keeps the two lists of a group in the shared memory of the block that also evaluates them (L83-87).  Here
// the walk and the evaluation are two kernels with different shapes: the walk is a chain of dependent cache round trips
// (pop -> load cell -> test -> push children) that wants many light warps per SM; the evaluation (walk_eval.cu) is a dense
// FP32 loop that wants 128 registers per thread.  The lists travel through device memory as 4-byte indices -- 4 B against
// ~20 x 64 flops per entry, i.e. nothing next to the arithmetic they feed.
//
// One warp walks one group at a time.  A warp claims a TASK of up to eight CONSECUTIVE groups (a super-group, see below:
// Morton neighbours test nearly the same cells), walks what they have in common once and then each of them.  Per group:
//   * frontier: a LIFO of OPENED NODES (first child, child count) in shared memory.  The paper walks breadth-first with two
//     stacks of cells (L83-87); the interaction lists are SETS, so any traversal order produces the same lists and counts.
//     A step pops up to four nodes and gives each of their (up to 8, consecutive) children to one lane: a node of the
//     sparse octree has ~7.8 children, so the lanes are full and the eight records of a node arrive as one 128 B line.
//     Depth-first popping bounds the frontier: the pop width shrinks when the stack nears its capacity and a reserve of
//     7 x 20 + slack entries always admits a pure depth-first descent, so the stack cannot overflow.
//   * each lane tests its cell with exactly the fp32 operations of DESIGN.md O9 (mac_accept).
//   * accepted cells -> the group's cell list; opened nodes -> back onto the stack (one 8-byte entry, ballot-compacted);
//     opened leaves -> a small queue that is expanded 32 leaves at a time into the group's particle list, minus the
//     group's own particles (A19).
// List memory: a warp takes chunks of the wave's list region from a device cursor; inside a chunk cell lists grow upward
// from the bottom, particle lists downward from the top, so both lists of a group are contiguous.  A group that does not
// fit the rest of its warp's chunk is walked again in a fresh chunk; a group that does not fit a whole chunk, or finds
// the region used up, is handed to the fused fallback kernel (walk.cu): the capacity of the list buffer bounds memory,
// never correctness.
#include <algorithm>
#include "walk_common.cuh"

namespace bh {

constexpr int kListWarps = 8;
constexpr int kListThreads = kListWarps * 32;
constexpr int kLStackCap = 512;       // opened nodes
constexpr int kLStackReserve = 160;   // >= 7 * 20 + 7: room for a pure depth-first descent
constexpr int kLeafQueue = 64;
constexpr int kSub = 2;               // sub-batches of 4 nodes (32 children) popped per step: 4 records in flight per lane

struct ListArena { uint32_t pc_top, pp_bot; };
struct WalkSums { unsigned long long pc, pp, mac; };
struct ListWarpShared {
    uint2 stack[kLStackCap];
    uint2 leafq[kLeafQueue];
};

// Expand `k` <= 32 queued leaves (entries q[0..k)) into the particle list, which grows downward from pp_bot.
// Returns false if the list does not fit above pc_top.
__device__ __forceinline__ bool flush_leaves(const uint2* q, int k, int lane, uint32_t gb, uint32_t ge, uint32_t* __restrict__ lists,
                                             uint32_t pc_top, uint32_t& pp_bot, uint32_t& npp) {
    uint32_t first = 0, cnt = 0;
    if (lane < k) { const uint2 e = q[lane]; first = e.x; cnt = e.y; }
    // [first, first + cnt) minus the group's own [gb, ge) = [first, a) and [b, first + cnt)
    const uint32_t end = first + cnt;
    const uint32_t a = min(end, max(first, gb));
    const uint32_t b = max(first, min(end, ge));
    const uint32_t n1 = a - first, kept = n1 + (end - b);
    int total;
    const int off = warp_excl_scan((int)kept, lane, total);
    npp += __reduce_add_sync(0xFFFFFFFFu, cnt);
    if ((uint32_t)total > pp_bot - pc_top) return false;
    pp_bot -= (uint32_t)total;
    uint32_t* dst = lists + pp_bot + off;
#pragma unroll 4
    for (uint32_t t = 0; t < kept; ++t) dst[t] = (t < n1) ? first + t : b + (t - n1);
    return true;
}

// ---- the walk of a SUPER-GROUP: kSG consecutive groups share the part of the walk that is the same for all of them.
// For the union box U of the groups (G inside U for every member G) the fp32 test of O9 is monotone: the per-axis distances
// of G are >= those of U, and <= e_k = max(Umax_k - com_k, com_k - Umin_k); hence
//     d2(U) >  r2open   =>  every member accepts the cell          (d2(G) >= d2(U), each operation rounds monotonically)
//     D2(U) <= r2open   =>  no member accepts it: opened by all    (d2(G) <= D2(U) = fma chain over e_k)
// and only the cells in between ("ambiguous") must be tested by every member on its own.  One warp walks the tree once
// with these two tests: cells accepted by all -> shared cell list, leaves opened by all -> shared particle list (unless the
// leaf holds particles of the super-group itself: own particles are cut out per member, A19), ambiguous cells -> frontier.
// Every member then copies the shared lists into its own lists (4 bytes per entry against ~120 instructions per MAC
// test and append) and continues the walk from the frontier with its own box.  The lists are sets, so the counts are
// exactly those of O9; which groups form a super-group depends on the group index only, never on the active subset.
constexpr int kSG = 8;                  // groups per super-group
constexpr int kAmbCap = 384;
struct SharedWalk {                     // the result of a shared walk: the two shared lists sit in the list region like a group's
    uint32_t amb[kAmbCap];
    uint32_t spc_off, n_spc, spp_off, n_spp, n_amb, leafsum, ok;
};

__device__ __forceinline__ void sg_classify(const float mn[3], const float mx[3], const float4& r, bool& acc_all, bool& open_all) {
    const float ax = __fsub_rn(mn[0], r.x), bx = __fsub_rn(r.x, mx[0]);
    const float ay = __fsub_rn(mn[1], r.y), by = __fsub_rn(r.y, mx[1]);
    const float az = __fsub_rn(mn[2], r.z), bz = __fsub_rn(r.z, mx[2]);
    const float dx = fmaxf(fmaxf(ax, bx), 0.0f), dy = fmaxf(fmaxf(ay, by), 0.0f), dz = fmaxf(fmaxf(az, bz), 0.0f);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    // e_k = max(Umax_k - com_k, com_k - Umin_k) = max(-bx, -ax): the same roundings, negated
    const float ex = fmaxf(-bx, -ax), ey = fmaxf(-by, -ay), ez = fmaxf(-bz, -az);
    const float D2 = __fmaf_rn(ez, ez, __fmaf_rn(ey, ey, __fmul_rn(ex, ex)));
    acc_all = d2 > r.w;
    open_all = !(D2 > r.w);
}

// The shared walk of one super-group (one warp).  The shared lists are written into this warp's chunk of the list region
// (cells upward from pc_top, particles downward from pp_bot, like a group's lists) and stay allocated; sw->ok = 0 when
// they do not fit or the frontier overflows: the members then walk alone.
__device__ __noinline__ void shared_walk(ListWarpShared* ws, SharedWalk* sw, const int lane, const float mn[3], const float mx[3],
                                         const uint32_t sb, const uint32_t se, const float4* __restrict__ trec, const uint2* __restrict__ tlink,
                                         uint32_t* __restrict__ lists, ListArena& ar, WalkSums& sums) {
    const uint32_t lt = (1u << lane) - 1u;
    const uint32_t pc0 = ar.pc_top, pp0 = ar.pp_bot;
    uint32_t pc_top = pc0, pp_bot = pp0;
    uint32_t n_amb = 0, leafsum = 0, nmac = 0;
    bool ok = pp0 > pc0;
    int sp = 1;
    if (lane == 0) ws->stack[0] = make_uint2(0u, 1u);
    __syncwarp();
    while (sp > 0 && ok) {
        // pop up to 4 kSub nodes; lane = (node r of a sub-batch, child c8); all records are requested before any is used
        int kpop = (kLStackCap - kLStackReserve - sp) / 7;
        kpop = max(1, min(kpop, 4 * kSub));
        kpop = min(kpop, sp);
        const int r = lane >> 3, c8 = lane & 7;
        bool valid[kSub];
        uint32_t cell[kSub];
        float4 r0[kSub];
        uint2 lk[kSub];
#pragma unroll
        for (int j = 0; j < kSub; ++j) {
            valid[j] = false;
            cell[j] = 0u;
            const int idx = 4 * j + r;
            if (idx < kpop) {
                const uint2 e = ws->stack[sp - 1 - idx];
                valid[j] = (uint32_t)c8 < e.y;
                cell[j] = e.x + (uint32_t)c8;
            }
        }
#pragma unroll
        for (int j = 0; j < kSub; ++j) {
            r0[j] = make_float4(0.f, 0.f, 0.f, 0.f);
            lk[j] = make_uint2(0u, 0u);
            if (valid[j]) { r0[j] = __ldg(trec + cell[j]); lk[j] = __ldg(tlink + cell[j]); }
        }
        sp -= kpop;
        __syncwarp();
#pragma unroll
        for (int j = 0; j < kSub; ++j) {
            if (4 * j >= kpop) break;
            bool acc_all = false, open_all = false;
            sg_classify(mn, mx, r0[j], acc_all, open_all);
            acc_all = acc_all && valid[j];
            const bool isleaf = (lk[j].y >> 31) != 0u;
            const uint32_t first = lk[j].x, cnt = lk[j].y & 0x7FFFFFFFu;
            const bool opened_node = valid[j] && !acc_all && open_all && !isleaf;
            const bool opened_leaf = valid[j] && !acc_all && open_all && isleaf && !(first < se && first + cnt > sb);   // no particle of the super-group in it
            const bool amb = valid[j] && !acc_all && !opened_node && !opened_leaf;
            nmac += (uint32_t)__popc(__ballot_sync(0xFFFFFFFFu, valid[j]));
            const uint32_t amask = __ballot_sync(0xFFFFFFFFu, acc_all);
            if (amask) {
                if (pc_top + __popc(amask) > pp_bot) { ok = false; break; }
                if (acc_all) lists[pc_top + __popc(amask & lt)] = cell[j];
                pc_top += __popc(amask);
            }
            const uint32_t nmask = __ballot_sync(0xFFFFFFFFu, opened_node);
            if (opened_node) ws->stack[sp + __popc(nmask & lt)] = lk[j];
            sp += __popc(nmask);
            const uint32_t bmask = __ballot_sync(0xFFFFFFFFu, amb);
            if (bmask) {
                if (n_amb + __popc(bmask) > kAmbCap) { ok = false; break; }
                if (amb) sw->amb[n_amb + __popc(bmask & lt)] = cell[j];
                n_amb += __popc(bmask);
            }
            const uint32_t lmask = __ballot_sync(0xFFFFFFFFu, opened_leaf);
            if (lmask) {                                                     // the leaf's particles -> shared particle list
                int total;
                const int off = warp_excl_scan(opened_leaf ? (int)cnt : 0, lane, total);
                if ((uint32_t)total > pp_bot - pc_top) { ok = false; break; }
                pp_bot -= (uint32_t)total;
                if (opened_leaf)
                    for (uint32_t t = 0; t < cnt; ++t) lists[pp_bot + off + t] = first + t;
                leafsum += (uint32_t)total;
            }
        }
        __syncwarp();
    }
    if (ok) { ar.pc_top = pc_top; ar.pp_bot = pp_bot; sums.mac += nmac; }     // the shared lists stay allocated
    if (lane == 0) {
        sw->spc_off = pc0; sw->n_spc = pc_top - pc0; sw->spp_off = pp_bot; sw->n_spp = pp0 - pp_bot;
        sw->n_amb = n_amb; sw->leafsum = leafsum; sw->ok = ok ? 1u : 0u;
    }
    __syncwarp();
}

// The walk of one group; `sw` != nullptr: continue from the shared walk of its super-group instead of starting at the root.
template <int kMac>
__device__ __forceinline__ bool list_group(ListWarpShared* ws, const int lane, const uint32_t g, const uint32_t gb, const uint32_t ge,
                                           const float mn[3], const float mx[3], const SharedWalk* sw,
                                           const float4* __restrict__ trec, const uint2* __restrict__ tlink,
                                           const float* __restrict__ box,
                                           uint32_t* __restrict__ lists, ListArena& ar, WalkListOut o, WalkSums& sums) {
    const uint32_t lt = (1u << lane) - 1u;
    const int ng = (int)(ge - gb);
    const uint32_t pc0 = ar.pc_top, pp0 = ar.pp_bot;
    uint32_t pc_top = pc0, pp_bot = pp0;
    uint32_t npp = 0, nmac = 0;
    bool fits = true;
    int sp = 0, lq = 0;

    // one test + append of a cell by every lane that holds one (cell, r0, lk valid where `valid`)
    auto classify = [&](bool valid, uint32_t cell, const float4& r0, const uint2& lk, const CellBox& cbx) -> bool {
        const bool accept = valid && (kMac == kMacMinDist ? mac_accept_box(mn, mx, cbx, r0.w) : mac_accept(mn, mx, r0));
        const bool isleaf = valid && !accept && (lk.y >> 31) != 0u;
        const bool isnode = valid && !accept && !isleaf;
        nmac += (uint32_t)__popc(__ballot_sync(0xFFFFFFFFu, valid));
        // ---- accepted cells -> cell list
        const uint32_t amask = __ballot_sync(0xFFFFFFFFu, accept);
        if (amask) {
            const uint32_t na = (uint32_t)__popc(amask);
            if (pc_top + na > pp_bot) return false;
            if (accept) lists[pc_top + (uint32_t)__popc(amask & lt)] = cell;
            pc_top += na;
        }
        // ---- opened nodes -> back onto the stack (the callers guarantee room for 32 entries)
        const uint32_t nmask = __ballot_sync(0xFFFFFFFFu, isnode);
        if (isnode) ws->stack[sp + __popc(nmask & lt)] = lk;
        sp += __popc(nmask);
        // ---- opened leaves -> queue; expanded 32 at a time
        const uint32_t lmask = __ballot_sync(0xFFFFFFFFu, isleaf);
        if (lmask) {
            if (isleaf) ws->leafq[lq + __popc(lmask & lt)] = make_uint2(lk.x, lk.y & 0x7FFFFFFFu);
            lq += __popc(lmask);
            __syncwarp();
            if (lq >= 32) {
                lq -= 32;
                if (!flush_leaves(ws->leafq + lq, 32, lane, gb, ge, lists, pc_top, pp_bot, npp)) return false;
            }
        }
        return true;
    };
    // the stack of opened nodes, until it is empty
    auto drain = [&]() {
        while (sp > 0 && fits) {
            // pop up to 4 kSub nodes; lane = (node r of a sub-batch, child c8); all records are requested before any is used
            int kpop = (kLStackCap - kLStackReserve - sp) / 7;
            kpop = max(1, min(kpop, 4 * kSub));
            kpop = min(kpop, sp);
            const int r = lane >> 3, c8 = lane & 7;
            bool valid[kSub];
            uint32_t cell[kSub];
            float4 r0[kSub];
            uint2 lk[kSub];
            CellBox cbx[kMac == kMacMinDist ? kSub : 1];
#pragma unroll
            for (int j = 0; j < kSub; ++j) {
                valid[j] = false;
                cell[j] = 0u;
                const int idx = 4 * j + r;
                if (idx < kpop) {
                    const uint2 e = ws->stack[sp - 1 - idx];
                    valid[j] = (uint32_t)c8 < e.y;
                    cell[j] = e.x + (uint32_t)c8;
                }
            }
#pragma unroll
            for (int j = 0; j < kSub; ++j) {
                r0[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                lk[j] = make_uint2(0u, 0u);
                if (valid[j]) {
                    r0[j] = __ldg(trec + cell[j]);
                    lk[j] = __ldg(tlink + cell[j]);
                    if (kMac == kMacMinDist) cbx[j] = load_cell_box(box, cell[j]);
                }
            }
            sp -= kpop;
            __syncwarp();                 // every lane has read its stack entries: the slots may be overwritten
#pragma unroll
            for (int j = 0; j < kSub; ++j) {
                if (4 * j >= kpop) break;
                if (!classify(valid[j], cell[j], r0[j], lk[j], cbx[kMac == kMacMinDist ? j : 0])) { fits = false; break; }
            }
            __syncwarp();
        }
    };

    if (sw == nullptr) {
        sp = 1;
        if (lane == 0) ws->stack[0] = make_uint2(0u, 1u);   // the root (A17) as the only child of a virtual node
        __syncwarp();
        drain();
    } else {
        // what every member of the super-group has in common: copy it
        const uint32_t nc = sw->n_spc, np = sw->n_spp;
        if (pc_top + nc + np > pp_bot) fits = false;
        if (fits) {
            const uint32_t* src_c = lists + sw->spc_off;
            const uint32_t* src_p = lists + sw->spp_off;
            for (uint32_t i0 = 0; i0 < nc; i0 += 256) {                 // eight loads in flight per lane
                uint32_t v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) v[u] = __ldcg(src_c + min(i0 + 32 * u + lane, nc - 1));
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (i0 + 32 * u + lane < nc) lists[pc_top + i0 + 32 * u + lane] = v[u];
            }
            pc_top += nc;
            pp_bot -= np;
            for (uint32_t i0 = 0; i0 < np; i0 += 256) {
                uint32_t v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) v[u] = __ldcg(src_p + min(i0 + 32 * u + lane, np - 1));
#pragma unroll
                for (int u = 0; u < 8; ++u)
                    if (i0 + 32 * u + lane < np) lists[pp_bot + i0 + 32 * u + lane] = v[u];
            }
            npp = sw->leafsum;
            // the ambiguous cells, 32 at a time, each followed by the walk below the nodes it opened
            const uint32_t na = sw->n_amb;
            for (uint32_t a0 = 0; a0 < na && fits; a0 += 32) {
                const bool valid = a0 + lane < na;
                const uint32_t cell = valid ? sw->amb[a0 + lane] : 0u;
                float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f);
                uint2 lk = make_uint2(0u, 0u);
                CellBox cbx;
                if (valid) {
                    r0 = __ldg(trec + cell);
                    lk = __ldg(tlink + cell);
                    if (kMac == kMacMinDist) cbx = load_cell_box(box, cell);
                }
                if (!classify(valid, cell, r0, lk, cbx)) { fits = false; break; }
                __syncwarp();
                drain();
            }
        }
    }
    if (fits && lq > 0) fits = flush_leaves(ws->leafq, lq, lane, gb, ge, lists, pc_top, pp_bot, npp);

    if (fits) {
        ar.pc_top = pc_top;
        ar.pp_bot = pp_bot;
        if (lane == 0) {
            o.g_pcoff[g] = pc0;
            o.g_ppoff[g] = pp_bot;
            o.g_lpp[g] = pp0 - pp_bot;
            o.g_npc[g] = pc_top - pc0;
            o.g_npp[g] = npp;
        }
        sums.pc += (unsigned long long)(pc_top - pc0) * (unsigned long long)ng;
        sums.pp += (unsigned long long)npp * (unsigned long long)ng;
        sums.mac += nmac;
    }
    __syncwarp();
    return fits;                       // false: nothing was committed (the entries written so far are simply abandoned)
}

// A chunk of the wave's list region for this warp (bump allocation from a device cursor).  False when the region is used up.
__device__ __forceinline__ bool alloc_chunk(WalkCtl* ctl, int wave, int lane, uint32_t region_base, uint32_t region_entries,
                                            uint32_t chunk_entries, ListArena& ar) {
    // the cursor saturates: once the region is used up nobody adds to it any more, so it can never wrap around and hand
    // out a chunk twice however many groups still ask
    uint32_t off = region_entries;
    if (lane == 0 && ld_relaxed_u32(&ctl->arena_next[wave]) < region_entries) off = atomicAdd(&ctl->arena_next[wave], chunk_entries);
    off = __shfl_sync(0xFFFFFFFFu, off, 0);
    if (off >= region_entries || region_entries - off < chunk_entries) { ar.pc_top = ar.pp_bot = 0u; return false; }
    ar.pc_top = region_base + off;
    ar.pp_bot = ar.pc_top + chunk_entries;
    return true;
}

constexpr size_t kListSmem = (sizeof(ListWarpShared) + sizeof(SharedWalk)) * kListWarps;   // per warp: its walk state + one shared walk

// The box of group g (A13).  A group that is a whole cell has that cell's box (exact min / max of the same particles); a
// chunk of an over-full leaf takes it from its particles (all lanes take part).
__device__ __forceinline__ void load_group_box(uint32_t g, uint32_t gb, uint32_t ge, int lane, const float4* __restrict__ pos,
                                               const float* __restrict__ box, const uint32_t* __restrict__ g_cell,
                                               const uint4* __restrict__ c_topo, float mn[3], float mx[3]) {
    const uint32_t gc = __ldg(g_cell + g);
    const uint2 pr = __ldg(reinterpret_cast<const uint2*>(c_topo + gc));     // (first particle, end particle) of the group's cell
    if (pr.y - pr.x == ge - gb) {
        const float* bb = box + 6 * (size_t)gc;
        mn[0] = __ldg(bb); mn[1] = __ldg(bb + 1); mn[2] = __ldg(bb + 2);
        mx[0] = __ldg(bb + 3); mx[1] = __ldg(bb + 4); mx[2] = __ldg(bb + 5);
    } else {
        group_box(pos, gb, (int)(ge - gb), lane, nullptr, mn, mx);
    }
}

template <int kMac>
__global__ void __launch_bounds__(kListThreads, 4) k_walk_lists(WalkListOut o, int wave, const float4* __restrict__ pos,
                                                                const float4* __restrict__ trec, const uint2* __restrict__ tlink,
                                                                const float* __restrict__ box, const uint32_t* __restrict__ g_cell,
                                                                const uint4* __restrict__ c_topo,
                                                                const uint32_t* __restrict__ g_begin, uint32_t* __restrict__ lists,
                                                                uint32_t region_base, uint32_t region_entries, uint32_t chunk_entries,
                                                                const uint8_t* __restrict__ g_active, int share) {
    extern __shared__ __align__(16) unsigned char list_smem[];
    ListWarpShared* s_ws = reinterpret_cast<ListWarpShared*>(list_smem);
    SharedWalk* s_sw = reinterpret_cast<SharedWalk*>(list_smem + sizeof(ListWarpShared) * kListWarps);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t g0 = o.ctl->wave_g[wave], g1 = o.ctl->wave_g[wave + 1];
    if (threadIdx.x == 0) atomicMin(&o.ctl->t_start[0][wave], global_ns());
    ListArena ar = {0u, 0u};           // this warp's current chunk of the list region: cell lists grow up, particle lists down
    uint32_t last_total = 0u;          // entries of the last group this warp listed: Morton neighbours need about as many
    WalkSums sums = {0ull, 0ull, 0ull};
    const bool sharing = share && kMac == kMacEq1;
    for (;;) {
        // every warp claims its own super-group: no warp ever waits for another.  Task t covers a FIXED range of groups (the
        // partition depends on the number of groups only, so the lists, and with them the order of the fp32 sums, do not
        // depend on timing or on the active subset): eight groups per task over the first 70 % of the groups, four up to
        // 93 %, then two -- small tasks at the end keep the tail of the kernel short.
        uint32_t claim = 0;
        if (lane == 0) claim = atomicAdd(&o.ctl->list_next[wave], 1u);
        claim = __shfl_sync(0xFFFFFFFFu, claim, 0);
        const uint32_t Gw = g1 - g0;
        // (few groups per warp, e.g. 16 K particles: a warp that walks for eight groups leaves seven warps idle: smaller tasks)
        const uint32_t szA = min(max(Gw / (gridDim.x * kListWarps), 1u), (uint32_t)kSG);
        const uint32_t nA = (uint32_t)(0.70f * (float)Gw) / szA, gA = nA * szA;
        const uint32_t szB = szA >= 4 ? szA / 2 : szA;
        const uint32_t nB = ((uint32_t)(0.93f * (float)Gw) > gA ? (uint32_t)(0.93f * (float)Gw) - gA : 0u) / szB, gB = gA + nB * szB;
        const uint32_t szC = szA >= 4 ? szA / 4 : szA;
        uint32_t off, sz;
        if (claim < nA) { off = claim * szA; sz = szA; }
        else if (claim < nA + nB) { off = gA + (claim - nA) * szB; sz = szB; }
        else { off = gB + (claim - nA - nB) * szC; sz = szC; }
        if (off >= Gw) break;
        const uint32_t base = g0 + off;
        const uint32_t nchunk = min(sz, g1 - base);
        const uint32_t s0 = 0u;
        // ---- warp w takes the super-group w of the chunk (groups base + kSG w ...): one shared walk, then its members one by
        //      one from where the shared walk stopped.  No warp waits for another inside a chunk.
        SharedWalk* sw = s_sw + warp;
        const uint32_t nm = s0 < nchunk ? min((uint32_t)kSG, nchunk - s0) : 0u;
        bool shared_ok = false;
        if (sharing && nm >= 2u) {
            bool any = false;
            for (uint32_t m = 0; m < nm; ++m) any = any || !(g_active && !__ldg(g_active + base + s0 + m));
            if (any) {
                // the union box of EVERY member, active or not: the split must not depend on the subset that is walked
                float un[3] = {INFINITY, INFINITY, INFINITY}, ux[3] = {-INFINITY, -INFINITY, -INFINITY};
                for (uint32_t m = 0; m < nm; ++m) {
                    const uint32_t g = base + s0 + m;
                    float mn[3], mx[3];
                    load_group_box(g, __ldg(g_begin + g), __ldg(g_begin + g + 1), lane, pos, box, g_cell, c_topo, mn, mx);
#pragma unroll
                    for (int k = 0; k < 3; ++k) { un[k] = fminf(un[k], mn[k]); ux[k] = fmaxf(ux[k], mx[k]); }
                }
                const uint32_t sb = __ldg(g_begin + base + s0), se = __ldg(g_begin + base + s0 + nm);
                if (ar.pp_bot - ar.pc_top < last_total + (last_total >> 1) + 256u) alloc_chunk(o.ctl, wave, lane, region_base, region_entries, chunk_entries, ar);
                shared_walk(&s_ws[warp], sw, lane, un, ux, sb, se, trec, tlink, lists, ar, sums);
                shared_ok = sw->ok != 0u;
            }
        }
        for (uint32_t m = 0; m < nm; ++m) {
            const uint32_t g = base + s0 + m;
            if (g_active && !__ldg(g_active + g)) {      // block time-steps: not in this walk's subset
                if (lane == 0) { o.g_pcoff[g] = kSkip; o.g_npc[g] = 0u; o.g_npp[g] = 0u; }
                continue;
            }
            const uint32_t gb = __ldg(g_begin + g), ge = __ldg(g_begin + g + 1);
            float mn[3], mx[3];
            load_group_box(g, gb, ge, lane, pos, box, g_cell, c_topo, mn, mx);
            const SharedWalk* swp = shared_ok ? sw : nullptr;
            // a fresh chunk if this one will probably not do; a second try in a fresh chunk if it did not; a group that does
            // not fit a whole chunk (or finds the region used up) goes to the fused kernel instead
            bool fresh = false;
            if (ar.pp_bot - ar.pc_top < last_total + (last_total >> 2) + 64u) {
                fresh = true;
                alloc_chunk(o.ctl, wave, lane, region_base, region_entries, chunk_entries, ar);
            }
            const uint32_t before = ar.pp_bot - ar.pc_top;
            bool ok = before != 0u && list_group<kMac>(&s_ws[warp], lane, g, gb, ge, mn, mx, swp, trec, tlink, box, lists, ar, o, sums);
            if (!ok && !fresh && alloc_chunk(o.ctl, wave, lane, region_base, region_entries, chunk_entries, ar)) {
                const uint32_t b2 = ar.pp_bot - ar.pc_top;
                ok = list_group<kMac>(&s_ws[warp], lane, g, gb, ge, mn, mx, swp, trec, tlink, box, lists, ar, o, sums);
                if (ok) last_total = b2 - (ar.pp_bot - ar.pc_top);
            } else if (ok) {
                last_total = before - (ar.pp_bot - ar.pc_top);
            }
            if (!ok && lane == 0) {
                o.g_pcoff[g] = kNone;
                o.deferred[atomicAdd(&o.ctl->n_deferred, 1u)] = g;
            }
            __syncwarp();
        }
    }
    if (threadIdx.x == 0) atomicMax(&o.ctl->t_end[0][wave], global_ns());
    if (lane == 0 && (sums.mac || sums.pc || sums.pp)) {
        atomicAdd(&o.sc->sum_pc, sums.pc);
        atomicAdd(&o.sc->sum_pp, sums.pp);
        atomicAdd(&o.sc->sum_mac, sums.mac);
    }
}

// Wave boundaries (first group whose first particle is >= w * wave_particles) and counter reset: one tiny launch per walk.
__global__ void k_walk_prepare(DevScalars* sc, WalkCtl* ctl, const uint32_t* __restrict__ g_begin, int nwaves, uint32_t wave_particles) {
    const int t = threadIdx.x;
    const uint32_t G = sc->n_groups;
    if (t <= nwaves) {
        uint32_t lo = 0, hi = G;           // lower_bound of t * wave_particles in g_begin[0..G)
        const unsigned long long target = (unsigned long long)t * wave_particles;
        if (t == nwaves) lo = G;
        else if (t == 0) lo = 0;           // (no search for the common one-wave walk)
        else
            while (lo < hi) {
                const uint32_t mid = (lo + hi) >> 1;
                if ((unsigned long long)g_begin[mid] < target) lo = mid + 1; else hi = mid;
            }
        ctl->wave_g[t] = lo;
        ctl->list_next[t] = 0;
        ctl->eval_next[t] = 0;
        ctl->arena_next[t] = 0;
        ctl->t_start[0][t] = ctl->t_start[1][t] = ~0ull;
        ctl->t_end[0][t] = ctl->t_end[1][t] = 0ull;
    }
    if (t == 0) {
        ctl->n_deferred = 0;
        ctl->fused_next = 0;
        sc->sum_pc = 0; sc->sum_pp = 0; sc->sum_mac = 0;
    }
}

int stage_walk_lists(bh_ctx* c, int wave, int grid, uint32_t region_base, uint32_t region_entries, cudaStream_t s) {
    // chunk: a third of a warp's even share of the region, within [4096, 65536] entries (a group's lists must fit one chunk)
    const uint32_t share = region_entries / ((uint32_t)grid * kListWarps * 3u);
    const uint32_t chunk_entries = std::min(std::max(std::min(share, 65536u), 4096u), region_entries);
    WalkListOut o = walk_list_out(c);
    if (c->mac_kind == kMacMinDist) {
        BH_LAUNCH(c, k_walk_lists<kMacMinDist>, grid, kListThreads, kListSmem, s, o, wave, c->ws.pos[c->cur], c->ws.trec, c->ws.tlink, c->ws.box, c->ws.g_cell,
                  c->ws.c_topo, c->ws.g_begin, c->ws.lists, region_base, region_entries, chunk_entries,
                  c->active ? c->ws.gflag : nullptr, c->walk_share);
        return BH_OK;
    }
    BH_LAUNCH(c, k_walk_lists<kMacEq1>, grid, kListThreads, kListSmem, s, o, wave, c->ws.pos[c->cur], c->ws.trec, c->ws.tlink, c->ws.box, c->ws.g_cell,
              c->ws.c_topo, c->ws.g_begin, c->ws.lists, region_base, region_entries, chunk_entries,
                  c->active ? c->ws.gflag : nullptr, c->walk_share);
    return BH_OK;
}

// Groups that hold at least one active particle (block time-steps): g_active[g] = any(active[gb .. ge)).
__global__ void __launch_bounds__(256) k_group_active(const DevScalars* __restrict__ sc, const uint32_t* __restrict__ g_begin,
                                                      const uint8_t* __restrict__ active, uint8_t* __restrict__ g_active) {
    const uint32_t G = sc->n_groups;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < G; g += gridDim.x * blockDim.x) {
        uint8_t any = 0;
        for (uint32_t i = g_begin[g]; i < g_begin[g + 1]; ++i) any |= active[i];
        g_active[g] = any ? 1 : 0;
    }
}

int stage_group_active(bh_ctx* c, const uint8_t* d_active, cudaStream_t s) {
    // ws.gflag is free after the build (it marks group starts per particle for S5 only): it now holds one flag per group
    const int grid = (int)std::min<int64_t>(div_up(c->n, 256), (int64_t)c->sm_count * 8);
    BH_LAUNCH(c, k_group_active, grid, 256, 0, s, c->ws.sc, c->ws.g_begin, d_active, c->ws.gflag);
    return BH_OK;
}

int walk_lists_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_lists<kMacEq1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kListSmem));
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_lists<kMacMinDist>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kListSmem));
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_lists<kMacEq1>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_lists<kMacMinDist>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    return BH_OK;
}

int stage_walk_prepare(bh_ctx* c, int nwaves, uint32_t wave_particles, cudaStream_t s) {
    BH_LAUNCH(c, k_walk_prepare, 1, kMaxWaves + 1, 0, s, c->ws.sc, c->ws.ctl, c->ws.g_begin, nwaves, wave_particles);
    return BH_OK;
}

}  // namespace bh
