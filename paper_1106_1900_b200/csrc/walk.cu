// walk.cu -- S7 + S8 sequencing, and the fused fallback kernel.
//
// bh_compute_forces runs the walk as
//   k_walk_prepare                       wave boundaries, counters                       (walk_lists.cu)
//   per wave:  k_walk_lists              S7: MAC walk -> interaction lists (indices)     (walk_lists.cu)
//              k_walk_eval               S8: forces + potentials from the lists          (walk_eval.cu)
//   k_walk_fused                         S7 + S8 of the groups whose lists did not fit   (this file; normally none)
// A "wave" is a contiguous range of particles (hence of groups) sized on the host so that its lists are expected to fit
// the list buffer of the workspace; nothing is read back, so the whole sequence can be captured into a CUDA graph.  A
// group whose lists fit neither a chunk of the list region nor what is left of it is deferred by k_walk_lists and handled
// here instead (the round-1 one-kernel walk): one warp per group, frontier LIFO, accepted cells and leaf particles staged
// in shared-memory rings of 64 entries and swept every 32 with the slot evaluation of walk_common.cuh.
// Capacity therefore bounds memory, never the result.
#include <algorithm>
#include <cmath>
#include "walk_common.cuh"

namespace bh {

constexpr int kWalkWarps = 8;
constexpr int kWalkThreads = kWalkWarps * 32;
constexpr int kStackCap = 1024;
constexpr int kStackReserve = 160;   // >= 7 * 20 + 7: room for a pure depth-first descent
constexpr int kRing = 64;            // ring capacity in entries (power of two, >= 63)
constexpr int kRingPairs = kRing / 2;

struct __align__(16) WarpShared {
    float pc[kRingPairs * kPcPair];
    float pp[kRingPairs * kPpPair];
    float4 own[64];                  // the group's particles (targets; sources of the self block)
    SlotTotals tot[kMaxSlots];
    uint32_t stack[kStackCap];
    uint32_t run_begin[32];
    uint32_t run_off[36];
};

// An odd tail gets a massless partner at the position of the last real entry (a position no target can coincide with).
__device__ __forceinline__ void pc_pad(float* ring, int e_last) {
    const float* s = ring + (e_last >> 1) * kPcPair + (e_last & 1);
    pc_store(ring, (e_last + 1) & (kRing - 1), s[0], s[2], s[4], 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f);
}
__device__ __forceinline__ void pp_pad(float* ring, int e_last) {
    const float* s = ring + (e_last >> 1) * kPpPair + (e_last & 1);
    pp_store(ring, (e_last + 1) & (kRing - 1), s[0], s[2], s[4], 0.f);
}

template <int kMac>
__device__ __noinline__ void walk_group(WarpShared* ws, const int lane, const uint32_t g, const uint32_t gb, const uint32_t ge,
                                        const float4* __restrict__ pos, const float4* __restrict__ trec, const uint2* __restrict__ tlink,
                                        const float* __restrict__ box, const float4* __restrict__ erec, float eps2, float4* __restrict__ acc_out,
                                        uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp, DevScalars* sc) {
    const uint32_t lt = (1u << lane) - 1u;
    const int ng = (int)(ge - gb);
    const Consts k = make_consts(eps2);
    float mn[3], mx[3];
    group_box(pos, gb, ng, lane, ws->own, mn, mx);
    const int m = (ng + 3) & ~3;
    totals_clear(ws->tot, lane);

    int sp = 1;
    if (lane == 0) ws->stack[0] = 0u;   // the root (A17)
    __syncwarp();
    int pc_head = 0, pc_cnt = 0, pp_head = 0, pp_cnt = 0;   // heads are even (entries are consumed 32 at a time)
    uint32_t npc = 0, npp = 0, nmac = 0;

    while (sp > 0) {
        int kpop = (kStackCap - kStackReserve - sp) / 7;
        kpop = max(1, min(kpop, 32));
        kpop = min(kpop, sp);
        const bool valid = lane < kpop;
        bool accept = false, isleaf = false, isnode = false;
        uint32_t cell = 0, first = 0, cnt = 0;
        if (valid) {
            cell = ws->stack[sp - 1 - lane];
            const float4 r0 = __ldg(trec + cell);
            const uint2 lk = __ldg(tlink + cell);
            accept = kMac == kMacMinDist ? mac_accept_box(mn, mx, load_cell_box(box, cell), r0.w) : mac_accept(mn, mx, r0);
            if (!accept) {
                first = lk.x;
                cnt = lk.y & 0x7FFFFFFFu;
                isleaf = (lk.y >> 31) != 0u;
                isnode = !isleaf;
            }
        }
        sp -= kpop;
        nmac += (uint32_t)kpop;
        __syncwarp();
        // ---- accepted cells -> p-c ring (the evaluation record is already in the ring's units: a plain copy)
        const uint32_t amask = __ballot_sync(0xFFFFFFFFu, accept);
        if (amask) {
            if (accept) {
                const float4 e0 = __ldg(erec + 3 * (size_t)cell), e1 = __ldg(erec + 3 * (size_t)cell + 1), e2 = __ldg(erec + 3 * (size_t)cell + 2);
                const int e = (pc_head + pc_cnt + __popc(amask & lt)) & (kRing - 1);
                pc_store(ws->pc, e, e0.x, e0.y, e0.z, e0.w, e1.x, e1.y, e1.z, e1.w, e2.x, e2.y, e2.z, e2.w);
            }
            const int na = __popc(amask);
            pc_cnt += na;
            npc += (uint32_t)na;
        }
        // ---- opened nodes -> children onto the stack
        const uint32_t nmask = __ballot_sync(0xFFFFFFFFu, isnode);
        if (nmask) {
            int total;
            const int off = warp_excl_scan(isnode ? (int)cnt : 0, lane, total);
            if (sp + total > kStackCap) {            // cannot happen (see kStackReserve); never write out of bounds
                if (lane == 0) atomicMin(&sc->status, (int)BH_ERR_CAPACITY);
                sp = 0;
                break;
            }
            if (isnode)
                for (uint32_t j = 0; j < cnt; ++j) ws->stack[sp + off + (int)j] = first + j;
            sp += total;
        }
        __syncwarp();
        // ---- opened leaves -> p-p ring (own particles skipped).  The particle indices are first laid out in the free
        //      space above the stack top (one store per particle), so that each lane then finds its source with one load.
        const uint32_t lmask = __ballot_sync(0xFFFFFFFFu, isleaf);
        if (lmask) {
            int total;
            const int off = warp_excl_scan(isleaf ? (int)cnt : 0, lane, total);
            npp += (uint32_t)total;
            const bool direct = total <= kStackCap - sp;
            const int nl = __popc(lmask);
            if (direct) {
                if (isleaf)
                    for (uint32_t j = 0; j < cnt; ++j) ws->stack[sp + off + (int)j] = first + j;
            } else if (isleaf) {                      // (overflow leaves, nearly full stack) search the runs instead
                const int r = __popc(lmask & lt);
                ws->run_begin[r] = first;
                ws->run_off[r] = (uint32_t)off;
            }
            __syncwarp();
            for (int t0 = 0; t0 < total; t0 += 32) {
                const int t = t0 + lane;
                bool keep = false;
                uint32_t src = 0;
                if (t < total) {
                    if (direct) {
                        src = ws->stack[sp + t];
                    } else {
                        int lo = 0, hi = nl - 1;
                        while (lo < hi) {
                            const int mid = (lo + hi + 1) >> 1;
                            if ((int)ws->run_off[mid] <= t) lo = mid; else hi = mid - 1;
                        }
                        src = ws->run_begin[lo] + (uint32_t)(t - (int)ws->run_off[lo]);
                    }
                    keep = !(src >= gb && src < ge);
                }
                const uint32_t kmask = __ballot_sync(0xFFFFFFFFu, keep);
                if (keep) {
                    const float4 p = __ldg(pos + src);
                    pp_store(ws->pp, (pp_head + pp_cnt + __popc(kmask & lt)) & (kRing - 1), p.x, p.y, p.z, p.w);
                }
                pp_cnt += __popc(kmask);
                __syncwarp();
                if (pp_cnt >= 32) {
                    eval_pp_all<false, kRingPairs, true>(ws->pp, ws->own, ws->tot, pp_head >> 1, 16, m, ng, k, lane);
                    pp_head = (pp_head + 32) & (kRing - 1);
                    pp_cnt -= 32;
                    __syncwarp();
                }
            }
            __syncwarp();
        }
        if (pc_cnt >= 32) {
            eval_pc_all<kRingPairs, true, false>(ws->pc, ws->own, ws->tot, pc_head >> 1, 16, m, ng, k, lane);
            pc_head = (pc_head + 32) & (kRing - 1);
            pc_cnt -= 32;
            __syncwarp();
        }
    }
    // ---- flush the rings (an odd tail gets a massless partner)
    if (pc_cnt > 0) {
        if ((pc_cnt & 1) && lane == 0) pc_pad(ws->pc, (pc_head + pc_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pc_all<kRingPairs, true, false>(ws->pc, ws->own, ws->tot, pc_head >> 1, (pc_cnt + 1) >> 1, m, ng, k, lane);
    }
    if (pp_cnt > 0) {
        if ((pp_cnt & 1) && lane == 0) pp_pad(ws->pp, (pp_head + pp_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pp_all<false, kRingPairs, true>(ws->pp, ws->own, ws->tot, pp_head >> 1, (pp_cnt + 1) >> 1, m, ng, k, lane);
    }
    __syncwarp();
    // ---- self block: the group's own particles, entry j = target index j, j != i
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) { const float4 p = ws->own[idx]; pp_store(ws->pp, idx, p.x, p.y, p.z, p.w); }
    }
    __syncwarp();
    if ((ng & 1) && lane == 0) pp_pad(ws->pp, ng - 1);
    __syncwarp();
    eval_pp_all<true, kRingPairs, true>(ws->pp, ws->own, ws->tot, 0, (ng + 1) >> 1, m, ng, k, lane);
    __syncwarp();
    totals_finish(ws->tot, m, lane, ng, gb, acc_out);
    __syncwarp();
    if (lane == 0) {
        g_npc[g] = npc;
        g_npp[g] = npp;
        atomicAdd(&sc->sum_pc, (unsigned long long)npc * (unsigned long long)ng);
        atomicAdd(&sc->sum_pp, (unsigned long long)npp * (unsigned long long)ng);
        atomicAdd(&sc->sum_mac, (unsigned long long)nmac);
    }
}

// The groups k_walk_lists deferred (ctl->n_deferred of them; with `all` != 0: every group, the list path is bypassed).
template <int kMac>
__global__ void __launch_bounds__(kWalkThreads, 2) k_walk_fused(DevScalars* sc, WalkCtl* ctl, int all, const uint32_t* __restrict__ deferred,
                                                                const float4* __restrict__ pos, const float4* __restrict__ trec,
                                                                const uint2* __restrict__ tlink, const float* __restrict__ box, const float4* __restrict__ erec,
                                                                const uint32_t* __restrict__ g_begin, float eps2, float4* __restrict__ acc_out,
                                                                uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp,
                                                                const uint8_t* __restrict__ g_active) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpShared* ws = reinterpret_cast<WarpShared*>(smem_raw) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    const uint32_t count = all ? sc->n_groups : ctl->n_deferred;
    if (count == 0) return;
    for (;;) {
        uint32_t i = 0;
        if (lane == 0) i = atomicAdd(&ctl->fused_next, 1u);
        i = __shfl_sync(0xFFFFFFFFu, i, 0);
        if (i >= count) break;
        const uint32_t g = all ? i : deferred[i];
        if (all && g_active && !__ldg(g_active + g)) {   // not in this walk's subset (the list path filters before deferring)
            if (lane == 0) { g_npc[g] = 0u; g_npp[g] = 0u; }
            continue;
        }
        const uint32_t gb = __ldg(g_begin + g), ge = __ldg(g_begin + g + 1);
        walk_group<kMac>(ws, lane, g, gb, ge, pos, trec, tlink, box, erec, eps2, acc_out, g_npc, g_npp, sc);
        __syncwarp();
    }
}

WalkListOut walk_list_out(bh_ctx* c) {
    WalkListOut o;
    o.sc = c->ws.sc;
    o.ctl = c->ws.ctl;
    o.g_pcoff = c->ws.g_pcoff;
    o.g_ppoff = c->ws.g_ppoff;
    o.g_lpp = c->ws.g_lpp;
    o.g_npc = c->ws.g_npc;
    o.g_npp = c->ws.g_npp;
    o.deferred = c->ws.deferred;
    return o;
}

int walk_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_fused<kMacEq1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(WarpShared) * kWalkWarps)));
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_fused<kMacMinDist>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(WarpShared) * kWalkWarps)));
    BH_CUDA(c, cudaStreamCreateWithFlags(&c->s_lists, cudaStreamNonBlocking));
    BH_CUDA(c, cudaStreamCreateWithFlags(&c->s_eval2, cudaStreamNonBlocking));
    BH_CUDA(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
    BH_CUDA(c, cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
    for (int k = 0; k <= kMaxWaves; ++k) {
        BH_CUDA(c, cudaEventCreateWithFlags(&c->ev_lists[k], cudaEventDisableTiming));
        BH_CUDA(c, cudaEventCreateWithFlags(&c->ev_eval[k], cudaEventDisableTiming));
    }
    return walk_eval_init(c);
}

int walk_destroy(bh_ctx* c) {
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    for (int k = 0; k <= kMaxWaves; ++k) {
        if (c->ev_lists[k]) cudaEventDestroy(c->ev_lists[k]);
        if (c->ev_eval[k]) cudaEventDestroy(c->ev_eval[k]);
    }
    if (c->s_lists) cudaStreamDestroy(c->s_lists);
    if (c->s_eval2) cudaStreamDestroy(c->s_eval2);
    return BH_OK;
}

// Expected list entries per particle (cells + particles per group / group size), from the measured c2 figures
// (80 at theta = 0.75, 189 at theta = 0.5; c5: 334 at theta = 0.4) and the theta^-3 growth of the opened volume; only
// sizes the waves (with a factor 1.5 on top; a group that still finds no room goes to the fused kernel).
static double list_entries_per_particle(float theta) { return 24.0 / ((double)theta * theta * theta) + 16.0; }

constexpr int kPipeEvalBlocks = 3;    // evaluation blocks per SM while a list walk runs beside them (12 warps x 128 registers)
constexpr int kPipeListBlocks = 1;    // ... which leaves registers and shared memory for this many list blocks per SM

// Waves are contiguous particle ranges whose lists are expected to fit the list buffer; normally there is one.  By
// default the waves run one after the other on the caller's stream (list walk, evaluation, list walk, ...).
// bh_config.walk_waves = k > 1 asks for a two-stage PIPELINE over at least k waves instead: the list walk of wave w + 1
// runs BESIDE the evaluation of wave w (internal stream s_lists); the evaluations alternate between the caller's stream
// and s_eval2 so that the tail of one wave overlaps the head of the next; the list buffer is used in halves (wave
// parity), and the list walk of wave w + 2 waits for the evaluation of wave w.  Everything is joined back into the
// caller's stream with events: no host synchronisation, and the fork/join pattern can be captured into a CUDA graph.
// Measured on B200 (c2, bh_get_walk_timeline): the pipeline does overlap, but it does not pay -- 12 evaluation warps +
// 8 list warps per SM take 2.96 ms (8 waves) against 2.38 ms for one wave: the list walk is bound by instruction issue
// (~5800 warp instructions per group), so beside the evaluation it starves.  Hence opt-in.
int stage_walk(bh_ctx* c, float theta, float eps, cudaStream_t s) {
    if (c->timing) stage_mark(c, 8, s);
    int rc = BH_OK;
    if (!(c->rec_valid && c->rec_theta == theta && c->rec_mac == c->mac_kind)) rc = stage_cell_record(c, theta, s);   // else: written by S6
    if (rc != BH_OK) return rc;
    if (c->timing) stage_mark(c, 9, s);
    const bool fused_only = c->walk_mode == 1;
    c->walk_split_timed = false;
    // ---- waves: each must fit the list buffer (pipelined: half of it) 1.5 times over
    const bool pipelined = c->walk_waves > 1;            // bh_config.walk_waves: 0 = as few waves as the buffer allows, one after the other
    const double need = 1.5 * list_entries_per_particle(theta) * (double)c->n;
    int64_t nwaves = (int64_t)std::ceil((pipelined ? 2.0 : 1.0) * need / (double)c->list_entries);
    nwaves = std::max<int64_t>(nwaves, c->walk_waves);
    nwaves = std::min<int64_t>(nwaves, std::max<int64_t>(1, c->n / 4096));
    nwaves = std::max<int64_t>(1, std::min<int64_t>(nwaves, kMaxWaves));
    const int64_t wave_particles = div_up(c->n, nwaves);
    if ((rc = stage_walk_prepare(c, (int)nwaves, (uint32_t)wave_particles, s)) != BH_OK) return rc;
    if (!fused_only) {
        const int W = (int)nwaves;
        const uint32_t half = (uint32_t)std::min<int64_t>(c->list_entries / 2, (int64_t)1 << 30);
        // one block of eight warps per ~128 particles (~7 groups); alone on the device: 4 resident blocks per SM
        const int grid_alone = (int)std::max<int64_t>(1, std::min<int64_t>(div_up(wave_particles, 128), (int64_t)c->sm_count * 4));
        const int grid_beside = (int)std::max<int64_t>(1, std::min<int64_t>(div_up(wave_particles, 128), (int64_t)c->sm_count * kPipeListBlocks));
        if (!pipelined || W == 1) {
            // one wave after the other on the caller's stream; every wave has the whole list buffer and the whole device
            const uint32_t whole = (uint32_t)std::min<int64_t>(c->list_entries, (int64_t)1 << 30);
            for (int w = 0; w < W; ++w) {
                if ((rc = stage_walk_lists(c, w, grid_alone, 0u, whole, s)) != BH_OK) return rc;
                if (W == 1 && c->timing) stage_mark(c, 11, s);
                if ((rc = stage_walk_eval(c, w, eps, 99, true, s)) != BH_OK) return rc;
                if (W == 1 && c->timing) stage_mark(c, 12, s);
            }
            c->walk_split_timed = c->timing && W == 1;
        } else {
            cudaStream_t sl = c->s_lists, s2 = c->s_eval2;
            BH_CUDA(c, cudaEventRecord(c->ev_fork, s));
            BH_CUDA(c, cudaStreamWaitEvent(sl, c->ev_fork, 0));
            BH_CUDA(c, cudaStreamWaitEvent(s2, c->ev_fork, 0));
            for (int w = 0; w < W; ++w) {
                // lists of wave w (nothing runs beside wave 0: it gets the whole device)
                if (w >= 2) BH_CUDA(c, cudaStreamWaitEvent(sl, c->ev_eval[w - 2], 0));
                const int grid = (w == 0) ? grid_alone : grid_beside;
                if ((rc = stage_walk_lists(c, w, grid, (w & 1) ? half : 0u, half, sl)) != BH_OK) return rc;
                BH_CUDA(c, cudaEventRecord(c->ev_lists[w], sl));
                // evaluation of wave w
                cudaStream_t se = (w & 1) ? s2 : s;
                BH_CUDA(c, cudaStreamWaitEvent(se, c->ev_lists[w], 0));
                if ((rc = stage_walk_eval(c, w, eps, (w + 1 < W) ? kPipeEvalBlocks : 99, false, se)) != BH_OK) return rc;
                BH_CUDA(c, cudaEventRecord(c->ev_eval[w], se));
            }
            // join: the caller's stream continues after every evaluation (and with them every list walk)
            for (int w = std::max(0, W - 2); w < W; ++w)
                if (w & 1) BH_CUDA(c, cudaStreamWaitEvent(s, c->ev_eval[w], 0));
        }
    }
    const size_t smem = sizeof(WarpShared) * kWalkWarps;
    if (c->mac_kind == kMacMinDist)
        BH_LAUNCH(c, k_walk_fused<kMacMinDist>, c->sm_count * 2, kWalkThreads, smem, s, c->ws.sc, c->ws.ctl, fused_only ? 1 : 0, c->ws.deferred,
                  c->ws.pos[c->cur], c->ws.trec, c->ws.tlink, c->ws.box, c->ws.erec, c->ws.g_begin, eps * eps, c->ws.acc, c->ws.g_npc, c->ws.g_npp,
                  c->active ? c->ws.gflag : nullptr);
    else
        BH_LAUNCH(c, k_walk_fused<kMacEq1>, c->sm_count * 2, kWalkThreads, smem, s, c->ws.sc, c->ws.ctl, fused_only ? 1 : 0, c->ws.deferred,
                  c->ws.pos[c->cur], c->ws.trec, c->ws.tlink, c->ws.box, c->ws.erec, c->ws.g_begin, eps * eps, c->ws.acc, c->ws.g_npc, c->ws.g_npp,
                  c->active ? c->ws.gflag : nullptr);
    if (c->timing) stage_mark(c, 10, s);
    return BH_OK;
}

}  // namespace bh
