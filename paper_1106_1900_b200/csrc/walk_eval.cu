// walk_eval.cu -- S8: evaluation of the interaction lists written by walk_lists.cu.
//
// One warp owns one group at a time (groups are independent units of work) and pulls the next group from a
// device counter.  The lists are streamed in batches of 64 entries ("Nblock"):
//   * the indices of batch b + 2 are loaded while the records of batch b + 1 are in flight and batch b is evaluated;
//   * records (48 B per accepted cell, 16 B per particle) are gathered with cp.async (LDGSTS) straight into a raw
//     shared-memory buffer -- no registers are held across the sweep, and the gather's L2 latency hides behind arithmetic;
//   * the raw records are then transposed into the pair-interleaved ring the packed FFMA2 sweep reads
//     (walk_common.cuh): entry p is paired with entry p + ceil(k/2) of a batch of k, an odd tail gets a massless partner.
// The group's own particles form the last, "self" block with j != i (A19).
#include <algorithm>
#include "walk_common.cuh"

namespace bh {

constexpr int kEvalWarps = 8;
constexpr int kEvalThreads = kEvalWarps * 32;
constexpr int kBatch = 64;                   // list entries per sweep
constexpr int kBatchPairs = kBatch / 2;

struct __align__(16) EvalShared {
    float ring[kBatchPairs * kPcPair];       // pair-interleaved operands of the current batch (p-c: 112 B / pair; p-p: 32 B / pair)
    float4 raw[kBatch * 3];                  // cp.async landing zone: 3 x float4 per cell, 1 x float4 per particle
    float4 own[64];                          // the group's particles (targets; sources of the self block)
    SlotTotals tot[kMaxSlots];
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void eval_group(EvalShared* ws, const int lane, const uint32_t gb, const int ng, const float4* __restrict__ pos,
                                           const float4* __restrict__ erec, const uint32_t* __restrict__ lpc, const int npc,
                                           const uint32_t* __restrict__ lpp, const int npp, const Consts& k, float4* __restrict__ acc_out) {
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) ws->own[idx] = __ldg(pos + gb + idx);
    }
    const int m = (ng + 3) & ~3;
    totals_clear(ws->tot, lane);

    const int nbpc = (npc + kBatch - 1) / kBatch, nbt = nbpc + (npp + kBatch - 1) / kBatch;
    // batch bi: p-c batches first, then p-p batches
    auto batch_len = [&](int bi) { return bi < nbpc ? min(kBatch, npc - kBatch * bi) : min(kBatch, npp - kBatch * (bi - nbpc)); };
    auto load_idx = [&](int bi, uint32_t& i0, uint32_t& i1) {
        if (bi >= nbt) return;
        const uint32_t* src = bi < nbpc ? lpc + kBatch * bi : lpp + kBatch * (bi - nbpc);
        const int len = batch_len(bi);
        if (lane < len) i0 = __ldg(src + lane);
        if (lane + 32 < len) i1 = __ldg(src + lane + 32);
    };
    auto issue = [&](int bi, uint32_t i0, uint32_t i1) {
        if (bi < nbt) {
            const int len = batch_len(bi);
            if (bi < nbpc) {
                if (lane < len) {
                    const float4* s = erec + 3 * (size_t)i0;
                    float4* d = ws->raw + 3 * lane;
                    cp_async16(d, s); cp_async16(d + 1, s + 1); cp_async16(d + 2, s + 2);
                }
                if (lane + 32 < len) {
                    const float4* s = erec + 3 * (size_t)i1;
                    float4* d = ws->raw + 3 * (lane + 32);
                    cp_async16(d, s); cp_async16(d + 1, s + 1); cp_async16(d + 2, s + 2);
                }
            } else {
                if (lane < len) cp_async16(ws->raw + lane, pos + i0);
                if (lane + 32 < len) cp_async16(ws->raw + lane + 32, pos + i1);
            }
        }
        cp_async_commit();
    };

    uint32_t i0 = 0, i1 = 0;
    load_idx(0, i0, i1);
    __syncwarp();                      // `own`, `tot` visible; the previous group's sweeps are done with ring / raw
    issue(0, i0, i1);
    load_idx(1, i0, i1);
    for (int bi = 0; bi < nbt; ++bi) {
        const int len = batch_len(bi), h = (len + 1) >> 1;
        cp_async_wait_all();
        __syncwarp();
        // ---- transpose raw -> ring: pair p = (entry p, entry p + h)
        if (lane < h) {
            const bool two = lane + h < len;
            if (bi < nbpc) {
                const float4* a = ws->raw + 3 * lane;
                const float4* b = ws->raw + 3 * (lane + h);
                const float4 a0 = a[0], a1 = a[1], a2 = a[2];
                float4 b0 = make_float4(a0.x, a0.y, a0.z, 0.f), b1 = make_float4(0.f, 0.f, 0.f, 0.f), b2 = b1;
                if (two) { b0 = b[0]; b1 = b[1]; b2 = b[2]; }
                float4* d = reinterpret_cast<float4*>(ws->ring + lane * kPcPair);
                d[0] = make_float4(a0.x, b0.x, a0.y, b0.y);
                d[1] = make_float4(a0.z, b0.z, a0.w, b0.w);
                d[2] = make_float4(a1.x, b1.x, a1.y, b1.y);
                d[3] = make_float4(a1.z, b1.z, a1.w, b1.w);
                d[4] = make_float4(a2.x, b2.x, a2.y, b2.y);
                d[5] = make_float4(a2.z, b2.z, a2.w, b2.w);
            } else {
                const float4 a0 = ws->raw[lane];
                float4 b0 = make_float4(a0.x, a0.y, a0.z, 0.f);
                if (two) b0 = ws->raw[lane + h];
                float4* d = reinterpret_cast<float4*>(ws->ring + lane * kPpPair);
                d[0] = make_float4(a0.x, b0.x, a0.y, b0.y);
                d[1] = make_float4(a0.z, b0.z, a0.w, b0.w);
            }
        }
        __syncwarp();
        // ---- request the next batch, then sweep this one while those copies are in flight
        issue(bi + 1, i0, i1);
        load_idx(bi + 2, i0, i1);
        if (bi < nbpc) eval_pc_all<kBatchPairs>(ws->ring, ws->own, ws->tot, 0, h, m, ng, k, lane);
        else eval_pp_all<false, kBatchPairs>(ws->ring, ws->own, ws->tot, 0, h, m, ng, k, lane);
        __syncwarp();
    }
    cp_async_wait_all();
    // ---- self block: the group's own particles, entry j = target index j, j != i
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) { const float4 p = ws->own[idx]; pp_store(ws->ring, idx, p.x, p.y, p.z, p.w); }
    }
    if ((ng & 1) && lane == 0) { const float4 p = ws->own[ng - 1]; pp_store(ws->ring, ng, p.x, p.y, p.z, 0.f); }
    __syncwarp();
    eval_pp_all<true, kBatchPairs>(ws->ring, ws->own, ws->tot, 0, (ng + 1) >> 1, m, ng, k, lane);
    __syncwarp();
    totals_finish(ws->tot, m, lane, ng, gb, acc_out);
    __syncwarp();
}

__global__ void __launch_bounds__(kEvalThreads, 2) k_walk_eval(WalkCtl* __restrict__ ctl, int wave, const float4* __restrict__ pos,
                                                               const float4* __restrict__ erec, const uint32_t* __restrict__ g_begin,
                                                               const uint32_t* __restrict__ lists, const uint32_t* __restrict__ g_pcoff,
                                                               const uint32_t* __restrict__ g_npc, const uint32_t* __restrict__ g_ppoff,
                                                               const uint32_t* __restrict__ g_lpp, float eps2, float4* __restrict__ acc_out) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvalShared* ws = reinterpret_cast<EvalShared*>(smem_raw) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    const uint32_t g0 = ctl->wave_g[wave], g1 = ctl->wave_g[wave + 1];
    const Consts k = make_consts(eps2);
    for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = g0 + atomicAdd(&ctl->eval_next[wave], 1u);
        g = __shfl_sync(0xFFFFFFFFu, g, 0);
        if (g >= g1) break;
        const uint32_t pcoff = __ldg(g_pcoff + g);
        if (pcoff == kNone) continue;          // deferred to the fused kernel
        const uint32_t gb = __ldg(g_begin + g), ge = __ldg(g_begin + g + 1);
        eval_group(ws, lane, gb, (int)(ge - gb), pos, erec, lists + pcoff, (int)__ldg(g_npc + g), lists + __ldg(g_ppoff + g),
                   (int)__ldg(g_lpp + g), k, acc_out);
    }
}

int walk_eval_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_eval, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(EvalShared) * kEvalWarps)));
    return BH_OK;
}

int stage_walk_eval(bh_ctx* c, int wave, float eps, cudaStream_t s) {
    const size_t smem = sizeof(EvalShared) * kEvalWarps;
    const int grid = c->sm_count * 2;
    BH_LAUNCH(c, k_walk_eval, grid, kEvalThreads, smem, s, c->ws.ctl, wave, c->ws.pos[c->cur], c->ws.erec, c->ws.g_begin, c->ws.lists,
              c->ws.g_pcoff, c->ws.g_npc, c->ws.g_ppoff, c->ws.g_lpp, eps * eps, c->ws.acc);
    return BH_OK;
}

}  // namespace bh
