// walk_eval.cu -- S8: evaluation of the interaction lists written by walk_lists.cu.
//
// One warp owns one group at a time (groups are independent units of work) and pulls the next group from a
// device counter.  The lists are streamed in batches of 128 entries ("Nblock"):
//   * the indices of batch b + 2 are loaded while the records of batch b + 1 are in flight and batch b is evaluated;
//   * records (48 B per accepted cell, 16 B per particle) are gathered with cp.async (LDGSTS) straight into a raw
//     shared-memory buffer -- no registers are held across the sweep, and the gather's L2 latency hides behind arithmetic;
//   * the raw records are then transposed into the pair-interleaved ring the packed FFMA2 sweep reads
//     (walk_common.cuh): entry p is paired with entry p + ceil(k/2) of a batch of k, an odd tail gets a massless partner.
// The group's own particles form the last, "self" block with j != i (A19).
#include <algorithm>
#include "walk_common.cuh"

namespace bh {

constexpr int kEvalWarps = 4;
constexpr int kEvalThreads = kEvalWarps * 32;
constexpr int kEvalBlocksPerSM = 3;          // 12 warps / SM at up to 168 registers: few, fat warps (two pairs in flight per lane)
constexpr int kBatch = 128;                  // list entries per sweep
constexpr int kBatchPairs = kBatch / 2;
constexpr int kPerLane = kBatch / 32;        // entries a lane gathers per batch

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

struct Idx { uint32_t v[kPerLane]; };

// A list (kPc: accepted cells, 48 B records; else: particles, 16 B) is streamed through raw -> ring -> sweep.
template <bool kPc>
__device__ __forceinline__ void load_idx(const uint32_t* __restrict__ list, int n, int b, int lane, Idx& ix) {
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const int e = b * kBatch + j * 32 + lane;
        if (e < n) ix.v[j] = __ldg(list + e);
    }
}
template <bool kPc>
__device__ __forceinline__ void issue(EvalShared* ws, const float4* __restrict__ src, int n, int b, int lane, const Idx& ix) {
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const int le = j * 32 + lane;
        if (b * kBatch + le < n) {
            if (kPc) {
                const float4* s = src + 3 * (size_t)ix.v[j];
                float4* d = ws->raw + 3 * le;
                cp_async16(d, s); cp_async16(d + 1, s + 1); cp_async16(d + 2, s + 2);
            } else {
                cp_async16(ws->raw + le, src + ix.v[j]);
            }
        }
    }
    cp_async_commit();
}
// raw -> ring: pair p = (entry p, entry p + h) of a batch of len entries, h = ceil(len / 2); an odd tail gets a massless
// partner at its own position (a position no target can coincide with).
template <bool kPc>
__device__ __forceinline__ void transpose(EvalShared* ws, int len, int h, int lane) {
#pragma unroll
    for (int j = 0; j < kBatchPairs / 32; ++j) {
        const int p = j * 32 + lane;
        if (p < h) {
            const bool two = p + h < len;
            if (kPc) {
                const float4* a = ws->raw + 3 * p;
                const float4* b = ws->raw + 3 * (p + h);
                const float4 a0 = a[0], a1 = a[1], a2 = a[2];
                float4 b0 = make_float4(a0.x, a0.y, a0.z, 0.f), b1 = make_float4(0.f, 0.f, 0.f, 0.f), b2 = b1;
                if (two) { b0 = b[0]; b1 = b[1]; b2 = b[2]; }
                float4* d = reinterpret_cast<float4*>(ws->ring + p * kPcPair);
                d[0] = make_float4(a0.x, b0.x, a0.y, b0.y);
                d[1] = make_float4(a0.z, b0.z, a0.w, b0.w);
                d[2] = make_float4(a1.x, b1.x, a1.y, b1.y);
                d[3] = make_float4(a1.z, b1.z, a1.w, b1.w);
                d[4] = make_float4(a2.x, b2.x, a2.y, b2.y);
                d[5] = make_float4(a2.z, b2.z, a2.w, b2.w);
            } else {
                const float4 a0 = ws->raw[p];
                float4 b0 = make_float4(a0.x, a0.y, a0.z, 0.f);
                if (two) b0 = ws->raw[p + h];
                float4* d = reinterpret_cast<float4*>(ws->ring + p * kPpPair);
                d[0] = make_float4(a0.x, b0.x, a0.y, b0.y);
                d[1] = make_float4(a0.z, b0.z, a0.w, b0.w);
            }
        }
    }
}

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
    const int nbpc = (npc + kBatch - 1) / kBatch, nbpp = (npp + kBatch - 1) / kBatch;

    Idx ix, ixp;
    load_idx<true>(lpc, npc, 0, lane, ix);
    load_idx<false>(lpp, npp, 0, lane, ixp);
    __syncwarp();                      // `own`, `tot` visible; the previous group's sweeps are done with ring / raw
    if (nbpc > 0) issue<true>(ws, erec, npc, 0, lane, ix); else issue<false>(ws, pos, npp, 0, lane, ixp);
    load_idx<true>(lpc, npc, 1, lane, ix);
    // ---- accepted cells
    for (int b = 0; b < nbpc; ++b) {
        const int len = min(kBatch, npc - kBatch * b), h = (len + 1) >> 1;
        cp_async_wait_all();
        __syncwarp();
        transpose<true>(ws, len, h, lane);
        __syncwarp();
        // request the next batch, then sweep this one while those copies are in flight
        if (b + 1 < nbpc) { issue<true>(ws, erec, npc, b + 1, lane, ix); load_idx<true>(lpc, npc, b + 2, lane, ix); }
        else issue<false>(ws, pos, npp, 0, lane, ixp);
        eval_pc_all<kBatchPairs, false, true>(ws->ring, ws->own, ws->tot, 0, h, m, ng, k, lane);
        __syncwarp();
    }
    // ---- particles of opened leaves
    if (nbpp > 1) load_idx<false>(lpp, npp, 1, lane, ixp);
    for (int b = 0; b < nbpp; ++b) {
        const int len = min(kBatch, npp - kBatch * b), h = (len + 1) >> 1;
        cp_async_wait_all();
        __syncwarp();
        transpose<false>(ws, len, h, lane);
        __syncwarp();
        if (b + 1 < nbpp) { issue<false>(ws, pos, npp, b + 1, lane, ixp); load_idx<false>(lpp, npp, b + 2, lane, ixp); }
        eval_pp_all<false, kBatchPairs, false>(ws->ring, ws->own, ws->tot, 0, h, m, ng, k, lane);
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
    eval_pp_all<true, kBatchPairs, false>(ws->ring, ws->own, ws->tot, 0, (ng + 1) >> 1, m, ng, k, lane);
    __syncwarp();
    totals_finish(ws->tot, m, lane, ng, gb, acc_out);
    __syncwarp();
}

__global__ void __launch_bounds__(kEvalThreads, kEvalBlocksPerSM) k_walk_eval(WalkCtl* __restrict__ ctl, int wave, const float4* __restrict__ pos,
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
    const int grid = c->sm_count * kEvalBlocksPerSM;
    BH_LAUNCH(c, k_walk_eval, grid, kEvalThreads, smem, s, c->ws.ctl, wave, c->ws.pos[c->cur], c->ws.erec, c->ws.g_begin, c->ws.lists,
              c->ws.g_pcoff, c->ws.g_npc, c->ws.g_ppoff, c->ws.g_lpp, eps * eps, c->ws.acc);
    return BH_OK;
}

}  // namespace bh
