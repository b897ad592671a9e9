// walk_eval.cu -- S8: evaluation of the interaction lists written by walk_lists.cu.
//
// One warp owns one group at a time (groups are independent units of work) and pulls the next group from a
// device counter.  What differs from the paper's one-thread-per-particle sweep, and why:
//   (1) FP32 rate.  On sm_100a the register file delivers two 32-bit words per lane and cycle, so a three-operand FFMA
//       cannot issue every cycle; the packed forms FFMA2 / FMUL2 / FADD2 with a broadcast scalar operand need fewer words
//       per flop and come closest to the 128 FP32 lanes/clk/SM.  A 64-bit register here holds TWO
//       TARGETS (particles of the group); the list entry is a scalar operand that the packed instructions broadcast to
//       both halves (the `.F32` operand form of the SASS), so the records are used exactly as they sit in memory: no
//       pairing of entries, no transposition, no padding entry.
//   (2) Lane use.  A group holds ng <= 64 targets (mean ~19; work-weighted mean ~27).  A lane serves R = 2, 4 or 6
//       targets (R/2 packed registers per coordinate); L = ceil(ng / R) lanes cover the group, and the warp is split into
//       S = floor(32 / L) such teams, each sweeping every S-th entry of the list ("up to 4 threads per particle",
//       PAPER.md:81, 97, taken to its end).  R is chosen per group to maximise the useful lanes ng S / (32 R) (c2: 91 %).
//       The sums stay in registers for the whole group; the S partial sums per target are added once, through shared
//       memory, in a fixed order (deterministic).
//   (3) Shared-memory delivery.  An entry costs three LDS.128 per lane whatever R is, so R = 4 or 6 halves or thirds the
//       shared-memory traffic per interaction; R = 2 sweeps two entries per iteration for independent work instead.
//   (4) The lists are streamed in batches of 128 entries ("Nblock"): while batch b is swept, the records of
//       batch b + 1 and the indices of batch b + 2 are copied by cp.async (LDGSTS) into the other halves of two double
//       buffers; no register waits for a load across the sweep, and the L2 latency hides behind arithmetic.
// The group's own particles form the last batch, with j != i (A19).
// Forces: DESIGN.md O10 -- 33 packed operations + 2 MUFU.RSQ per entry and target pair (p-c), 13 + 2 (p-p).
#include <algorithm>
#include "walk_common.cuh"

namespace bh {

constexpr int kEvalWarps = 4;
constexpr int kEvalThreads = kEvalWarps * 32;
constexpr int kEvalBlocksPerSM = 4;          // 16 warps / SM at <= 128 registers
constexpr int kBatch = 128;                  // list entries per batch
constexpr int kPerLane = kBatch / 32;        // entries a lane gathers per batch

struct __align__(16) EvalShared {
    float4 buf[2][kBatch * 3];               // cp.async landing zones: 3 x float4 per cell, 1 x float4 per particle
    uint32_t idx[2][kBatch];                 // list indices of the next batches (cp.async as well)
    float tx[64], ty[64], tz[64];            // negated target coordinates: a lane reads its pairs with one 64-bit load each
};

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// The evaluation of one group with R = 2 * R2 targets per lane.  Batches: nbpc of accepted cells, nbpp of particles of
// opened leaves, then the group's own particles.
template <int R2>
__device__ __forceinline__ void eval_group(EvalShared* ws, const int lane, const uint32_t gb, const int ng, const float4* __restrict__ pos,
                                           const float4* __restrict__ erec, const uint32_t* __restrict__ lpc, const int npc,
                                           const uint32_t* __restrict__ lpp, const int npp, const Consts& k, float4* __restrict__ acc_out) {
    constexpr int R = 2 * R2;
    constexpr int U = R2 == 1 ? 2 : 1;           // entries per iteration: two independent chains per lane in every case but R2 = 3 (three)
    const int L = (ng + R - 1) / R, S = 32 / L;
    const int team = lane / L, tl = lane - team * L;
    const bool active = team < S;
    const int t0 = tl * R;                       // first target of this lane
    f2 ntx[R2], nty[R2], ntz[R2];
    Acc2 a[R2];
    // targets: staged through shared memory so that every packed pair arrives in an aligned register pair (one LDS.64)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int t = lane + 32 * h;
        const float4 P = __ldg(pos + gb + min(t, ng - 1));   // idle targets shadow the last particle
        ws->tx[t] = -P.x; ws->ty[t] = -P.y; ws->tz[t] = -P.z;
    }
    __syncwarp();
#pragma unroll
    for (int j = 0; j < R2; ++j) {
        const int t = min(t0 + 2 * j, 62);
        ntx[j] = *reinterpret_cast<const f2*>(ws->tx + t);
        nty[j] = *reinterpret_cast<const f2*>(ws->ty + t);
        ntz[j] = *reinterpret_cast<const f2*>(ws->tz + t);
        a[j].ax = a[j].ay = a[j].az = a[j].p = 0ull;
    }
    const int nbpc = (npc + kBatch - 1) / kBatch, nbpp = (npp + kBatch - 1) / kBatch;
    const int nb = nbpc + nbpp + 1;
    const int e0 = active ? team : (1 << 28);    // idle lanes (32 - S L of them) skip the sweeps

    auto batch_len = [&](int b) { return b < nbpc ? min(kBatch, npc - kBatch * b) : b < nbpc + nbpp ? min(kBatch, npp - kBatch * (b - nbpc)) : ng; };
    // copy the list indices of batch b (cells or particles; the self batch has none) into half b & 1 of the index buffer.
    // They travel by cp.async like the records, so no register waits for them: lane l fetches and later reads entries
    // l, l + 32, ... itself.
    auto fetch_idx = [&](int b) {
        if (b >= nbpc + nbpp) return;
        const uint32_t* src = b < nbpc ? lpc + b * kBatch : lpp + (b - nbpc) * kBatch;
        const int len = batch_len(b);
        uint32_t* dst = ws->idx[b & 1];
#pragma unroll
        for (int j = 0; j < kPerLane; ++j) {
            const int le = j * 32 + lane;
            if (le < len) cp_async4(dst + le, src + le);
        }
    };
    // gather the records of batch b into half b & 1 of the record buffer
    auto issue = [&](int b) {
        float4* dst = ws->buf[b & 1];
        const uint32_t* sidx = ws->idx[b & 1];
        const int len = batch_len(b);
        if (b < nbpc) {
#pragma unroll
            for (int j = 0; j < kPerLane; ++j) {
                const int le = j * 32 + lane;
                if (le < len) {
                    const float4* s = erec + 3 * (size_t)sidx[le];
                    float4* d = dst + 3 * le;
                    cp_async16(d, s); cp_async16(d + 1, s + 1); cp_async16(d + 2, s + 2);
                }
            }
        } else if (b < nbpc + nbpp) {
#pragma unroll
            for (int j = 0; j < kPerLane; ++j) {
                const int le = j * 32 + lane;
                if (le < len) cp_async16(dst + le, pos + sidx[le]);
            }
        } else {
#pragma unroll
            for (int j = 0; j < kPerLane; ++j) {
                const int le = j * 32 + lane;
                if (le < len) cp_async16(dst + le, pos + gb + le);
            }
        }
    };

    __syncwarp();                      // the previous group's reduction is done with the buffers
    fetch_idx(0);
    cp_async_commit();
    cp_async_wait_all();               // (the only index round trip that nothing hides: one per group)
    issue(0);
    fetch_idx(1);
    cp_async_commit();
    for (int b = 0; b < nb; ++b) {
        cp_async_wait_all();
        __syncwarp();                  // batch b (and the indices of b + 1) have landed; everyone is done sweeping batch b - 1
        if (b + 1 < nb) { issue(b + 1); fetch_idx(b + 2); cp_async_commit(); }
        const float4* buf = ws->buf[b & 1];
        const int len = batch_len(b);
        if (b < nbpc) {
            const float4* p = buf + 3 * min(e0, len);
            const float4* const end = buf + 3 * len;
            const int step = 3 * S;
            if (U == 2) {
                for (; p + step < end; p += 2 * step) {
                    const float4 v0 = p[0], v1 = p[1], v2 = p[2];
                    const float4 w0 = p[step], w1 = p[step + 1], w2 = p[step + 2];
#pragma unroll
                    for (int j = 0; j < R2; ++j) pc_bc(v0, v1, v2, ntx[j], nty[j], ntz[j], k, a[j]);
#pragma unroll
                    for (int j = 0; j < R2; ++j) pc_bc(w0, w1, w2, ntx[j], nty[j], ntz[j], k, a[j]);
                }
            }
            for (; p < end; p += step) {
                const float4 v0 = p[0], v1 = p[1], v2 = p[2];
#pragma unroll
                for (int j = 0; j < R2; ++j) pc_bc(v0, v1, v2, ntx[j], nty[j], ntz[j], k, a[j]);
            }
        } else if (b + 1 < nb) {
            const float4* p = buf + min(e0, len);
            const float4* const end = buf + len;
            for (; p + S < end; p += 2 * S) {
                const float4 v = p[0], w = p[S];
#pragma unroll
                for (int j = 0; j < R2; ++j) pp_bc<false>(v, ntx[j], nty[j], ntz[j], k, a[j], 0, 0, 0);
#pragma unroll
                for (int j = 0; j < R2; ++j) pp_bc<false>(w, ntx[j], nty[j], ntz[j], k, a[j], 0, 0, 0);
            }
            for (; p < end; p += S) {
                const float4 v = p[0];
#pragma unroll
                for (int j = 0; j < R2; ++j) pp_bc<false>(v, ntx[j], nty[j], ntz[j], k, a[j], 0, 0, 0);
            }
        } else {
            for (int e = e0; e < len; e += S) {
                const float4 v = buf[e];
#pragma unroll
                for (int j = 0; j < R2; ++j) pp_bc<true>(v, ntx[j], nty[j], ntz[j], k, a[j], e, t0 + 2 * j, ng);
            }
        }
    }
    __syncwarp();                      // every lane is done with the last batch
    // ---- add the S partial sums of every target in team order and store (ax, ay, az, phi)
    float4* red = ws->buf[0];
    const int mpad = L * R;
    if (active) {
#pragma unroll
        for (int j = 0; j < R2; ++j) {
            float xl, xh, yl, yh, zl, zh, pl, ph;
            upk(a[j].ax, xl, xh); upk(a[j].ay, yl, yh); upk(a[j].az, zl, zh); upk(a[j].p, pl, ph);
            red[team * mpad + t0 + 2 * j] = make_float4(xl, yl, zl, pl);
            red[team * mpad + t0 + 2 * j + 1] = make_float4(xh, yh, zh, ph);
        }
    }
    __syncwarp();
    for (int t = lane; t < ng; t += 32) {
        float4 r = red[t];
        for (int s = 1; s < S; ++s) {
            const float4 q = red[s * mpad + t];
            r.x += q.x; r.y += q.y; r.z += q.z; r.w += q.w;
        }
        acc_out[gb + t] = make_float4(r.x, r.y, r.z, -r.w);
    }
}

// Targets per lane (R = 2 R2) that maximise the useful lanes ng S / (32 R); ties go to the larger R (less shared-memory traffic).
__device__ __forceinline__ int choose_r2(int ng) {
    const int s1 = 32 / ((ng + 1) / 2), s2 = 32 / ((ng + 3) / 4), s3 = 32 / ((ng + 5) / 6);
    const int q1 = 6 * s1, q2 = 3 * s2, q3 = 2 * s3;
    if (q3 >= q2 && q3 >= q1) return 3;
    if (q2 >= q1) return 2;
    return 1;
}

__global__ void __launch_bounds__(kEvalThreads, kEvalBlocksPerSM) k_walk_eval(const DevScalars* __restrict__ sc, WalkCtl* __restrict__ ctl, int wave, const float4* __restrict__ pos,
                                                               const float4* __restrict__ erec, const uint32_t* __restrict__ g_begin,
                                                               const uint32_t* __restrict__ lists, const uint32_t* __restrict__ g_pcoff,
                                                               const uint32_t* __restrict__ g_npc, const uint32_t* __restrict__ g_ppoff,
                                                               const uint32_t* __restrict__ g_lpp, float eps2, float4* __restrict__ acc_out, int by_class) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    EvalShared* ws = reinterpret_cast<EvalShared*>(smem_raw) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    const uint32_t g0 = ctl->wave_g[wave], g1 = ctl->wave_g[wave + 1];
    const Consts k = make_consts(eps2);
    if (threadIdx.x == 0) atomicMin(&ctl->t_start[1][wave], global_ns());
    // three sweeps over the wave's groups with one counter: first the groups with more than 3 times the average work
    // (targets x list entries), then those above 1.5 times, then the rest -- the long groups start early and the kernel
    // ends on short ones (the order in which groups are evaluated does not touch their sums).  The class of a group must
    // be the same for every warp that looks at it, so `by_class` is only set when nothing adds to the interaction sums
    // while this kernel runs (one wave after the other); beside a concurrent list walk (pipelined waves) there is one sweep.
    const uint32_t G = g1 - g0;
    const uint32_t nsweeps = by_class ? 3u : 1u;
    const unsigned long long total = sc->sum_pc + sc->sum_pp;                 // interactions listed so far (all waves up to this one)
    const unsigned long long mean = total / max(sc->n_groups, 1u);
    for (;;) {
        uint32_t i = 0;
        if (lane == 0) i = atomicAdd(&ctl->eval_next[wave], 1u);
        i = __shfl_sync(0xFFFFFFFFu, i, 0);
        if (i >= nsweeps * G) break;
        const uint32_t sweep = i >= 2u * G ? 2u : i >= G ? 1u : 0u;
        const uint32_t g = g0 + (i - sweep * G);
        const uint32_t pcoff = __ldg(g_pcoff + g);
        if (pcoff >= kSkip) continue;          // deferred to the fused kernel (kNone) or not in this walk's subset (kSkip)
        const uint32_t gb = __ldg(g_begin + g), ge = __ldg(g_begin + g + 1);
        const int ng = (int)(ge - gb), npc = (int)__ldg(g_npc + g), npp = (int)__ldg(g_lpp + g);
        const unsigned long long work = (unsigned long long)ng * (unsigned long long)(npc + npp);
        const uint32_t cls = !by_class ? 0u : 2ull * work > 6ull * mean ? 0u : 2ull * work > 3ull * mean ? 1u : 2u;
        if (cls != sweep) continue;            // another sweep's
        const uint32_t* lpc = lists + pcoff;
        const uint32_t* lpp = lists + __ldg(g_ppoff + g);
        switch (choose_r2(ng)) {
            case 1: eval_group<1>(ws, lane, gb, ng, pos, erec, lpc, npc, lpp, npp, k, acc_out); break;
            case 2: eval_group<2>(ws, lane, gb, ng, pos, erec, lpc, npc, lpp, npp, k, acc_out); break;
            default: eval_group<3>(ws, lane, gb, ng, pos, erec, lpc, npc, lpp, npp, k, acc_out); break;
        }
        __syncwarp();
    }
    if (lane == 0) atomicMax(&ctl->t_end[1][wave], global_ns());
}

int walk_eval_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_eval, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(EvalShared) * kEvalWarps)));
    // the same (largest) shared-memory carve-out as k_walk_lists, so that blocks of both kernels can share an SM
    BH_CUDA(c, cudaFuncSetAttribute(k_walk_eval, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared));
    return walk_lists_init(c);
}

int stage_walk_eval(bh_ctx* c, int wave, float eps, int blocks_per_sm, bool by_class, cudaStream_t s) {
    const size_t smem = sizeof(EvalShared) * kEvalWarps;
    const int grid = c->sm_count * std::min(blocks_per_sm, kEvalBlocksPerSM);
    BH_LAUNCH(c, k_walk_eval, grid, kEvalThreads, smem, s, c->ws.sc, c->ws.ctl, wave, c->ws.pos[c->cur], c->ws.erec, c->ws.g_begin, c->ws.lists,
              c->ws.g_pcoff, c->ws.g_npc, c->ws.g_ppoff, c->ws.g_lpp, eps * eps, c->ws.acc, by_class ? 1 : 0);
    return BH_OK;
}

}  // namespace bh
