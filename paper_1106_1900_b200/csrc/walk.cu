// walk.cu -- S7 group tree-walk with the MAC of Eq.1 and S8 force evaluation, fused.
//
// One warp owns one group at a time (groups are independent units of work) and pulls the next group
// from a device counter.  Per group:
//   * frontier: a LIFO of cell indices in shared memory.  The paper walks breadth-first with two stacks (L83-87); the
//     interaction lists are SETS, so any traversal order produces the same lists and counts.  Depth-first popping of up
//     to 32 cells per step bounds the frontier: the pop width shrinks when the stack nears its capacity and a reserve
//     of 7 x 20 + slack entries always admits a pure depth-first descent, so the stack cannot overflow.
//   * each lane tests one cell:  d = distance from the group's tight box to the cell's centre of mass,
//     accept iff d^2 > r2open = (l/theta + delta)^2  (Eq.1), in exactly the fp32 operations of DESIGN.md O9.
//   * accepted cells are staged (48 B each) in a shared-memory ring; opened leaves contribute their particles (16 B each)
//     to a second ring; whenever a ring holds 32 entries every lane sweeps them for its own target particle(s)
//     ("each thread ... progresses over the data in the on-chip memory and accumulates partial interactions").
//   * the group's own particles are skipped while staging and handled by a final self block with j != i (A19).
// Forces: Plummer-softened p-p, and p-c with monopole + quadrupole (second-order expansion of the softened kernel,
// DESIGN.md O10).  fp32 FMA arithmetic + MUFU.RSQ; partial sums per 32-entry batch are added to the running totals.
#include <algorithm>
#include "bh_internal.cuh"

namespace bh {

constexpr int kWalkWarps = 8;
constexpr int kWalkThreads = kWalkWarps * 32;
constexpr int kStackCap = 1024;
constexpr int kStackReserve = 160;   // >= 7 * 20 + 7: room for a pure depth-first descent
constexpr int kRing = 64;            // ring capacity (entries), power of two, >= 63

struct __align__(16) WarpShared {
    float4 pc[kRing][3];             // (com.xyz, M) (1.5 Qxx, 1.5 Qyy, 1.5 Qzz, 1.5 Qxy) (1.5 Qxz, 1.5 Qyz, -T/2, -3T/2)
    float4 pp[kRing];                // (x, y, z, m)
    uint32_t stack[kStackCap];
    uint32_t run_begin[32];
    uint32_t run_off[36];
};

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ int warp_excl_scan(int v, int lane, int& total) {
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    total = __shfl_sync(0xFFFFFFFFu, inc, 31);
    return inc - v;
}

struct Acc4 { float x, y, z, p; };   // acceleration and MINUS the potential

// p-c: 36 fp32 operations + 1 rsqrt per interaction.  Staged values: M, Q'' = 1.5 Q, nTh = -T/2, n3Th = -3T/2.
//   -phi += M/rho + nTh/rho^3 + w''/rho^5,          w'' = dr.Q''.dr = 1.5 w
//   a    += dr (M/rho^3 + n3Th/rho^5 + 5 w''/rho^7) - 2 q''/rho^5,   q'' = Q'' dr = 1.5 q
template <int NT>
__device__ __forceinline__ void eval_pc(const WarpShared* ws, int head, int count, const float (&tx)[NT], const float (&ty)[NT],
                                        const float (&tz)[NT], Acc4 (&acc)[NT], float eps2) {
    Acc4 loc[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) loc[t] = Acc4{0.f, 0.f, 0.f, 0.f};
#pragma unroll 4
    for (int j = 0; j < count; ++j) {
        const int e = (head + j) & (kRing - 1);
        const float4 a = ws->pc[e][0], b = ws->pc[e][1], c = ws->pc[e][2];
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const float dx = a.x - tx[t], dy = a.y - ty[t], dz = a.z - tz[t];
            const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
            const float ri = rsqrt_approx(r2);
            const float ri2 = ri * ri, ri3 = ri * ri2, ri5 = ri3 * ri2, ri7 = ri5 * ri2;
            const float qx = fmaf(b.x, dx, fmaf(b.w, dy, c.x * dz));
            const float qy = fmaf(b.w, dx, fmaf(b.y, dy, c.y * dz));
            const float qz = fmaf(c.x, dx, fmaf(c.y, dy, b.z * dz));
            const float w = fmaf(dx, qx, fmaf(dy, qy, dz * qz));
            loc[t].p = fmaf(a.w, ri, fmaf(c.z, ri3, fmaf(w, ri5, loc[t].p)));
            const float br = fmaf(5.0f * w, ri7, fmaf(c.w, ri5, a.w * ri3));
            const float c5 = -2.0f * ri5;
            loc[t].x = fmaf(qx, c5, fmaf(dx, br, loc[t].x));
            loc[t].y = fmaf(qy, c5, fmaf(dy, br, loc[t].y));
            loc[t].z = fmaf(qz, c5, fmaf(dz, br, loc[t].z));
        }
    }
#pragma unroll
    for (int t = 0; t < NT; ++t) { acc[t].x += loc[t].x; acc[t].y += loc[t].y; acc[t].z += loc[t].z; acc[t].p += loc[t].p; }
}

// p-p: 13 fp32 operations + 1 rsqrt.  kSelf: sources are the group's own particles; entry j is target index j (skip j == i).
template <int NT, bool kSelf>
__device__ __forceinline__ void eval_pp(const WarpShared* ws, int head, int count, const float (&tx)[NT], const float (&ty)[NT],
                                        const float (&tz)[NT], Acc4 (&acc)[NT], float eps2, int lane) {
    Acc4 loc[NT];
#pragma unroll
    for (int t = 0; t < NT; ++t) loc[t] = Acc4{0.f, 0.f, 0.f, 0.f};
#pragma unroll 4
    for (int j = 0; j < count; ++j) {
        const float4 s = ws->pp[(head + j) & (kRing - 1)];
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const float dx = s.x - tx[t], dy = s.y - ty[t], dz = s.z - tz[t];
            const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
            float ri = rsqrt_approx(r2);
            if (kSelf) ri = (j == lane + 32 * t) ? 0.0f : ri;
            const float ri2 = ri * ri;
            const float mr = s.w * ri;
            const float mr3 = mr * ri2;
            loc[t].p += mr;
            loc[t].x = fmaf(dx, mr3, loc[t].x);
            loc[t].y = fmaf(dy, mr3, loc[t].y);
            loc[t].z = fmaf(dz, mr3, loc[t].z);
        }
    }
#pragma unroll
    for (int t = 0; t < NT; ++t) { acc[t].x += loc[t].x; acc[t].y += loc[t].y; acc[t].z += loc[t].z; acc[t].p += loc[t].p; }
}

template <int NT>
__device__ __forceinline__ void walk_group(WarpShared* ws, const int lane, const uint32_t g, const uint32_t gb, const uint32_t ge,
                                           const float4* __restrict__ pos, const float4* __restrict__ rec, float eps2,
                                           float4* __restrict__ acc_out, uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp,
                                           DevScalars* sc) {
    const uint32_t lt = (1u << lane) - 1u;
    const int ng = (int)(ge - gb);
    float tx[NT], ty[NT], tz[NT];
    Acc4 acc[NT];
    float4 tp[NT];
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const int idx = lane + 32 * t;
        tp[t] = pos[gb + min(idx, ng - 1)];          // idle lanes shadow the last particle (results discarded)
        tx[t] = tp[t].x; ty[t] = tp[t].y; tz[t] = tp[t].z;
        acc[t] = Acc4{0.f, 0.f, 0.f, 0.f};
        mn[0] = fminf(mn[0], tx[t]); mx[0] = fmaxf(mx[0], tx[t]);
        mn[1] = fminf(mn[1], ty[t]); mx[1] = fmaxf(mx[1], ty[t]);
        mn[2] = fminf(mn[2], tz[t]); mx[2] = fmaxf(mx[2], tz[t]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            mn[k] = fminf(mn[k], __shfl_xor_sync(0xFFFFFFFFu, mn[k], o));
            mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xFFFFFFFFu, mx[k], o));
        }

    int sp = 1;
    if (lane == 0) ws->stack[0] = 0u;   // the root (A17)
    __syncwarp();
    int pc_head = 0, pc_cnt = 0, pp_head = 0, pp_cnt = 0;
    uint32_t npc = 0, npp = 0, nmac = 0;

    while (sp > 0) {
        int k = (kStackCap - kStackReserve - sp) / 7;
        k = max(1, min(k, 32));
        k = min(k, sp);
        const bool valid = lane < k;
        uint32_t cell = 0;
        if (valid) cell = ws->stack[sp - 1 - lane];
        sp -= k;
        nmac += (uint32_t)k;
        __syncwarp();
        bool accept = false, isleaf = false, isnode = false;
        float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f);
        uint32_t first = 0, cnt = 0;
        if (valid) {
            r0 = __ldg(rec + 4 * (size_t)cell);
            const float dx = fmaxf(fmaxf(__fsub_rn(mn[0], r0.x), __fsub_rn(r0.x, mx[0])), 0.0f);
            const float dy = fmaxf(fmaxf(__fsub_rn(mn[1], r0.y), __fsub_rn(r0.y, mx[1])), 0.0f);
            const float dz = fmaxf(fmaxf(__fsub_rn(mn[2], r0.z), __fsub_rn(r0.z, mx[2])), 0.0f);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            accept = d2 > r0.w;
            if (!accept) {
                const float4 l = __ldg(rec + 4 * (size_t)cell + 3);
                first = __float_as_uint(l.x);
                cnt = __float_as_uint(l.y);
                isleaf = __float_as_uint(l.z) != 0u;
                isnode = !isleaf;
            }
        }
        // ---- accepted cells -> p-c ring
        const uint32_t amask = __ballot_sync(0xFFFFFFFFu, accept);
        if (amask) {
            if (accept) {
                const float4 r1 = __ldg(rec + 4 * (size_t)cell + 1), r2 = __ldg(rec + 4 * (size_t)cell + 2);
                const float T = (r1.y + r1.z) + r1.w;
                const int slot = (pc_head + pc_cnt + __popc(amask & lt)) & (kRing - 1);
                ws->pc[slot][0] = make_float4(r0.x, r0.y, r0.z, r1.x);
                ws->pc[slot][1] = make_float4(1.5f * r1.y, 1.5f * r1.z, 1.5f * r1.w, 1.5f * r2.x);
                ws->pc[slot][2] = make_float4(1.5f * r2.y, 1.5f * r2.z, -0.5f * T, -1.5f * T);
            }
            const int na = __popc(amask);
            pc_cnt += na;
            npc += (uint32_t)na;
            __syncwarp();
            if (pc_cnt >= 32) {
                eval_pc<NT>(ws, pc_head, 32, tx, ty, tz, acc, eps2);
                pc_head = (pc_head + 32) & (kRing - 1);
                pc_cnt -= 32;
                __syncwarp();
            }
        }
        // ---- opened leaves -> p-p ring (own particles skipped)
        const uint32_t lmask = __ballot_sync(0xFFFFFFFFu, isleaf);
        if (lmask) {
            int total;
            const int off = warp_excl_scan(isleaf ? (int)cnt : 0, lane, total);
            npp += (uint32_t)total;
            const int nl = __popc(lmask);
            if (isleaf) {
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
                    int lo = 0, hi = nl - 1;
                    while (lo < hi) {
                        const int mid = (lo + hi + 1) >> 1;
                        if ((int)ws->run_off[mid] <= t) lo = mid; else hi = mid - 1;
                    }
                    src = ws->run_begin[lo] + (uint32_t)(t - (int)ws->run_off[lo]);
                    keep = !(src >= gb && src < ge);
                }
                const uint32_t kmask = __ballot_sync(0xFFFFFFFFu, keep);
                if (keep) ws->pp[(pp_head + pp_cnt + __popc(kmask & lt)) & (kRing - 1)] = __ldg(pos + src);
                pp_cnt += __popc(kmask);
                __syncwarp();
                if (pp_cnt >= 32) {
                    eval_pp<NT, false>(ws, pp_head, 32, tx, ty, tz, acc, eps2, lane);
                    pp_head = (pp_head + 32) & (kRing - 1);
                    pp_cnt -= 32;
                    __syncwarp();
                }
            }
            __syncwarp();
        }
        // ---- opened nodes -> children onto the stack
        const uint32_t nmask = __ballot_sync(0xFFFFFFFFu, isnode);
        if (nmask) {
            int total;
            const int off = warp_excl_scan(isnode ? (int)cnt : 0, lane, total);
            if (sp + total > kStackCap) {            // cannot happen (see header); never write out of bounds
                if (lane == 0) atomicMin(&sc->status, (int)BH_ERR_CAPACITY);
                sp = 0;
                break;
            }
            if (isnode)
                for (uint32_t j = 0; j < cnt; ++j) ws->stack[sp + off + (int)j] = first + j;
            sp += total;
            __syncwarp();
        }
    }
    // ---- flush the rings
    if (pc_cnt > 0) eval_pc<NT>(ws, pc_head, pc_cnt, tx, ty, tz, acc, eps2);
    if (pp_cnt > 0) eval_pp<NT, false>(ws, pp_head, pp_cnt, tx, ty, tz, acc, eps2, lane);
    __syncwarp();
    // ---- self block: the group's own particles, j != i
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) ws->pp[idx] = tp[t];
    }
    __syncwarp();
    eval_pp<NT, true>(ws, 0, ng, tx, ty, tz, acc, eps2, lane);
    __syncwarp();
#pragma unroll
    for (int t = 0; t < NT; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) acc_out[gb + idx] = make_float4(acc[t].x, acc[t].y, acc[t].z, -acc[t].p);
    }
    if (lane == 0) {
        g_npc[g] = npc;
        g_npp[g] = npp;
        atomicAdd(&sc->sum_pc, (unsigned long long)npc * (unsigned long long)ng);
        atomicAdd(&sc->sum_pp, (unsigned long long)npp * (unsigned long long)ng);
        atomicAdd(&sc->sum_mac, (unsigned long long)nmac);
    }
}

__global__ void __launch_bounds__(kWalkThreads, 2) k_walk(DevScalars* sc, const float4* __restrict__ pos, const float4* __restrict__ rec,
                                                          const uint32_t* __restrict__ g_begin, float eps2, float4* __restrict__ acc_out,
                                                          uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpShared* ws = reinterpret_cast<WarpShared*>(smem_raw) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    const uint32_t ngroups = sc->n_groups;
    for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(&sc->walk_next, 1u);
        g = __shfl_sync(0xFFFFFFFFu, g, 0);
        if (g >= ngroups) break;
        const uint32_t gb = __ldg(g_begin + g), ge = __ldg(g_begin + g + 1);
        if (ge - gb <= 32u)
            walk_group<1>(ws, lane, g, gb, ge, pos, rec, eps2, acc_out, g_npc, g_npp, sc);
        else
            walk_group<2>(ws, lane, g, gb, ge, pos, rec, eps2, acc_out, g_npc, g_npp, sc);
        __syncwarp();
    }
}

__global__ void k_reset_counters(DevScalars* sc) {
    if (threadIdx.x == 0) { sc->walk_next = 0; sc->sum_pc = 0; sc->sum_pp = 0; sc->sum_mac = 0; }
}

int walk_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_walk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(WarpShared) * kWalkWarps)));
    return BH_OK;
}

int stage_walk(bh_ctx* c, float theta, float eps, cudaStream_t s) {
    if (c->timing) cudaEventRecord(c->ev[8], s);
    int rc = stage_cell_record(c, theta, s);
    if (rc != BH_OK) return rc;
    BH_LAUNCH(c, k_reset_counters, 1, 32, 0, s, c->ws.sc);
    if (c->timing) cudaEventRecord(c->ev[9], s);
    const size_t smem = sizeof(WarpShared) * kWalkWarps;
    const int grid = c->sm_count * 2;
    BH_LAUNCH(c, k_walk, grid, kWalkThreads, smem, s, c->ws.sc, c->ws.pos[c->cur], c->ws.rec, c->ws.g_begin, eps * eps, c->ws.acc,
              c->ws.g_npc, c->ws.g_npp);
    if (c->timing) cudaEventRecord(c->ev[10], s);
    return BH_OK;
}

}  // namespace bh
