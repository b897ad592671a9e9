// blockstep.cu -- block time-steps ("time-step calculation ... on the GPU", 105 "... or on a subset of
// particles in case of the block-time step regime", 264-266), in the reading A29 of DESIGN.md.
//
// Every particle i carries (x_i, v_i, a_i) at its own time t_i = tick_i dt_max / 2^R and a step dt_i = dt_max / 2^rung_i.
// One system step (bh_block_step):
//   k_block_next      tick_next = min_i (tick_i + 2^(R - rung_i))
//   k_block_predict   active_i = (tick_i + step_i == tick_next); the active particles are predicted:
//                     x = fmaf(a, (h/2) h, fmaf(v, h, x)), h = dt_i           (the leapfrog predictor of Hut et al., L105)
//   S6 on the existing cells, only where an active particle sits below (L266) -- or S0-S6 when the caller asks for a
//   rebuild, after which k_block_permute makes the block state follow the sort
//   S7 + S8 of the groups with an active particle (L264)
//   k_block_correct   v = fmaf(a_old + a_new, h/2, v); a_i = a_new; tick_i = tick_next; new rung from
//                     tau = eta sqrt(len / |a|): the smallest r with dt_max / 2^r <= tau that the time allows
//   k_block_degrade   sum of the interactions of the walked groups now / when each was first walked on these cells:
//                     the caller rebuilds when the ratio has grown (L266 "a considerable decline in performance")
// All arithmetic in single fp32 operations, as the oracle states them (orc_rungs, orc_block_*).
#include <algorithm>
#include <cstddef>
#include "bh_internal.cuh"

namespace bh {

__device__ __forceinline__ uint8_t rung_of(float4 a, float len, float eta, float dt_max, int R, int lowest) {
    const float a2 = __fmaf_rn(a.z, a.z, __fmaf_rn(a.y, a.y, __fmul_rn(a.x, a.x)));
    const float amag = __fsqrt_rn(a2);
    const float tau = __fmul_rn(eta, __fsqrt_rn(__fdiv_rn(len, amag)));     // |a| = 0: +inf
    int r = 0;
    while (r < R && !(ldexpf(dt_max, -r) <= tau)) ++r;
    return (uint8_t)max(r, lowest);
}

__global__ void __launch_bounds__(256) k_block_init(const float4* __restrict__ acc, int n, float len, float eta, float dt_max, int R,
                                                    float4* __restrict__ accb, uint32_t* __restrict__ tick, uint8_t* __restrict__ rung,
                                                    uint32_t* __restrict__ g_base, DevScalars* sc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { sc->tick_next[0] = 0xFFFFFFFFu; sc->tick_next[1] = 0xFFFFFFFFu; sc->n_active = 0; sc->deg_now = 0; sc->deg_base = 0; }
    if (i >= n) return;
    const float4 a = acc[i];
    accb[i] = a;
    tick[i] = 0u;
    rung[i] = rung_of(a, len, eta, dt_max, R, 0);
    g_base[i] = 0u;
}

__global__ void __launch_bounds__(256) k_block_next(const uint32_t* __restrict__ tick, const uint8_t* __restrict__ rung, int n, int R,
                                                    uint32_t* tick_next) {
    uint32_t m = 0xFFFFFFFFu;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) m = min(m, tick[i] + (1u << (R - rung[i])));
    m = __reduce_min_sync(0xFFFFFFFFu, m);
    __shared__ uint32_t sm[8];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) m = min(m, sm[w]);
        atomicMin(tick_next, m);
    }
}

__global__ void __launch_bounds__(256) k_block_predict(float4* __restrict__ pos, const float4* __restrict__ vel, const float4* __restrict__ accb,
                                                       const uint32_t* __restrict__ tick, const uint8_t* __restrict__ rung, int n, int R,
                                                       float dt_max, const uint32_t* __restrict__ tick_next, uint8_t* __restrict__ active,
                                                       DevScalars* sc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool act = false;
    if (i < n) {
        const int r = rung[i];
        act = tick[i] + (1u << (R - r)) == *tick_next;
        active[i] = act ? 1 : 0;
        if (act) {
            const float h = ldexpf(dt_max, -r);
            const float hh = __fmul_rn(__fmul_rn(0.5f, h), h);
            float4 p = pos[i];
            const float4 v = vel[i], a = accb[i];
            p.x = __fmaf_rn(a.x, hh, __fmaf_rn(v.x, h, p.x));
            p.y = __fmaf_rn(a.y, hh, __fmaf_rn(v.y, h, p.y));
            p.z = __fmaf_rn(a.z, hh, __fmaf_rn(v.z, h, p.z));
            pos[i] = p;
        }
    }
    const uint32_t b = __ballot_sync(0xFFFFFFFFu, act);
    if ((threadIdx.x & 31) == 0 && b) atomicAdd(&sc->n_active, (uint32_t)__popc(b));
}

// After a rebuild: the block state follows the sort (perm[j] = position before the build of the j-th sorted particle).
__global__ void __launch_bounds__(256) k_block_permute(const uint32_t* __restrict__ perm, int n, const float4* __restrict__ accb_in,
                                                       const uint32_t* __restrict__ tick_in, const uint8_t* __restrict__ rung_in,
                                                       const uint8_t* __restrict__ act_in, float4* __restrict__ accb, uint32_t* __restrict__ tick,
                                                       uint8_t* __restrict__ rung, uint8_t* __restrict__ act, uint32_t* __restrict__ g_base) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const uint32_t s = perm[j];
    accb[j] = accb_in[s];
    tick[j] = tick_in[s];
    rung[j] = rung_in[s];
    act[j] = act_in[s];
    g_base[j] = 0u;                                        // new groups: no reference interaction counts yet
}

__global__ void __launch_bounds__(256) k_block_correct(float4* __restrict__ vel, float4* __restrict__ accb, const float4* __restrict__ acc,
                                                       uint32_t* __restrict__ tick, uint8_t* __restrict__ rung, const uint8_t* __restrict__ active,
                                                       int n, int R, float dt_max, float len, float eta, const uint32_t* __restrict__ tick_next,
                                                       uint32_t* tick_next_idle, DevScalars* sc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        *tick_next_idle = 0xFFFFFFFFu;                      // the other parity's slot, for the next step
        // ticks are 32-bit: tick + 2^(R - rung) must not wrap.  Within two longest steps of 2^32 the deferred status says so
        // (this step and the next are still exact); the caller starts over with bh_block_init.
        if (*tick_next >= 0xFFFFFFFFu - (2u << R)) atomicMin(&sc->status, (int)BH_ERR_STATE);
    }
    if (i >= n || !active[i]) return;
    const uint32_t now = *tick_next;
    const int r = rung[i];
    const float hh = __fmul_rn(0.5f, ldexpf(dt_max, -r));
    const float4 a0 = accb[i], a1 = acc[i];
    float4 v = vel[i];
    v.x = __fmaf_rn(__fadd_rn(a0.x, a1.x), hh, v.x);
    v.y = __fmaf_rn(__fadd_rn(a0.y, a1.y), hh, v.y);
    v.z = __fmaf_rn(__fadd_rn(a0.z, a1.z), hh, v.z);
    vel[i] = v;
    accb[i] = a1;
    tick[i] = now;
    const int lowest = now ? max(R - (__ffs((int)now) - 1), 0) : 0;      // a longer step only starts at a multiple of it
    rung[i] = rung_of(a1, len, eta, dt_max, R, lowest);
}

// Interactions of the groups walked in this step, now and when each was first walked on the current cells.
__global__ void __launch_bounds__(256) k_block_degrade(DevScalars* sc, const uint8_t* __restrict__ g_active, const uint32_t* __restrict__ g_npc,
                                                       const uint32_t* __restrict__ g_npp, uint32_t* __restrict__ g_base) {
    const uint32_t G = sc->n_groups;
    unsigned long long now = 0, base = 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < G; g += gridDim.x * blockDim.x) {
        if (!g_active[g]) continue;
        const uint32_t c = g_npc[g] + g_npp[g];
        uint32_t b = g_base[g];
        if (b == 0u) { b = c; g_base[g] = c; }
        now += c;
        base += b;
    }
    now = __reduce_add_sync(0xFFFFFFFFu, (unsigned)(now & 0xFFFFFFFFu)) + ((unsigned long long)__reduce_add_sync(0xFFFFFFFFu, (unsigned)(now >> 32)) << 32);
    base = __reduce_add_sync(0xFFFFFFFFu, (unsigned)(base & 0xFFFFFFFFu)) + ((unsigned long long)__reduce_add_sync(0xFFFFFFFFu, (unsigned)(base >> 32)) << 32);
    if ((threadIdx.x & 31) == 0 && now) { atomicAdd(&sc->deg_now, now); atomicAdd(&sc->deg_base, base); }
}

int stage_block_init(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    c->bcur = 0;
    BH_LAUNCH(c, k_block_init, (unsigned)div_up(n, 256), 256, 0, s, c->ws.acc, n, c->blk_len, c->blk_eta, c->blk_dt_max, c->blk_R, c->ws.accb[0],
              c->ws.tick[0], c->ws.rung[0], c->ws.g_base, c->ws.sc);
    return BH_OK;
}

int stage_block_predict(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n, b = c->bcur;
    uint32_t* tn = &c->ws.sc->tick_next[c->blk_steps & 1];
    const int grid = (int)std::min<int64_t>(div_up(n, 256), (int64_t)c->sm_count * 8);
    // n_active, deg_now, deg_base and nothing else (the sort's words behind them keep their values: sort_retries counts since bh_create)
    BH_CUDA(c, cudaMemsetAsync(&c->ws.sc->n_active, 0, offsetof(DevScalars, sort_skip) - offsetof(DevScalars, n_active), s));
    BH_LAUNCH(c, k_block_next, grid, 256, 0, s, c->ws.tick[b], c->ws.rung[b], n, c->blk_R, tn);
    BH_LAUNCH(c, k_block_predict, (unsigned)div_up(n, 256), 256, 0, s, c->ws.pos[c->cur], c->ws.vel[c->cur], c->ws.accb[b], c->ws.tick[b], c->ws.rung[b],
              n, c->blk_R, c->blk_dt_max, tn, c->ws.bactive[b], c->ws.sc);
    return BH_OK;
}

int stage_block_permute(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n, a = c->bcur, b = c->bcur ^ 1;
    BH_LAUNCH(c, k_block_permute, (unsigned)div_up(n, 256), 256, 0, s, c->ws.val[c->sorted], n, c->ws.accb[a], c->ws.tick[a], c->ws.rung[a],
              c->ws.bactive[a], c->ws.accb[b], c->ws.tick[b], c->ws.rung[b], c->ws.bactive[b], c->ws.g_base);
    c->bcur = b;
    return BH_OK;
}

int stage_block_correct(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n, b = c->bcur;
    uint32_t* tn = &c->ws.sc->tick_next[c->blk_steps & 1];
    uint32_t* idle = &c->ws.sc->tick_next[(c->blk_steps + 1) & 1];
    BH_LAUNCH(c, k_block_correct, (unsigned)div_up(n, 256), 256, 0, s, c->ws.vel[c->cur], c->ws.accb[b], c->ws.acc, c->ws.tick[b], c->ws.rung[b],
              c->ws.bactive[b], n, c->blk_R, c->blk_dt_max, c->blk_len, c->blk_eta, tn, idle, c->ws.sc);
    const int grid = (int)std::min<int64_t>(div_up(n, 256), (int64_t)c->sm_count * 4);
    BH_LAUNCH(c, k_block_degrade, grid, 256, 0, s, c->ws.sc, c->ws.gflag, c->ws.g_npc, c->ws.g_npp, c->ws.g_base);
    return BH_OK;
}

}  // namespace bh
