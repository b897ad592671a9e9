// tree.cu -- S4 sparse octree (cells + links) and S5 groups.
// PAPER.md:63-65 (Fig.1-2) defines the tree level by level: mask keys, group equal prefixes of unflagged particles,
// <= nleaf -> leaf.  That tree is a pure function of the sorted keys, and this file builds the identical arrays in
// one streaming pass instead of ~20 dependent mask/compact rounds:
//   cl(i)  = number of leading levels on which key[i-1] and key[i] agree  (XOR + count-leading-zeros),
//   fl(i)  = cl(i) + 1 = first level at which particle i starts a new run     (fl(0) = fl(n) = 0; identical keys: 21),
//   dep(i) = level of the leaf holding i = min(1 + max_{s in [i-nleaf, i]} cl(key[s], key[s+nleaf]), 20)
//            (a level-L run through i holds > nleaf particles iff some window of nleaf+1 sorted keys around i agrees on L levels).
// A cell of level L starts at boundary i iff fl(i) <= L <= dep(i) and ends at boundary j iff fl(j) <= L <= dep(j-1).
// Numbering (level-major, ascending first particle) = exclusive scan of the per-(level, tile) start counts.
#include <algorithm>
#include "bh_internal.cuh"

namespace bh {

__device__ __forceinline__ int common_level(uint64_t a, uint64_t b) {
    const uint64_t x = a ^ b;
    if (x == 0) return kMaxLevel;
    const int msb = 63 - __clzll((long long)x);
    return (59 - msb) / 3;
}

// fl, dep and the per-(level, tile) counts of cell starts.  One boundary per thread; boundaries 0..n.
__global__ void __launch_bounds__(kTreeTile) k_bounds_count(const uint64_t* __restrict__ key, int n, int nleaf, int tiles,
                                                            uint8_t* __restrict__ fl, uint8_t* __restrict__ dep,
                                                            uint32_t* __restrict__ tile_cnt) {
    __shared__ uint64_t skey[kTreeTile + 2 * kHaloMax];
    __shared__ int8_t sw[kTreeTile + kHaloMax];
    __shared__ uint32_t scnt[kLevels];
    const int t0 = blockIdx.x * kTreeTile;
    const int g0 = t0 - kHaloMax;                       // global index of skey[0]
    for (int j = threadIdx.x; j < kTreeTile + 2 * kHaloMax; j += kTreeTile) {
        const int gi = g0 + j;
        skey[j] = (gi >= 0 && gi < n) ? key[gi] : 0ull;
    }
    if (threadIdx.x < kLevels) scnt[threadIdx.x] = 0;
    __syncthreads();
    // sw[j] = cl(key[s], key[s+nleaf]) for s = g0 + j (window of nleaf+1 keys), -1 where the window leaves [0, n)
    for (int j = threadIdx.x; j < kTreeTile + kHaloMax; j += kTreeTile) {
        const int s = g0 + j;
        int w = -1;
        if (s >= 0 && s + nleaf < n) w = common_level(skey[j], skey[j + nleaf]);
        sw[j] = (int8_t)w;
    }
    __syncthreads();
    const int i = t0 + threadIdx.x;
    if (i <= n) {
        const int j = threadIdx.x + kHaloMax;
        int myfl = 0;
        if (i > 0 && i < n) myfl = common_level(skey[j - 1], skey[j]) + 1;
        fl[i] = (uint8_t)myfl;
        if (i < n) {
            int m = -1;
            for (int k = 0; k <= nleaf; ++k) m = max(m, (int)sw[j - k]);
            const int d = min(m + 1, kMaxLevel);
            dep[i] = (uint8_t)d;
            for (int L = myfl; L <= d; ++L) atomicAdd(&scnt[L], 1u);
        }
    }
    __syncthreads();
    if (threadIdx.x < kLevels) tile_cnt[(size_t)threadIdx.x * tiles + blockIdx.x] = scnt[threadIdx.x];
}

__global__ void k_tree_finalize(const uint32_t* __restrict__ tile_base, int tiles, const uint32_t* __restrict__ d_total,
                                uint32_t max_cells, DevScalars* sc) {
    const int t = threadIdx.x;
    __shared__ uint32_t lo[kLevels + 1];
    if (t < kLevels) lo[t] = tile_base[(size_t)t * tiles];
    if (t == kLevels) lo[t] = *d_total;
    __syncthreads();
    // more cells than the workspace holds: report it and publish an EMPTY tree, so that every later stage is a no-op
    const bool overflow = lo[kLevels] > max_cells;
    if (t <= kLevels) sc->level_offset[t] = overflow ? 0u : lo[t];
    if (t == 0) {
        int nl = 0;
        for (int L = 0; L < kLevels; ++L) if (lo[L + 1] > lo[L]) nl = L + 1;
        sc->n_cells = overflow ? 0u : lo[kLevels];
        sc->n_levels = overflow ? 0u : (uint32_t)nl;
        if (overflow) atomicMin(&sc->status, (int)BH_ERR_CAPACITY);
    }
}

// Emit the cell arrays.  S[L] = global index a level-L cell starting at this boundary would get.
__global__ void __launch_bounds__(kTreeTile) k_emit_cells(const uint8_t* __restrict__ fl, const uint8_t* __restrict__ dep, int n, int tiles,
                                                          const uint32_t* __restrict__ tile_base, uint32_t max_cells,
                                                          uint32_t* __restrict__ c_pbegin, uint32_t* __restrict__ c_pend,
                                                          uint32_t* __restrict__ c_cbegin, uint32_t* __restrict__ c_cend,
                                                          uint32_t* __restrict__ c_parent, uint32_t* __restrict__ c_arrive) {
    constexpr int kWarps = kTreeTile / 32;
    __shared__ uint32_t wc[kLevels][kWarps];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    const int i = blockIdx.x * kTreeTile + threadIdx.x;
    int myfl = 255, mydep = -1, prevdep = -1;
    if (i <= n) {
        myfl = fl[i];
        if (i < n) mydep = dep[i];
        if (i > 0) prevdep = dep[i - 1];
    }
    uint32_t S[kLevels + 1];
#pragma unroll
    for (int L = 0; L < kLevels; ++L) {
        const bool st = (myfl <= L) && (L <= mydep);
        const uint32_t b = __ballot_sync(0xFFFFFFFFu, st);
        S[L] = __popc(b & lt);
        if (lane == 0) wc[L][w] = __popc(b);
    }
    S[kLevels] = 0;
    __syncthreads();
    if (threadIdx.x < kLevels) {
        uint32_t run = tile_base[(size_t)threadIdx.x * tiles + blockIdx.x];
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) {
            const uint32_t t = wc[threadIdx.x][ww];
            wc[threadIdx.x][ww] = run;
            run += t;
        }
    }
    __syncthreads();
#pragma unroll
    for (int L = 0; L < kLevels; ++L) S[L] += wc[L][w];
    if (i > n) return;
#pragma unroll
    for (int L = 0; L < kLevels; ++L) {
        if (myfl <= L && L <= mydep) {           // a level-L cell starts here
            const uint32_t c = S[L];
            if (c < max_cells) {
                c_pbegin[c] = (uint32_t)i;
                const bool leaf = (L == mydep);
                c_cbegin[c] = leaf ? 0u : S[L + 1];
                if (leaf) c_cend[c] = 0u;
                uint32_t par = kNone;
                if (L > 0) par = (myfl <= L - 1) ? S[L - 1] : S[L - 1] - 1u;
                c_parent[c] = par;
                c_arrive[c] = 0u;                // children counted in by k_moments
            }
        }
        if (i > 0 && myfl <= L && L <= prevdep) {   // a level-L cell ends here
            const uint32_t c = S[L] - 1u;
            if (c < max_cells) {
                c_pend[c] = (uint32_t)i;
                if (L < prevdep) c_cend[c] = S[L + 1];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ S5
// groups are tree cells with <= ncrit particles; here the highest such cells (A12), in particle order.
__global__ void __launch_bounds__(256) k_group_mark(const DevScalars* __restrict__ sc, int ncrit,
                                                    const uint32_t* __restrict__ c_pbegin, const uint32_t* __restrict__ c_pend,
                                                    const uint32_t* __restrict__ c_cbegin, const uint32_t* __restrict__ c_cend,
                                                    const uint32_t* __restrict__ c_parent,
                                                    uint8_t* __restrict__ gflag, uint32_t* __restrict__ gcell_at) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const uint32_t b = c_pbegin[c], cnt = c_pend[c] - b;
        const uint32_t par = c_parent[c];
        const bool parent_big = (par == kNone) || (c_pend[par] - c_pbegin[par] > (uint32_t)ncrit);
        if (!parent_big) continue;
        if (cnt <= (uint32_t)ncrit) {
            gflag[b] = 1;
            gcell_at[b] = c;
        } else if (c_cend[c] == c_cbegin[c]) {     // overflow leaf at the deepest level: chunks of ncrit
            for (uint32_t o = 0; o < cnt; o += ncrit) {
                gflag[b + o] = 1;
                gcell_at[b + o] = c;
            }
        }
    }
}

__global__ void __launch_bounds__(256) k_group_write(const uint8_t* __restrict__ gflag, const uint32_t* __restrict__ gscan,
                                                     const uint32_t* __restrict__ gcell_at, int n,
                                                     uint32_t* __restrict__ g_begin, uint32_t* __restrict__ g_cell, DevScalars* sc) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && gflag[i]) {
        const uint32_t g = gscan[i];
        g_begin[g] = (uint32_t)i;
        g_cell[g] = gcell_at[i];
    }
    if (i == n) g_begin[sc->n_groups] = (uint32_t)n;   // sentinel; n_groups was written by the scan
}

// ------------------------------------------------------------------------------------------ export
__global__ void __launch_bounds__(256) k_export(const DevScalars* __restrict__ sc, const uint64_t* __restrict__ key,
                                                const uint32_t* __restrict__ c_pbegin, const uint32_t* __restrict__ c_pend,
                                                const uint32_t* __restrict__ c_cbegin, const uint32_t* __restrict__ c_cend,
                                                const uint32_t* __restrict__ c_parent, const float4* __restrict__ trec, const double* __restrict__ mom64,
                                                int32_t* __restrict__ e_level, uint64_t* __restrict__ e_prefix, uint32_t* __restrict__ e_pcount,
                                                int32_t* __restrict__ e_cbegin, int32_t* __restrict__ e_nchild, int32_t* __restrict__ e_parent,
                                                float* __restrict__ e_mom32, float* __restrict__ e_r2open) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        int L = 0;
        while (L < kMaxLevel && c >= sc->level_offset[L + 1]) ++L;
        e_level[c] = L;
        const uint32_t b = c_pbegin[c];
        e_prefix[c] = (L == 0) ? 0ull : (key[b] >> (60 - 3 * L));
        e_pcount[c] = c_pend[c] - b;
        const uint32_t cb = c_cbegin[c], ce = c_cend[c];
        e_cbegin[c] = (ce == cb) ? -1 : (int32_t)cb;
        e_nchild[c] = (int32_t)(ce - cb);
        e_parent[c] = (c_parent[c] == kNone) ? -1 : (int32_t)c_parent[c];
        float* m = e_mom32 + 10 * (size_t)c;
#pragma unroll
        for (int k = 0; k < 10; ++k) m[k] = (float)mom64[10 * (size_t)c + k];   // the fp32 roundings the walk record is built from
        e_r2open[c] = trec[c].w;
    }
}

// ------------------------------------------------------------------------------------------ host side
int stage_cells(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    const int tiles = (int)div_up((int64_t)n + 1, kTreeTile);
    const uint64_t* key = c->ws.key[c->sorted];
    BH_LAUNCH(c, k_bounds_count, tiles, kTreeTile, 0, s, key, n, (int)c->nleaf, tiles, c->ws.fl, c->ws.dep, c->ws.tile_cnt);
    int rc = scan_u32(c, c->ws.tile_cnt, c->ws.tile_base, (int64_t)kLevels * tiles, &c->ws.sc->n_cells, s);
    if (rc != BH_OK) return rc;
    BH_LAUNCH(c, k_tree_finalize, 1, 32, 0, s, c->ws.tile_base, tiles, &c->ws.sc->n_cells, (uint32_t)c->max_cells, c->ws.sc);
    BH_LAUNCH(c, k_emit_cells, tiles, kTreeTile, 0, s, c->ws.fl, c->ws.dep, n, tiles, c->ws.tile_base, (uint32_t)c->max_cells,
              c->ws.c_pbegin, c->ws.c_pend, c->ws.c_cbegin, c->ws.c_cend, c->ws.c_parent, c->ws.c_arrive);
    return BH_OK;
}

int stage_groups(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    BH_CUDA(c, cudaMemsetAsync(c->ws.gflag, 0, (size_t)n, s));
    const int grid = (int)std::min<int64_t>(div_up(c->max_cells, 256), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_group_mark, grid, 256, 0, s, c->ws.sc, (int)c->ncrit, c->ws.c_pbegin, c->ws.c_pend, c->ws.c_cbegin,
              c->ws.c_cend, c->ws.c_parent, c->ws.gflag, c->ws.gcell_at);
    int rc = scan_u8(c, c->ws.gflag, c->ws.gscan, n, &c->ws.sc->n_groups, s);
    if (rc != BH_OK) return rc;
    BH_LAUNCH(c, k_group_write, (unsigned)div_up((int64_t)n + 1, 256), 256, 0, s, c->ws.gflag, c->ws.gscan, c->ws.gcell_at, n,
              c->ws.g_begin, c->ws.g_cell, c->ws.sc);
    return BH_OK;
}

int stage_export(bh_ctx* c, cudaStream_t s) {
    const int grid = (int)std::min<int64_t>(div_up(c->max_cells, 256), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_export, grid, 256, 0, s, c->ws.sc, c->ws.key[c->sorted], c->ws.c_pbegin, c->ws.c_pend, c->ws.c_cbegin,
              c->ws.c_cend, c->ws.c_parent, c->ws.trec, c->ws.mom64, c->ws.e_level, c->ws.e_prefix, c->ws.e_pcount, c->ws.e_cbegin,
              c->ws.e_nchild, c->ws.e_parent, c->ws.e_mom32, c->ws.e_r2open);
    return BH_OK;
}

}  // namespace bh
