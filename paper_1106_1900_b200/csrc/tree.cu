// tree.cu -- S4 sparse octree (cells + links) and S5 groups.
// PAPER.md:63-65 (Fig.1-2) defines the tree level by level: mask keys, group equal prefixes of unflagged particles,
// <= nleaf -> leaf; PAPER.md:75 takes the groups from the tree cells (<= ncrit particles).  Both are pure functions of
// the sorted keys, and this file builds the identical arrays in TWO launches instead of ~20 dependent mask/compact
// rounds plus a link kernel:
//   cl(a, b) = number of leading levels on which two keys agree  (XOR + count-leading-zeros),
//   fl(i)  = cl(key[i-1], key[i]) + 1 = first level at which particle i starts a new run   (fl(0) = fl(n) = 0),
//   dep(i) = level of the leaf holding i = min(1 + max_{s in [i-nleaf, i]} cl(key[s], key[s+nleaf]), 20)
//            (a level-L run through i holds > nleaf particles iff some window of nleaf+1 sorted keys around i agrees on L levels),
//   glv(i) = 1 + max_{s in [i-ncrit, i]} cl(key[s], key[s+ncrit]) = the highest level at which i's run holds <= ncrit particles.
// A cell of level L starts at boundary i iff fl(i) <= L <= dep(i) and ends at boundary j iff fl(j) <= L <= dep(j-1).
// A group starts at i iff a cell of level glv(i) starts there (glv <= dep: the group is that cell, A12), or -- a leaf that
// holds more than ncrit particles (level-20 overflow, or nleaf > ncrit) -- iff i is a multiple of ncrit past the leaf's
// first particle (found by a binary search over the sorted keys).
// k_bounds computes fl, dep, the group marks and the per-(row, tile) counts of starts (rows: levels 0..20, then groups);
// the LAST block to finish scans every row over the tiles (no extra launch).  k_emit numbers the cells level-major in
// ascending first particle (= the exclusive scans) and writes begin / end / first child / child end / parent, the groups,
// and the tree's scalars.  No atomics touch the topology: the result is deterministic.
#include <algorithm>
#include "bh_internal.cuh"

namespace bh {

constexpr int kTreeThreads = 256;                  // a block handles a tile of kTreeTile = 1024 boundaries
constexpr int kTreeWarps = kTreeThreads / 32;
constexpr int kTreePer = kTreeTile / kTreeThreads; // 4
constexpr int kWin = kTreeTile + 2 * kHaloMax;     // keys a tile looks at: [t0 - 64, t0 + 1024 + 64)

// cl for 60-bit keys: (clz - 4) / 3, the division as a multiplication (exact for 0..60)
__device__ __forceinline__ int common_level_fast(uint64_t a, uint64_t b) {
    const uint64_t x = a ^ b;
    if (x == 0) return kMaxLevel;
    return ((__clzll((long long)x) - 4) * 43) >> 7;
}

// max of the int8 table t over [first, last] (inclusive; first > last: -1): bytes up to a word boundary, whole words, bytes
__device__ __forceinline__ int range_max(const int8_t* t, int first, int last) {
    int m = -1;
    int x = first;
    for (; x <= last && (x & 3); ++x) m = max(m, (int)t[x]);
    uint32_t wm = 0x80808080u;
    for (; x + 3 <= last; x += 4) wm = __vmaxs4(wm, *reinterpret_cast<const uint32_t*>(t + x));
    for (; x <= last; ++x) m = max(m, (int)t[x]);
    m = max(m, max(max((int)(int8_t)(wm & 0xFF), (int)(int8_t)((wm >> 8) & 0xFF)), max((int)(int8_t)((wm >> 16) & 0xFF), (int)(int8_t)(wm >> 24))));
    return m;
}

// Window maxima of four consecutive positions: out[b] = max t[j0 + b - w .. j0 + b], b = 0..3 (w >= 0).
__device__ __forceinline__ void window_max4(const int8_t* t, int j0, int w, int out[4]) {
    if (w < 3) {
#pragma unroll
        for (int b = 0; b < 4; ++b) out[b] = range_max(t, j0 + b - w, j0 + b);
        return;
    }
    const int common = range_max(t, j0 + 3 - w, j0);                 // shared by all four windows
    const int l0 = t[j0 - w], l1 = t[j0 + 1 - w], l2 = t[j0 + 2 - w];
    const int r1 = t[j0 + 1], r2 = t[j0 + 2], r3 = t[j0 + 3];
    out[0] = max(common, max(l0, max(l1, l2)));
    out[1] = max(common, max(max(l1, l2), r1));
    out[2] = max(common, max(l2, max(r1, r2)));
    out[3] = max(common, max(r1, max(r2, r3)));
}

template <int kNleaf, int kNcrit>      // compile-time leaf / group sizes (0: the run-time arguments)
__global__ void __launch_bounds__(kTreeThreads) k_bounds(const uint64_t* __restrict__ key, int n, int nleaf_rt, int ncrit_rt, int tiles,
                                                         uint8_t* __restrict__ fl, uint8_t* __restrict__ dep, uint8_t* __restrict__ gl,
                                                         uint32_t* tile_cnt) {
    __shared__ uint64_t skey[kWin];
    __shared__ __align__(4) int8_t ta[kWin + 8], tb[kWin + 8];   // cl(key[s], key[s + nleaf]) and cl(key[s], key[s + ncrit]), s = g0 + index
    __shared__ uint32_t scnt[kTreeRows];
    const int nleaf = kNleaf ? kNleaf : nleaf_rt, ncrit = kNcrit ? kNcrit : ncrit_rt;
    const int tid = threadIdx.x;
    const int t0 = blockIdx.x * kTreeTile;
    const int g0 = t0 - kHaloMax;                       // global index of skey[0]
    for (int j = tid; j < kWin; j += kTreeThreads) {
        const int gi = g0 + j;
        skey[j] = (gi >= 0 && gi < n) ? key[gi] : 0ull;
    }
    if (tid < kTreeRows) scnt[tid] = 0u;
    __syncthreads();
    for (int j = tid; j < kWin; j += kTreeThreads) {     // -1 where the window leaves [0, n) (or the part of the table a tile needs)
        const int s = g0 + j;
        int a = -1, b = -1;
        if (s >= 0 && s + nleaf < n && j + nleaf < kWin) a = common_level_fast(skey[j], skey[j + nleaf]);
        if (s >= 0 && s + ncrit < n && j + ncrit < kWin) b = common_level_fast(skey[j], skey[j + ncrit]);
        ta[j] = (int8_t)a;
        tb[j] = (int8_t)b;
    }
    __syncthreads();
    // ---- four consecutive boundaries per thread
    const int i0 = t0 + kTreePer * tid, j0 = kTreePer * tid + kHaloMax;
    int wl[4], wc[4];
    window_max4(ta, j0, nleaf, wl);
    window_max4(tb, j0, ncrit, wc);
    uint32_t pfl = 0, pdep = 0, pgl = 0;                 // four bytes each
#pragma unroll
    for (int b = 0; b < kTreePer; ++b) {
        const int i = i0 + b, j = j0 + b;
        int myfl = 0, d = 0, glev = 0xFF;
        if (i <= n) {
            if (i > 0 && i < n) myfl = common_level_fast(skey[j - 1], skey[j]) + 1;
            if (i < n) {
                d = min(wl[b] + 1, kMaxLevel);
                const int gv = wc[b] + 1;
                bool gstart;
                int gcell_level = gv;
                if (gv <= d) {
                    gstart = myfl <= gv;                                     // the group is the level-gv cell, which starts here
                } else {                                                      // a leaf with more than ncrit particles: chunks of ncrit
                    gcell_level = d;
                    const int sh = 60 - 3 * d;
                    const uint64_t target = (skey[j] >> sh) << sh;            // smallest key of the leaf's key range
                    int lo = 0, hi = i;                                       // first particle of the leaf = lower_bound(target)
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        if (__ldg(key + mid) < target) lo = mid + 1; else hi = mid;
                    }
                    gstart = ((i - lo) % ncrit) == 0;
                }
                if (gstart) { glev = gcell_level; atomicAdd(&scnt[kLevels], 1u); }
                for (int L = myfl; L <= d; ++L) atomicAdd(&scnt[L], 1u);       // cells that start here (0.24 per particle)
            }
        }
        pfl |= (uint32_t)myfl << (8 * b);
        pdep |= (uint32_t)d << (8 * b);
        pgl |= (uint32_t)glev << (8 * b);
    }
    if (i0 <= n) {                                       // the arrays are padded to whole words
        *reinterpret_cast<uint32_t*>(fl + i0) = pfl;
        *reinterpret_cast<uint32_t*>(dep + i0) = pdep;
        *reinterpret_cast<uint32_t*>(gl + i0) = pgl;
    }
    __syncthreads();
    if (tid < kTreeRows) tile_cnt[(size_t)tid * tiles + blockIdx.x] = scnt[tid];
}

// Exclusive scan of every row of tile_cnt over the tiles, in place, and the row totals: one warp (one block, so that every
// row has an SM's load / store path to itself) per row; a lane scans a contiguous run of the row, all loads in flight at once.
__global__ void __launch_bounds__(32) k_scan_rows(uint32_t* tile_cnt, uint32_t* row_total, int tiles) {
    const int lane = threadIdx.x, r = blockIdx.x;
    {
        uint32_t* row = tile_cnt + (size_t)r * tiles;
        uint32_t carry = 0;
        for (int base = 0; base < tiles; base += 32 * 40) {
            const int per = min(40, (min(tiles - base, 32 * 40) + 31) / 32);   // entries per lane in this stretch
            const int first = base + lane * per;
            uint32_t x[40];
#pragma unroll
            for (int q = 0; q < 40; ++q) {                       // every load is requested before any is used
                const int t = min(first + q, tiles - 1);
                x[q] = __ldcg(row + t);
            }
            uint32_t sum = 0;
#pragma unroll
            for (int q = 0; q < 40; ++q) {
                if (!(q < per && first + q < tiles)) x[q] = 0u;
                sum += x[q];
            }
            uint32_t inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, inc, o);
                if (lane >= o) inc += u;
            }
            uint32_t run = carry + inc - sum;
#pragma unroll
            for (int q = 0; q < 40; ++q) {
                if (q < per && first + q < tiles) row[first + q] = run;
                run += x[q];
            }
            carry += __shfl_sync(0xFFFFFFFFu, inc, 31);
        }
        if (lane == 0) row_total[r] = carry;
    }
}

// Emit the cell arrays and the groups.  A level-L cell that starts at boundary i gets the index
//   S(L, i) = level_offset[L] + (level-L starts in earlier tiles) + (level-L starts before i in this tile),
// the last term from one ballot per level and warp.  Starts are sparse (0.24 per particle), so every thread only walks
// the levels at which a cell really starts or ends at its boundary.
__global__ void __launch_bounds__(kTreeThreads) k_emit(const uint8_t* __restrict__ fl, const uint8_t* __restrict__ dep, const uint8_t* __restrict__ gl,
                                                       int n, int tiles, const uint32_t* __restrict__ tile_base, const uint32_t* __restrict__ row_total,
                                                       uint32_t max_cells, uint4* __restrict__ c_topo, uint32_t* __restrict__ c_parent,
                                                       uint32_t* __restrict__ g_begin, uint32_t* __restrict__ g_cell, DevScalars* sc) {
    __shared__ uint32_t bal[kTreeWarps][kTreeRows];      // ballots of the current 256 boundaries: who starts a cell of level L / a group
    __shared__ uint32_t wpre[kTreeWarps][kTreeRows];     // starts in the earlier warps of this round + everything before (the running base)
    __shared__ uint32_t base[kTreeRows];
    __shared__ uint32_t s_overflow;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;
    if (w == 0) {
        // level offsets from the row totals (level-major numbering); more cells than the workspace holds: report it and
        // publish an EMPTY tree, so that every later stage is a no-op
        const uint32_t tot = lane < kTreeRows ? row_total[lane] : 0u;
        const uint32_t tb = lane < kTreeRows ? tile_base[(size_t)lane * tiles + blockIdx.x] : 0u;
        const uint32_t cells = lane < kLevels ? tot : 0u;
        uint32_t inc = cells;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += u;
        }
        const uint32_t off = inc - cells;                              // lane L: first cell of level L; lane kLevels: all cells
        const uint32_t ncell = __shfl_sync(0xFFFFFFFFu, inc, 31);
        const uint32_t levels = __ballot_sync(0xFFFFFFFFu, cells != 0u);
        const uint32_t ngroups = __shfl_sync(0xFFFFFFFFu, tot, kLevels);
        const bool overflow = ncell > max_cells;
        if (lane == 0) s_overflow = overflow ? 1u : 0u;
        if (lane < kTreeRows) base[lane] = (lane < kLevels ? off : 0u) + tb;   // groups are numbered from 0
        if (blockIdx.x == 0) {
            if (lane <= kLevels) sc->level_offset[lane] = overflow ? 0u : off;
            if (lane == 0) {
                sc->n_cells = overflow ? 0u : ncell;
                sc->n_levels = overflow ? 0u : (uint32_t)(32 - __clz(levels));
                sc->n_groups = overflow ? 0u : ngroups;
                if (overflow) atomicMin(&sc->status, (int)BH_ERR_CAPACITY);
                else g_begin[ngroups] = (uint32_t)n;                   // sentinel
            }
        }
    }
    __syncthreads();
    if (s_overflow) return;
    auto S = [&](int L) { return wpre[w][L] + (uint32_t)__popc(bal[w][L] & lt); };
    for (int r = 0; r < kTreePer; ++r) {
        const int i = blockIdx.x * kTreeTile + r * kTreeThreads + tid;
        int myfl = 255, mydep = -1, prevdep = -1, mygl = 255;
        if (i <= n) {
            myfl = fl[i];
            if (i < n) { mydep = dep[i]; mygl = gl[i]; }
            if (i > 0) prevdep = dep[i - 1];
        }
        uint32_t mine = 0;
#pragma unroll
        for (int L = 0; L < kLevels; ++L) {
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, (myfl <= L) && (L <= mydep));
            if (lane == L) mine = b;
        }
        {
            const uint32_t b = __ballot_sync(0xFFFFFFFFu, mygl != 255);
            if (lane == kLevels) mine = b;
        }
        if (lane < kTreeRows) bal[w][lane] = mine;
        __syncthreads();
        if (tid < kTreeRows) {
            uint32_t run = base[tid];
#pragma unroll
            for (int ww = 0; ww < kTreeWarps; ++ww) {
                wpre[ww][tid] = run;
                run += __popc(bal[ww][tid]);
            }
            base[tid] = run;
        }
        __syncthreads();
        if (i <= n) {
            const int top = max(mydep, prevdep);
            for (int L = myfl; L <= top; ++L) {
                const uint32_t sL = S(L);
                if (L <= mydep) {                        // a level-L cell starts here
                    uint32_t* t = reinterpret_cast<uint32_t*>(c_topo + sL);      // (first particle, end particle, first child, end child)
                    t[0] = (uint32_t)i;
                    const bool leaf = (L == mydep);
                    t[2] = leaf ? 0u : S(L + 1);
                    if (leaf) t[3] = 0u;
                    uint32_t par = kNone;
                    if (L > 0) par = (myfl <= L - 1) ? S(L - 1) : S(L - 1) - 1u;
                    c_parent[sL] = par;
                }
                if (i > 0 && L <= prevdep) {             // a level-L cell ends here
                    uint32_t* t = reinterpret_cast<uint32_t*>(c_topo + (sL - 1u));
                    t[1] = (uint32_t)i;
                    if (L < prevdep) t[3] = S(L + 1);
                }
            }
            if (mygl != 255) {                           // the group's cell (a chunk of an over-full leaf: that leaf)
                const uint32_t g = S(kLevels);
                g_begin[g] = (uint32_t)i;
                g_cell[g] = (myfl <= mygl) ? S(mygl) : S(mygl) - 1u;
            }
        }
        __syncthreads();                                 // bal / wpre are rewritten by the next round
    }
}

// ------------------------------------------------------------------------------------------ export
__global__ void __launch_bounds__(256) k_export(const DevScalars* __restrict__ sc, const uint64_t* __restrict__ key,
                                                const uint4* __restrict__ c_topo, const uint32_t* __restrict__ c_parent, const float4* __restrict__ trec, const double* __restrict__ mom64,
                                                int32_t* __restrict__ e_level, uint64_t* __restrict__ e_prefix, uint32_t* __restrict__ e_pbegin, uint32_t* __restrict__ e_pcount,
                                                int32_t* __restrict__ e_cbegin, int32_t* __restrict__ e_nchild, int32_t* __restrict__ e_parent,
                                                float* __restrict__ e_mom32, float* __restrict__ e_r2open) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        int L = 0;
        while (L < kMaxLevel && c >= sc->level_offset[L + 1]) ++L;
        e_level[c] = L;
        const uint4 t = c_topo[c];
        const uint32_t b = t.x;
        e_prefix[c] = (L == 0) ? 0ull : (key[b] >> (60 - 3 * L));
        e_pbegin[c] = b;
        e_pcount[c] = t.y - b;
        const uint32_t cb = t.z, ce = t.w;
        e_cbegin[c] = (ce == cb) ? -1 : (int32_t)cb;
        e_nchild[c] = (int32_t)(ce - cb);
        e_parent[c] = (c_parent[c] == kNone) ? -1 : (int32_t)c_parent[c];
        float* m = e_mom32 + 10 * (size_t)c;
#pragma unroll
        for (int k = 0; k < 10; ++k) m[k] = (float)mom64[10 * (size_t)c + k];   // the fp32 roundings (the walk's own records: bh_tree_view.cell_trec / cell_erec)
        e_r2open[c] = trec[c].w;
    }
}

// ------------------------------------------------------------------------------------------ host side
int stage_cells(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    const int tiles = (int)div_up((int64_t)n + 1, kTreeTile);
    const uint64_t* key = c->ws.key[c->sorted];
    if (c->nleaf == 16 && c->ncrit == 64)
        BH_LAUNCH(c, (k_bounds<16, 64>), tiles, kTreeThreads, 0, s, key, n, 16, 64, tiles, c->ws.fl, c->ws.dep, c->ws.gl, c->ws.tile_cnt);
    else
        BH_LAUNCH(c, (k_bounds<0, 0>), tiles, kTreeThreads, 0, s, key, n, (int)c->nleaf, (int)c->ncrit, tiles, c->ws.fl, c->ws.dep, c->ws.gl, c->ws.tile_cnt);
    BH_LAUNCH(c, k_scan_rows, kTreeRows, 32, 0, s, c->ws.tile_cnt, c->ws.row_total, tiles);
    if (c->timing) stage_mark(c, 5, s);
    BH_LAUNCH(c, k_emit, tiles, kTreeThreads, 0, s, c->ws.fl, c->ws.dep, c->ws.gl, n, tiles, c->ws.tile_cnt, c->ws.row_total, (uint32_t)c->max_cells,
              c->ws.c_topo, c->ws.c_parent, c->ws.g_begin, c->ws.g_cell, c->ws.sc);
    return BH_OK;
}

int stage_export(bh_ctx* c, cudaStream_t s) {
    const int grid = (int)std::min<int64_t>(div_up(c->max_cells, 256), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_export, grid, 256, 0, s, c->ws.sc, c->ws.key[c->sorted], c->ws.c_topo, c->ws.c_parent, c->ws.trec, c->ws.mom64,
              c->ws.e_level, c->ws.e_prefix, c->ws.e_pbegin, c->ws.e_pcount, c->ws.e_cbegin,
              c->ws.e_nchild, c->ws.e_parent, c->ws.e_mom32, c->ws.e_r2open);
    return BH_OK;
}

}  // namespace bh
