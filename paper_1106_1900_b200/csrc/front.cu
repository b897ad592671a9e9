// front.cu -- S0 domain box, S1 Morton keys, S2 stable LSD radix sort and S3 reorder in ONE cooperative launch, for
// inputs whose sort tiles are all resident on the device at once (n <= 8192 x SMs: 1.2 M particles on B200).
// PAPER.md:374-392 (keys), PAPER.md:350-370 (split / radix sort), PAPER.md:174 ("moving").
//
// Why: at 1 M particles the whole front end moves ~0.3 GB that sits in the 126 MB L2; the round-1 sequence of 14
// launches (box, domain, keys, 8 sort passes with a decoupled look-back each, reorder) spent its time in launch gaps and
// in the look-back chain, not in bandwidth.  Here one block of 1024 threads per SM owns one tile of up to 8192 particles for
// the whole kernel:
//   * the box is reduced per tile and combined by every block after a grid barrier (no atomics, no reset launch);
//   * the keys are made in registers and go straight into the first sort pass (the unsorted keys are never written);
//   * a pass = rank the tile (one ballot per digit bit, or MATCH.ANY where a row of 32 keys holds few distinct digits),
//     publish the tile's digit counts as a row of a [tiles][256] matrix (+ a reduction into the sums of its group of 16
//     tiles), GRID BARRIER, sum the group sums and the rows of the earlier tiles of the own group (all co-resident: no
//     look-back chain), exchange through shared memory, scatter, GRID BARRIER;
//   * THE SHORT SORT: the passes cover only the leading 8 x short_passes key bits; what is left to do is to order each run
//     of keys with equal leading bits by the trailing bits (equal keys in their original order), which the fix-up does in
//     a shared-memory window, and the particles are scattered to their final places from registers (S3).  A run too long
//     for the window raises a flag that every block reads behind the closing barrier; the full 8-pass sort then follows
//     in the same launch, from the keys made afresh.
// The barriers are counters in the workspace (cooperative launch guarantees co-residency): barrier k of an attempt is
// passed at k x blocks arrivals, the closing barrier counts on a word that only grows, so block 0 can zero the others.
// Values other blocks wrote during this launch are read with ld.global.cg: L1 may hold lines from earlier passes.
// Result: the stable order of the 60-bit keys, identical to keys_sort.cu's, which serves larger inputs.
#include <algorithm>
#include <cstdio>
#include "bh_internal.cuh"


namespace bh {

constexpr int kFrontThreads = 1024;                             // 1024: one block per SM (half as many arrivals at every grid barrier); 512: two
constexpr int kFrontBlocksPerSM = 1024 / kFrontThreads;
constexpr int kFrontWarps = kFrontThreads / 32;
constexpr int kFrontItems = 8;                                  // keys per thread
constexpr int kFrontTile = kFrontThreads * kFrontItems;         // most keys of a tile (block)
constexpr int kFrontParts = kFrontThreads / kRadix;             // threads per digit in the prefix step

struct FrontArgs {
    const float4* pos_in;
    const float4* vel_in;
    const uint32_t* id_in;
    float4* pos_out;
    float4* vel_out;
    uint32_t* id_out;
    int n;
    int tile_n;          // keys per tile (block): a multiple of kFrontThreads, <= kFrontTile; the tiles are spread evenly over the SMs
    int fuse_reorder;
    uint64_t* key0;
    uint64_t* key1;
    uint32_t* val0;
    uint32_t* val1;
    DevScalars* sc;
    float* part;         // [tiles][8]   per-tile box: min xyz, max xyz, bad flag
    uint32_t* matrix;    // [tiles][256] digit counts of every tile in the current pass
    uint32_t* gsum;      // [8][groups][256] digit counts per pass and group of 16 tiles; zero on entry, zeroed again on exit
    uint32_t* bar;       // [5]          control words, zero between launches: [0] arrivals at the barriers of the first sort, [1] arrivals at
                         //              the closing barriers (only ever grows), [2] arrivals at the barriers of a full re-sort,
                         //              [3] "the short sort met a run of equal leading bits it could not finish" (set in the fix-up)
    int short_passes;    // passes of the first sort: 8 = all 60 bits; < 8: only the leading 8 x short_passes bits, then the fix-up
};

constexpr int kFewDigits = 8;   // distinct digits in a row of 32 keys up to which MATCH.ANY beats nine ballots
constexpr int kFixHalo = 64;   // the fix-up of the short sort finishes runs of keys with equal leading bits of at most this length

__device__ __forceinline__ uint64_t dilate20f(uint32_t v) {
    uint64_t x = v & 0xFFFFFu;
    x = (x | (x << 32)) & 0x001F00000000FFFFull;
    x = (x | (x << 16)) & 0x001F0000FF0000FFull;
    x = (x | (x << 8)) & 0x100F00F00F00F00Full;
    x = (x | (x << 4)) & 0x10C30C30C30C30C3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

// (x - lo) * 2^sh truncated and clamped to 20 bits.  The subtraction is the only rounding (O2): `scale` = 2^sh exactly
// when sh is in the normal range (the product of a float and a power of two is exact unless it underflows, and then it is
// < 1 either way); otherwise ldexpf.  cvt.rzi.u32.f32 truncates, sends negatives and NaN to 0 and saturates.
__device__ __forceinline__ uint32_t grid_coordf(float x, float lo, int sh, float scale) {
    const float d = __fsub_rn(x, lo);
    const float s = scale != 0.0f ? __fmul_rn(d, scale) : ldexpf(d, sh);
    return min(__float2uint_rz(s), (1u << kKeyBits) - 1u);
}

// exclusive prefix of v over the first 256 threads of the block (threads >= 256 pass 0); every thread gets
// the prefix of its own index
__device__ __forceinline__ uint32_t block_excl_scan512(uint32_t v, uint32_t* wsum /*[kFrontWarps]*/) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint32_t base = 0;
#pragma unroll
    for (int k = 0; k < kFrontWarps; ++k) {
        const uint32_t s = wsum[k];
        if (k < w) base += s;
    }
    __syncthreads();
    return base + inc - v;
}

__global__ void __launch_bounds__(kFrontThreads, kFrontBlocksPerSM) k_front(const FrontArgs a) {
    extern __shared__ __align__(16) unsigned char xch[];
    uint64_t* skey = reinterpret_cast<uint64_t*>(xch);
    uint32_t* sval = reinterpret_cast<uint32_t*>(xch + kFrontTile * 8);
    __shared__ uint16_t wcnt[kFrontWarps][kRadix];
    __shared__ uint32_t gbase[kRadix], lbase[kRadix], ex2[kFrontParts][kRadix], tot2[kFrontParts][kRadix];
    __shared__ uint32_t wsum[kFrontWarps];
    __shared__ float redf[kFrontWarps][8];
    __shared__ float s_lo[3];
    __shared__ int s_sh;

    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t tile = blockIdx.x, T = gridDim.x, G = (T + 15u) >> 4;
    const int n = a.n;
    const int pw = a.tile_n / kFrontWarps;                                // keys per warp (a multiple of 32)
    const int wbase = (int)tile * a.tile_n + w * pw;                      // warp w owns a contiguous run: order = (warp, iteration, lane)
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t b0 = 0, nbar = 0;                             // barrier bookkeeping (thread 0)
    if (tid == 0) b0 = ld_acquire_u32(a.bar + 1);

    // ---------------------------------------------------------------- S0: box of this tile
    {
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        int bad = 0;
#pragma unroll
        for (int it = 0; it < kFrontItems; ++it) {
            const int i = wbase + it * 32 + lane;
            if (it * 32 < pw && i < n) {
                const float4 p = a.pos_in[i];
                bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w) && p.w > 0.0f);
                mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
                mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
                mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                mn[k] = fminf(mn[k], __shfl_xor_sync(0xFFFFFFFFu, mn[k], o));
                mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xFFFFFFFFu, mx[k], o));
            }
            bad |= __shfl_xor_sync(0xFFFFFFFFu, bad, o);
        }
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { redf[w][k] = mn[k]; redf[w][3 + k] = mx[k]; }
            redf[w][6] = bad ? 1.0f : 0.0f;
        }
        __syncthreads();
        if (tid < 7) {
            float v = redf[0][tid];
            for (int ww = 1; ww < kFrontWarps; ++ww) v = tid < 3 ? fminf(v, redf[ww][tid]) : fmaxf(v, redf[ww][tid]);
            a.part[(size_t)tile * 8 + tid] = v;
        }
    }
    grid_barrier(a.bar, ++nbar * T, a.sc);

    // ---------------------------------------------------------------- domain (every block, redundantly): DESIGN.md O1
    {
        float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
        float bad = 0.0f;
        for (uint32_t t = tid; t < T; t += kFrontThreads) {
            const float4 p0 = __ldcg(reinterpret_cast<const float4*>(a.part + (size_t)t * 8));
            const float4 p1 = __ldcg(reinterpret_cast<const float4*>(a.part + (size_t)t * 8 + 4));
            mn[0] = fminf(mn[0], p0.x); mn[1] = fminf(mn[1], p0.y); mn[2] = fminf(mn[2], p0.z);
            mx[0] = fmaxf(mx[0], p0.w); mx[1] = fmaxf(mx[1], p1.x); mx[2] = fmaxf(mx[2], p1.y);
            bad = fmaxf(bad, p1.z);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                mn[k] = fminf(mn[k], __shfl_xor_sync(0xFFFFFFFFu, mn[k], o));
                mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xFFFFFFFFu, mx[k], o));
            }
            bad = fmaxf(bad, __shfl_xor_sync(0xFFFFFFFFu, bad, o));
        }
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { redf[w][k] = mn[k]; redf[w][3 + k] = mx[k]; }
            redf[w][6] = bad;
        }
        __syncthreads();
        if (tid == 0) {
            float lo[3], hi[3], anybad = 0.0f;
            for (int k = 0; k < 3; ++k) { lo[k] = redf[0][k]; hi[k] = redf[0][3 + k]; }
            for (int ww = 0; ww < kFrontWarps; ++ww) {
                for (int k = 0; k < 3; ++k) { lo[k] = fminf(lo[k], redf[ww][k]); hi[k] = fmaxf(hi[k], redf[ww][3 + k]); }
                anybad = fmaxf(anybad, redf[ww][6]);
            }
            float ext = 0.0f;
            for (int k = 0; k < 3; ++k) ext = fmaxf(ext, __fsub_rn(hi[k], lo[k]));
            int status = anybad > 0.0f ? (int)BH_ERR_NONFINITE : (int)BH_OK;
            if (!isfinite(ext)) { status = (int)BH_ERR_NONFINITE; ext = 1.0f; }
            if (ext == 0.0f) ext = 1.0f;
            int e = 0;
            (void)frexpf(ext, &e);                         // cube side 2^e: the smallest power of two strictly above the extent
            for (int k = 0; k < 3; ++k) s_lo[k] = lo[k];
            s_sh = kKeyBits - e;
            if (tile == 0) {
                for (int k = 0; k < 3; ++k) { a.sc->lo[k] = lo[k]; a.sc->hi[k] = hi[k]; }
                a.sc->dom_e = e;
                a.sc->status = status;
                a.sc->n_cells = 0; a.sc->n_groups = 0; a.sc->n_levels = 0;
                a.bar[3] = 0u;                                  // (nobody looks at it before the fix-up, many barriers from here)
                a.sc->sort_skip = (uint32_t)(kSortPasses - min(a.short_passes, kSortPasses));
            }
        }
        __syncthreads();
    }

    // Two attempts at most.  The first sorts by the leading 8 x short_passes bits of the key only (LSD over those bits,
    // stable) and then finishes every run of keys with equal leading bits in place (the fix-up below); if a run is too long for
    // that, every block learns so at the closing barrier and the second attempt is the full 8-pass sort from the keys made
    // afresh.  Either way the result is THE stable order of the 60-bit keys, in buffer 1.
    const int cnt_tile = min(a.tile_n, n - (int)tile * a.tile_n);
    uint32_t* barw = a.bar;                                   // counter of this attempt's barriers (continues the count of S0's)
    bool gather = a.fuse_reorder != 0;                        // S3 as a gather by the finished permutation (after a full sort)
#pragma unroll 1
    for (int attempt = 0; attempt < 2; ++attempt) {
        const bool full = attempt == 1 || a.short_passes >= kSortPasses;
        const int npass = full ? kSortPasses : a.short_passes;
        const int shift0 = full ? 0 : 60 - kRadixBits * npass;           // the short sort covers bits [shift0, 60)
        const int flip = full ? 0 : (npass - 1) & 1;                      // pass p writes buffer (p + flip) & 1: the last write of an attempt lands in buffer 1
        if (attempt == 1 && tile == 0 && tid == 0) a.sc->sort_retries += 1u;

        // ------------------------------------------------------------ S1: keys, in registers
        uint64_t k[kFrontItems];
        uint32_t v[kFrontItems];
        {
            const float lox = s_lo[0], loy = s_lo[1], loz = s_lo[2];
            const int sh = s_sh;
            const float scale = (sh >= -126 && sh <= 127) ? __int_as_float((127 + sh) << 23) : 0.0f;
#pragma unroll
            for (int it = 0; it < kFrontItems; ++it) {
                const int i = wbase + it * 32 + lane;
                k[it] = 0ull;
                v[it] = (uint32_t)i;
                if (it * 32 < pw && i < n) {
                    const float4 p = a.pos_in[i];
                    k[it] = (dilate20f(grid_coordf(p.x, lox, sh, scale)) << 2) | (dilate20f(grid_coordf(p.y, loy, sh, scale)) << 1) | dilate20f(grid_coordf(p.z, loz, sh, scale));
                }
            }
        }

        // ------------------------------------------------------------ S2: passes of 8 bits
#pragma unroll 1
        for (int pass = 0; pass < npass; ++pass) {
            const int shift = shift0 + pass * kRadixBits;
            const int ob = (pass + flip) & 1;                             // pass p reads what pass p - 1 wrote
            const uint64_t* kin = ob ? a.key0 : a.key1;
            const uint32_t* vin = ob ? a.val0 : a.val1;
            uint64_t* kout = ob ? a.key1 : a.key0;
            uint32_t* vout = ob ? a.val1 : a.val0;
            if (pass > 0) {
#pragma unroll
                for (int it = 0; it < kFrontItems; ++it) {
                    const int i = wbase + it * 32 + lane;
                    const bool ok = it * 32 < pw && i < n;
                    k[it] = ok ? __ldcg(kin + i) : 0ull;
                    v[it] = ok ? __ldcg(vin + i) : 0u;
                }
            }
            for (int j = tid; j < kFrontWarps * kRadix / 2; j += kFrontThreads) reinterpret_cast<uint32_t*>(&wcnt[0][0])[j] = 0u;
            __syncthreads();
            uint32_t rank[kFrontItems];
            bool few = pass > 0;                                               // (warp-uniform)
#pragma unroll
            for (int it = 0; it < kFrontItems; ++it) {
                if (it * 32 >= pw) { rank[it] = 0u; continue; }                // (warp-uniform)
                const int i = wbase + it * 32 + lane;
                const bool ok = i < n;
                const uint32_t d = (uint32_t)(k[it] >> shift) & (kRadix - 1);
                // the lanes of this row with the same digit: MATCH costs one round per distinct value, the ballots a fixed nine
                // votes; the row before says which is cheaper (leading digits of clustered inputs take few values per row)
                uint32_t peers;
                if (few) {
                    peers = __match_any_sync(0xFFFFFFFFu, ok ? d : (uint32_t)kRadix);
                } else {
                    peers = __ballot_sync(0xFFFFFFFFu, ok);
                    if (!ok) peers = ~peers;
#pragma unroll
                    for (int b = 0; b < kRadixBits; ++b) {
                        const bool bit = (d >> b) & 1u;
                        const uint32_t m = __ballot_sync(0xFFFFFFFFu, bit);
                        peers &= bit ? m : ~m;
                    }
                }
                const uint32_t before = __popc(peers & lt);
                few = __popc(__ballot_sync(0xFFFFFFFFu, before == 0u)) <= kFewDigits;
                uint32_t old = 0;
                if (ok) old = wcnt[w][d];
                __syncwarp();
                if (ok && before == 0) wcnt[w][d] = (uint16_t)(old + __popc(peers));
                __syncwarp();
                rank[it] = old + before;
            }
            __syncthreads();
            // digit = tid (first 256 threads): exclusive prefix over the warps, the tile's count; publish it
            uint32_t tcount = 0;
            if (tid < kRadix) {
#pragma unroll
                for (int ww = 0; ww < kFrontWarps; ++ww) {
                    const uint32_t t = wcnt[ww][tid];
                    wcnt[ww][tid] = (uint16_t)tcount;
                    tcount += t;
                }
                a.matrix[(size_t)tile * kRadix + tid] = tcount;
                if (tcount) atomicAdd(a.gsum + ((size_t)pass * kFrontGroupCap + (tile >> 4)) * kRadix + tid, tcount);
            }
            const uint32_t dstart = block_excl_scan512(tcount, wsum);             // first slot of digit d inside the tile, sorted by digit
            grid_barrier(barw, ++nbar * T, a.sc);
            // keys of this digit in the whole input (-> first output slot of the digit) and in the earlier tiles: the sums of the
            // groups of 16 tiles + the rows of the earlier tiles of this tile's own group; split between the two halves of the block
            {
                const int d = tid & (kRadix - 1), h = tid >> 8;
                const uint32_t* gs = a.gsum + (size_t)pass * kFrontGroupCap * kRadix + d;
                const uint32_t myg = tile >> 4;
                uint32_t tot = 0, ex = 0;
#pragma unroll 8
                for (uint32_t g = h; g < G; g += kFrontParts) {
                    const uint32_t x = __ldcg(gs + (size_t)g * kRadix);
                    tot += x;
                    if (g < myg) ex += x;
                }
#pragma unroll 8
                for (uint32_t t = (myg << 4) + h; t < tile; t += kFrontParts) ex += __ldcg(a.matrix + (size_t)t * kRadix + d);
                ex2[h][d] = ex;
                tot2[h][d] = tot;
            }
            __syncthreads();
            uint32_t gh = 0u, exs = 0u;
            if (tid < kRadix) {
#pragma unroll
                for (int hh = 0; hh < kFrontParts; ++hh) { gh += tot2[hh][tid]; exs += ex2[hh][tid]; }
            }
            const uint32_t dbase = block_excl_scan512(gh, wsum);                  // first output slot of digit d
            if (tid < kRadix) {
                gbase[tid] = dbase + exs - dstart;          // output slot = gbase[digit] + slot inside the sorted tile
                lbase[tid] = dstart;
            }
            __syncthreads();
            // exchange through shared memory: the tile leaves sorted by digit, so every digit's run is written contiguously
#pragma unroll
            for (int it = 0; it < kFrontItems; ++it) {
                const int i = wbase + it * 32 + lane;
                if (it * 32 < pw && i < n) {
                    const uint32_t dg = (uint32_t)(k[it] >> shift) & (kRadix - 1);
                    const uint32_t lp = lbase[dg] + wcnt[w][dg] + rank[it];
                    skey[lp] = k[it];
                    sval[lp] = v[it];
                }
            }
            __syncthreads();
#pragma unroll 4
            for (int lp = tid; lp < cnt_tile; lp += kFrontThreads) {
                const uint64_t kk = skey[lp];
                const uint32_t dst = gbase[(uint32_t)(kk >> shift) & (kRadix - 1)] + (uint32_t)lp;
                kout[dst] = kk;
                vout[dst] = sval[lp];
            }
            if (full && pass + 1 == npass) grid_barrier_last(a.bar + 1, b0, (uint32_t)(attempt + 1) * T, barw, a.sc);
            else grid_barrier(barw, ++nbar * T, a.sc);
            if (tile < G && tid < kRadix) a.gsum[((size_t)pass * kFrontGroupCap + tile) * kRadix + tid] = 0u;   // everyone has read it: zero for the next launch
        }
        if (full) break;

        uint32_t src[kFrontItems];                                        // fix-up: where each of this thread's keys comes from / goes to
        int dst[kFrontItems];
        // ------------------------------------------------------------ fix-up of the short sort (buffer 0 -> buffer 1)
        // Buffer 0 is ordered by the leading bits, keys with equal leading bits in their original order.  The stable order of
        // the full keys differs from it only inside each run of equal leading bits: a key goes to (start of its run) + (number
        // of keys of the run that are smaller, or equal and earlier).  A tile reads its own positions plus kFixHalo on either
        // side; a run that reaches the edge of that window, or is longer than 2 x kFixHalo, is left to the full sort.
        {
            const int w0 = (int)tile * a.tile_n;
            const int wlo = max(w0 - kFixHalo, 0), whi = min(w0 + cnt_tile + kFixHalo, n);
            const int wn = max(whi - wlo, 0);
            for (int j = tid; j < wn; j += kFrontThreads) skey[j] = __ldcg(a.key0 + wlo + j);
            __syncthreads();
            bool giveup = false;
#pragma unroll
            for (int it = 0; it < kFrontItems; ++it) {                    // (the permutation entries are requested first: nothing below waits for them)
                const int lp = tid + it * kFrontThreads;
                src[it] = lp < cnt_tile ? __ldcg(a.val0 + w0 + lp) : 0u;
            }
#pragma unroll
            for (int it = 0; it < kFrontItems; ++it) {
                const int lp = tid + it * kFrontThreads;
                dst[it] = -1;
                if (lp >= cnt_tile) continue;
                const int p = w0 - wlo + lp;
                const uint64_t kp = skey[p], top = kp >> shift0;
                int s0 = p;
                while (s0 > 0 && (skey[s0 - 1] >> shift0) == top) --s0;
                if ((s0 == 0 && wlo > 0) || p - s0 > 2 * kFixHalo) giveup = true;
                int r = 0, q = s0;
                for (; q < wn && q - s0 <= 2 * kFixHalo; ++q) {
                    const uint64_t kq = skey[q];
                    if ((kq >> shift0) != top) break;
                    r += (kq < kp || (kq == kp && q < p)) ? 1 : 0;
                }
                if ((q == wn && whi < n) || q - s0 > 2 * kFixHalo) giveup = true;
                dst[it] = wlo + s0 + r;                                   // (inside [wlo, whi) even when this run is given up)
                a.key1[dst[it]] = kp;
                a.val1[dst[it]] = src[it];
            }
            if (giveup) atomicOr(a.bar + 3, 1u);
        }
        grid_barrier_last(a.bar + 1, b0, T, barw, a.sc);
        if (__ldcg(a.bar + 3) == 0u) {                                    // (the same for every thread of the grid; reset by the next launch)
            // S3 as a scatter: the destinations are still in registers; behind the closing barrier, so that the barrier does
            // not wait for these stores
            if (a.fuse_reorder) {
#pragma unroll
                for (int h = 0; h < kFrontItems; h += 4) {                // four gathers in flight per array
                    float4 x[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) if (dst[h + u] >= 0) x[u] = a.pos_in[src[h + u]];
#pragma unroll
                    for (int u = 0; u < 4; ++u) if (dst[h + u] >= 0) a.pos_out[dst[h + u]] = x[u];
#pragma unroll
                    for (int u = 0; u < 4; ++u) if (dst[h + u] >= 0) x[u] = a.vel_in[src[h + u]];
#pragma unroll
                    for (int u = 0; u < 4; ++u) if (dst[h + u] >= 0) a.vel_out[dst[h + u]] = x[u];
                }
                uint32_t y[kFrontItems];
#pragma unroll
                for (int it = 0; it < kFrontItems; ++it) if (dst[it] >= 0) y[it] = a.id_in[src[it]];
#pragma unroll
                for (int it = 0; it < kFrontItems; ++it) if (dst[it] >= 0) a.id_out[dst[it]] = y[it];
            }
            gather = false;
            break;
        }
        barw = a.bar + 2;
        nbar = 0;
    }

    // ---------------------------------------------------------------- S3: gather by the permutation (sorted keys / perm are in buffer 1)
    if (gather) {
#pragma unroll 2
        for (int it = 0; it < kFrontItems; ++it) {
            const int j = wbase + it * 32 + lane;
            if (it * 32 < pw && j < n) {
                const uint32_t src = __ldcg(a.val1 + j);
                a.pos_out[j] = a.pos_in[src];
                a.vel_out[j] = a.vel_in[src];
                a.id_out[j] = a.id_in[src];
            }
        }
    }
}

int front_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_front, cudaFuncAttributeMaxDynamicSharedMemorySize, kFrontTile * 12));
    int per_sm = 0;
    BH_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_front, kFrontThreads, kFrontTile * 12));
    int coop = 0;
    BH_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device));
    c->front_max_tiles = coop ? std::min<int64_t>((int64_t)per_sm * c->sm_count, kFrontTileCap) : 0;
    return BH_OK;
}

bool front_fits(const bh_ctx* c) { return c->front_enabled && div_up(c->n, kFrontTile) <= c->front_max_tiles; }

// Keys per tile: the input spread evenly over every resident block slot (one per SM), in multiples of the block size.
static int front_tile(const bh_ctx* c) {
    const int64_t t = div_up(div_up(c->n, c->front_max_tiles), kFrontThreads) * kFrontThreads;
    return (int)std::min<int64_t>(std::max<int64_t>(t, kFrontThreads), kFrontTile);
}

// Passes of the short sort: the leading floor(log2 n) + 20 bits of the key, in whole digits.  With n particles spread over the
// cube, runs of keys that agree on that many leading bits hold a handful of particles even in the core of a Plummer sphere
// (1 M particles, 40 bits: longest run 5); what is more strongly clustered than that is caught by the fix-up and re-sorted in full.
static int front_short_passes(int64_t n) {
    int lg = 0;
    while ((int64_t(2) << lg) <= n) ++lg;
    return std::min(kSortPasses, (lg + 20 + kRadixBits - 1) / kRadixBits);
}

// S0-S2 (and S3 unless velocities / ids are still arriving on the side stream) in one cooperative launch.
int stage_front(bh_ctx* c, bool fuse_reorder, cudaStream_t s) {
    const int n = (int)c->n;
    const int tile_n = front_tile(c);
    const int tiles = (int)div_up(n, tile_n);
    const int a0 = c->cur, b0 = c->cur ^ 1;
    FrontArgs a;
    a.pos_in = c->ws.pos[a0]; a.vel_in = c->ws.vel[a0]; a.id_in = c->ws.idb[a0];
    a.pos_out = c->ws.pos[b0]; a.vel_out = c->ws.vel[b0]; a.id_out = c->ws.idb[b0];
    a.n = n;
    a.tile_n = tile_n;
    a.fuse_reorder = fuse_reorder ? 1 : 0;
    a.key0 = c->ws.key[0]; a.key1 = c->ws.key[1];
    a.val0 = c->ws.val[0]; a.val1 = c->ws.val[1];
    a.sc = c->ws.sc;
    a.part = c->ws.front_part;
    a.matrix = c->ws.front_matrix;
    a.gsum = c->ws.front_gsum;
    a.bar = c->ws.front_bar;
    a.short_passes = c->front_full ? kSortPasses : front_short_passes(c->n);
    void* args[] = {(void*)&a};
    cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_front, dim3(tiles), dim3(kFrontThreads), args, (size_t)kFrontTile * 12, s);
    c->launches += 1;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return BH_ERR_CUDA; }
    c->sorted = 1;                 // the last write of either attempt lands in buffer 1
    if (fuse_reorder) c->cur = b0;
    return BH_OK;
}

}  // namespace bh
