// keys_sort.cu -- S0 domain box, S1 Morton keys, S2 stable LSD radix sort, S3 reorder, for inputs of any size (inputs whose sort
// tiles are all resident at once take the single cooperative launch of front.cu instead).  S2 is the SHORT sort of DESIGN.md
// section 8: k_sort_passes (all radix passes over the leading key bits in one cooperative launch), k_sort_fix (every run of equal
// leading bits finished in place), and the launches of a full re-sort that return at once unless the fix-up asked for it.
// PAPER.md:374-392 (Appendix B: keys), PAPER.md:350-370 (Appendix A: scan, split, radix sort), PAPER.md:174 ("moving").
#include <algorithm>
#include "bh_internal.cuh"

namespace bh {

// ------------------------------------------------------------------------------------------ S0
__device__ __forceinline__ uint32_t f2ord(float f) {
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord2f(uint32_t u) {
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u);
}

// Also decides how much of the key this build's first sort looks at (the short sort, see k_sort_fix): the tree of the
// previous build on this context had n_levels levels, so keys that agree on 3 n_levels leading bits were at most nleaf then
// (and are few now: particles move little between two builds); the first sort covers those bits in whole digits.  (Fewer
// bits were tried: 3 (n_levels - 2) saves a pass at 16 M but the fix-up's loops over runs of ~17 keys cost more than the pass.)
// No previous tree, an overflowed one, or short_ok = 0: all 8 passes.  A wrong guess costs time, never the result.
__global__ void k_reset_build(DevScalars* sc, int short_ok) {
    const int t = threadIdx.x;
    if (t < 3) { sc->bb_min[t] = 0xFFFFFFFFu; sc->bb_max[t] = 0u; }
    if (t == 0) {
        const uint32_t L = sc->n_levels;
        uint32_t np = kSortPasses;
        if (short_ok && L > 0u) np = min((uint32_t)kSortPasses, (3u * L + kRadixBits - 1u) / kRadixBits);
        sc->sort_skip = kSortPasses - np;
        sc->sort_redo = 0u;
        sc->status = BH_OK; sc->n_cells = 0; sc->n_groups = 0; sc->n_levels = 0;
    }
}

// Which of the two key / permutation buffers the sort of this build starts in, so that its last write lands in buffer 0:
// the first sort makes np = 8 - skip passes plus the fix-up (none when np = 8), the re-sort 8 passes.
__device__ __forceinline__ uint32_t sort_start_buffer(uint32_t skip, int redo) {
    if (redo || skip == 0u) return 0u;
    return (kSortPasses - skip + 1u) & 1u;
}

// Per-axis min / max (exact) and input validation (A27: finite positions, finite mass > 0).
__global__ void __launch_bounds__(256) k_bbox(const float4* __restrict__ pos, int n, DevScalars* sc) {
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    int bad = 0;
    const int stride = gridDim.x * blockDim.x;
    for (int i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < n; i0 += 4 * stride) {
        float4 q[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) q[u] = pos[min(i0 + u * stride, n - 1)];   // four loads in flight (a repeated last particle changes nothing)
#pragma unroll
        for (int u = 0; u < 4; ++u) {
        const float4 p = q[u];
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
    __shared__ float smn[8][3], smx[8][3];
    __shared__ int sbad[8];
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { smn[w][k] = mn[k]; smx[w][k] = mx[k]; }
        sbad[w] = bad;
    }
    __syncthreads();
    if (threadIdx.x < 3) {          // one atomic pair per axis per block
        const int k = threadIdx.x;
        float a = smn[0][k], b = smx[0][k];
#pragma unroll
        for (int ww = 1; ww < 8; ++ww) { a = fminf(a, smn[ww][k]); b = fmaxf(b, smx[ww][k]); }
        atomicMin(&sc->bb_min[k], f2ord(a));
        atomicMax(&sc->bb_max[k], f2ord(b));
    }
    if (threadIdx.x == 32) {
        int any = 0;
#pragma unroll
        for (int ww = 0; ww < 8; ++ww) any |= sbad[ww];
        if (any) atomicMin(&sc->status, (int)BH_ERR_NONFINITE);
    }
}

// Cube side 2^e with frexpf(ext) = (mu, e): the smallest power of two strictly above the extent (O1).
__global__ void k_domain(DevScalars* sc) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    float ext = 0.0f;
    for (int k = 0; k < 3; ++k) {
        const float lo = ord2f(sc->bb_min[k]), hi = ord2f(sc->bb_max[k]);
        sc->lo[k] = lo;
        sc->hi[k] = hi;
        ext = fmaxf(ext, __fsub_rn(hi, lo));
    }
    if (!isfinite(ext)) { atomicMin(&sc->status, (int)BH_ERR_NONFINITE); ext = 1.0f; }
    if (ext == 0.0f) ext = 1.0f;
    int e = 0;
    (void)frexpf(ext, &e);
    sc->dom_e = e;
}

// ------------------------------------------------------------------------------------------ S1
// 20-bit dilate: bit b -> bit 3b (64-bit shift-and-mask form; the paper's List 1 is the 10-bit version).
__device__ __forceinline__ uint64_t dilate20(uint32_t v) {
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
__device__ __forceinline__ uint32_t grid_coord(float x, float lo, int sh, float scale) {
    const float d = __fsub_rn(x, lo);
    const float s = scale != 0.0f ? __fmul_rn(d, scale) : ldexpf(d, sh);
    return min(__float2uint_rz(s), (1u << kKeyBits) - 1u);
}

// Also counts, for every sort pass, how many keys carry each digit value (ghist[pass][digit]): the sort then needs no
// histogram pass of its own.
// redo = 1: the keys again for the full re-sort, only if the fix-up asked for it.
__global__ void __launch_bounds__(256) k_keys(const float4* __restrict__ pos, int n, DevScalars* __restrict__ sc,
                                              uint64_t* __restrict__ key0, uint64_t* __restrict__ key1, uint32_t* __restrict__ val0,
                                              uint32_t* __restrict__ val1, uint32_t* __restrict__ ghist, int redo) {
    if (redo && sc->sort_redo == 0u) return;
    if (redo && blockIdx.x == 0 && threadIdx.x == 0) sc->sort_retries += 1u;
    const uint32_t skip = sc->sort_skip;
    const uint32_t sb = sort_start_buffer(skip, redo);
    uint64_t* __restrict__ key = sb ? key1 : key0;
    uint32_t* __restrict__ val = sb ? val1 : val0;
    __shared__ uint32_t h[kSortPasses * kRadix];
    for (int j = threadIdx.x; j < kSortPasses * kRadix; j += blockDim.x) h[j] = 0;
    __syncthreads();
    const float lox = sc->lo[0], loy = sc->lo[1], loz = sc->lo[2];
    const int sh = kKeyBits - sc->dom_e;
    const float scale = (sh >= -126 && sh <= 127) ? __int_as_float((127 + sh) << 23) : 0.0f;
    const int stride = gridDim.x * blockDim.x;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    float4 pn = i < n ? pos[i] : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    for (; i < n; i += stride) {
        const float4 p = pn;
        if (i + stride < n) pn = pos[i + stride];          // (the next particle is on its way while this one is encoded)
        const uint32_t ix = grid_coord(p.x, lox, sh, scale), iy = grid_coord(p.y, loy, sh, scale), iz = grid_coord(p.z, loz, sh, scale);
        const uint64_t k = (dilate20(ix) << 2) | (dilate20(iy) << 1) | dilate20(iz);   // x most significant in a triple (A4)
        key[i] = k;
        val[i] = (uint32_t)i;
        // digit histograms: of the passes the first sort makes (digits skip..7); the re-sort adds those of the digits below
#pragma unroll
        for (int q = 0; q < kSortPasses; ++q)
            if (redo ? q < (int)skip : q >= (int)skip) atomicAdd(&h[q * kRadix + ((uint32_t)(k >> (q * kRadixBits)) & (kRadix - 1))], 1u);
    }
    __syncthreads();
    for (int j = threadIdx.x; j < kSortPasses * kRadix; j += blockDim.x)
        if (h[j]) atomicAdd(&ghist[j], h[j]);
}

__global__ void k_iota(uint32_t* dst, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = (uint32_t)i;
}

// ------------------------------------------------------------------------------------------ block scan
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
    // returns the exclusive prefix of v over the block
    constexpr int kW = kSortThreads / 32;
    __shared__ uint32_t wsum[kW];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    uint32_t base = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < kW; ++k) {
        const uint32_t s = wsum[k];
        if (k < w) base += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return base + inc - v;
}

// ------------------------------------------------------------------------------------------ S2
// Stable LSD radix sort, 8 bits per pass (the paper's 1-bit split generalised: PAPER.md:352, 362).  The digit
// histograms of the passes were counted while the keys were made (k_keys).  A pass ranks a tile of
// 4096 keys, publishes the tile's digit counts and obtains the counts of all earlier tiles by a decoupled look-back
// (status word = flag | count: AGGREGATE = this tile only, PREFIX = this tile and all before it), so no key is read
// twice and there is no separate histogram or scan launch.  Tiles are numbered by an atomic ticket, so a tile only ever
// waits for tiles whose blocks are already running: the look-back cannot deadlock.
constexpr int kFew = 8;          // a warp whose keys carry at most this many distinct digit values ranks them leader by leader
constexpr int kLook = 8;         // earlier tiles a digit thread reads per round trip of the look-back
constexpr uint32_t kFlagAgg = 1u << 30, kFlagPrefix = 2u << 30, kCountMask = (1u << 30) - 1u;
constexpr uint32_t kSpinLimit = 1u << 22;   // ~1 s of polling

__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(uint32_t* p, uint32_t v) {
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// One tile of one pass.  Warp w of the block owns the contiguous sub-tile [w*256, (w+1)*256): order = (warp, iteration, lane).
// Returns false when the pass has no tile left (every thread of the block gets the same answer).
__device__ __forceinline__ bool radix_tile(const uint64_t* __restrict__ key_in, const uint32_t* __restrict__ val_in, int n, int tiles, int pass,
                                           const uint32_t* __restrict__ ghist, uint32_t* ticket, uint32_t* status,
                                           uint64_t* __restrict__ key_out, uint32_t* __restrict__ val_out, DevScalars* sc) {
    const int shift = pass * kRadixBits;
    constexpr int kWarps = kSortThreads / 32;
    constexpr int kIters = kSortTile / kWarps / 32;   // 16
    __shared__ uint16_t wcnt[kWarps][kRadix];      // (a warp holds kSortTile / kWarps <= 512 keys)
    __shared__ uint32_t gbase[kRadix], lbase[kRadix];
    __shared__ uint32_t s_tile;
    extern __shared__ __align__(16) unsigned char xch[];
    uint64_t* skey = reinterpret_cast<uint64_t*>(xch);
    uint32_t* sval = reinterpret_cast<uint32_t*>(xch + kSortTile * 8);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();                                   // (the previous tile of this block is done with the shared arrays)
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    for (int j = threadIdx.x; j < kWarps * kRadix / 2; j += kSortThreads) reinterpret_cast<uint32_t*>(&wcnt[0][0])[j] = 0u;
    __syncthreads();
    const uint32_t tile = s_tile;
    if (tile >= (uint32_t)tiles) return false;

    const int wbase = (int)tile * kSortTile + w * (kIters * 32);
    const uint32_t lt = (1u << lane) - 1u;
    uint64_t k[kIters];
    uint32_t v[kIters];
    uint32_t rank[kIters];
#pragma unroll
    for (int it = 0; it < kIters; ++it) {
        const int i = wbase + it * 32 + lane;
        const bool ok = i < n;
        k[it] = ok ? key_in[i] : 0ull;
        v[it] = ok ? val_in[i] : 0u;
    }
    bool few = pass >= kSortPasses / 2;              // (warp-uniform)
#pragma unroll
    for (int it = 0; it < kIters; ++it) {
        const int i = wbase + it * 32 + lane;
        const bool ok = i < n;
        const uint32_t d = (uint32_t)(k[it] >> shift) & (kRadix - 1);
        // lanes with the same digit: MATCH costs one round per distinct value, the ballots a fixed nine votes; the row before
        // says which is cheaper (the leading digits of clustered inputs take few values per row of 32 keys)
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
        few = __popc(__ballot_sync(0xFFFFFFFFu, before == 0u)) <= kFew;
        uint32_t old = 0;
        if (ok) old = wcnt[w][d];
        __syncwarp();
        if (ok && before == 0) wcnt[w][d] = (uint16_t)(old + __popc(peers));
        __syncwarp();
        rank[it] = old + before;
    }
    __syncthreads();
    // ---- digit = threadIdx.x (the first 256 threads): exclusive prefix over the warps, the tile's count, and the look-back
    // over earlier tiles
    const uint32_t d = threadIdx.x;
    const bool isd = d < (uint32_t)kRadix;
    uint32_t tcount = 0;
    uint32_t excl = 0;
    if (isd) {
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) {
            const uint32_t t = wcnt[ww][d];
            wcnt[ww][d] = (uint16_t)tcount;
            tcount += t;
        }
        if (tile == 0) {
            st_relaxed(status + d, kFlagPrefix | tcount);
        } else {
            st_relaxed(status + (size_t)tile * kRadix + d, kFlagAgg | tcount);
            // look back kLook tiles per round trip; the words are consumed in order, nearest tile first
            int t = (int)tile - 1;
            uint32_t spins = 0;
            bool done = false;
            while (!done) {
                uint32_t wd[kLook];
#pragma unroll
                for (int j = 0; j < kLook; ++j) wd[j] = (t - j >= 0) ? ld_relaxed(status + (size_t)(t - j) * kRadix + d) : kFlagPrefix;
                int used = 0;
#pragma unroll
                for (int j = 0; j < kLook; ++j) {
                    if (done || used != j) continue;
                    if (wd[j] & kFlagPrefix) { excl += wd[j] & kCountMask; done = true; }
                    else if (wd[j] & kFlagAgg) { excl += wd[j] & kCountMask; used = j + 1; }
                }
                t -= used;                                   // resume at the first tile that had nothing to report yet
                if (!done && used == 0 && ++spins > kSpinLimit) { atomicMin(&sc->status, (int)BH_ERR_CUDA); break; }   // never hang the device
            }
            st_relaxed(status + (size_t)tile * kRadix + d, kFlagPrefix | (excl + tcount));
        }
    }
    uint32_t dummy;
    const uint32_t dbase = block_exclusive_scan(isd ? ghist[d] : 0u, &dummy);   // first output slot of digit d
    const uint32_t dstart = block_exclusive_scan(tcount, &dummy);               // first slot of digit d inside the tile, sorted by digit
    if (isd) {
        gbase[d] = dbase + excl - dstart;                                       // output slot = gbase[digit] + slot inside the sorted tile
        lbase[d] = dstart;
    }
    __syncthreads();
    // ---- exchange through shared memory: the tile leaves sorted by digit, so every digit's run is written contiguously
#pragma unroll
    for (int it = 0; it < kIters; ++it) {
        const int i = wbase + it * 32 + lane;
        if (i < n) {
            const uint32_t dg = (uint32_t)(k[it] >> shift) & (kRadix - 1);
            const uint32_t lp = lbase[dg] + wcnt[w][dg] + rank[it];
            skey[lp] = k[it];
            sval[lp] = v[it];
        }
    }
    __syncthreads();
    const int cnt = min(kSortTile, n - (int)tile * kSortTile);
#pragma unroll 4
    for (int lp = threadIdx.x; lp < cnt; lp += kSortThreads) {
        const uint64_t kk = skey[lp];
        const uint32_t dst = gbase[(uint32_t)(kk >> shift) & (kRadix - 1)] + (uint32_t)lp;
        key_out[dst] = kk;
        val_out[dst] = sval[lp];
    }
    return true;
}

// All passes of a sort in ONE cooperative launch: the first sort (redo = 0: the passes from digit sort_skip up) or the full
// re-sort (redo = 1: returns at once unless the fix-up asked for it).  The resident blocks draw tiles from the pass's ticket
// counter until it runs out (a tile only ever waits for tiles with smaller tickets, whose blocks are running: the look-back
// cannot deadlock), then meet at a grid barrier: the next pass reads what this one scattered.  Buffers alternate from
// sort_start_buffer().  (One launch per pass cost ~4 us per launch, and the number of passes is only known on the device:
// eight launches for the first sort and nine for the re-sort, most of them returning at once.)
__global__ void __launch_bounds__(kSortThreads, 2) k_sort_passes(uint64_t* key0, uint64_t* key1, uint32_t* val0, uint32_t* val1, int n, int tiles, int redo,
                                                              const uint32_t* __restrict__ ghist, uint32_t* ticket, uint32_t* status,
                                                              DevScalars* sc, uint32_t* bar /* [2]: arrivals, closing arrivals */) {
    const uint32_t skip = redo ? 0u : sc->sort_skip;
    if (redo && sc->sort_redo == 0u) return;                                   // (the whole grid, before any barrier)
    uint32_t b0 = 0, nbar = 0;
    if (threadIdx.x == 0) b0 = ld_acquire_u32(bar + 1);
    const uint32_t sb = sort_start_buffer(skip, redo);
#pragma unroll 1
    for (int pass = (int)skip; pass < kSortPasses; ++pass) {
        const uint32_t ib = (sb + (uint32_t)pass - skip) & 1u;
        const uint64_t* key_in = ib ? key1 : key0;
        const uint32_t* val_in = ib ? val1 : val0;
        uint64_t* key_out = ib ? key0 : key1;
        uint32_t* val_out = ib ? val0 : val1;
        while (radix_tile(key_in, val_in, n, tiles, pass, ghist + pass * kRadix, ticket + pass, status + (size_t)pass * kRadix * tiles, key_out, val_out, sc)) {}
        if (pass + 1 < kSortPasses) grid_barrier(bar, ++nbar * gridDim.x, sc);
        else grid_barrier_last(bar + 1, b0, gridDim.x, bar, sc);              // (puts bar[0] back to zero for the next launch)
    }
}

// The fix-up of the short sort.  After the passes over the digits above bit 8 skip, buffer 1 is ordered by those leading bits,
// keys with equal leading bits in their original order; the stable order of the full keys differs from it only inside each
// run of equal leading bits: a key goes to (start of its run) + (number of keys of the run that are smaller, or equal and
// earlier).  A tile of 4096 positions reads kFixHaloBig more on either side; a run that reaches the edge of that window (or
// is longer than twice the halo) cannot be finished here: sort_redo makes the kernels that follow sort again, in full.
constexpr int kFixHaloBig = 256;
__global__ void __launch_bounds__(kSortThreads) k_sort_fix(const uint64_t* __restrict__ kin, const uint32_t* __restrict__ vin, int n,
                                                           uint64_t* __restrict__ kout, uint32_t* __restrict__ vout, DevScalars* sc) {
    const uint32_t skip = sc->sort_skip;
    if (skip == 0u) return;
    const int cut = (int)skip * kRadixBits;
    __shared__ uint64_t skey[kSortTile + 2 * kFixHaloBig];
    const int w0 = (int)blockIdx.x * kSortTile;
    const int own = min(kSortTile, n - w0);
    const int wlo = max(w0 - kFixHaloBig, 0), whi = min(w0 + own + kFixHaloBig, n);
    const int wn = whi - wlo;
    for (int j = threadIdx.x; j < wn; j += kSortThreads) skey[j] = kin[wlo + j];
    __syncthreads();
    bool giveup = false;
    for (int lp = threadIdx.x; lp < own; lp += kSortThreads) {
        const int p = w0 - wlo + lp;
        const uint64_t kp = skey[p], top = kp >> cut;
        int s0 = p;
        while (s0 > 0 && p - s0 <= 2 * kFixHaloBig && (skey[s0 - 1] >> cut) == top) --s0;
        if ((s0 == 0 && wlo > 0) || p - s0 > 2 * kFixHaloBig) giveup = true;
        int r = 0, q = s0;
        for (; q < wn && q - s0 <= 2 * kFixHaloBig; ++q) {
            const uint64_t kq = skey[q];
            if ((kq >> cut) != top) break;
            r += (kq < kp || (kq == kp && q < p)) ? 1 : 0;
        }
        if ((q == wn && whi < n) || q - s0 > 2 * kFixHaloBig) giveup = true;
        const int dst = wlo + s0 + r;                                    // (inside [wlo, whi) even when this run is given up)
        kout[dst] = kp;
        vout[dst] = vin[w0 + lp];
    }
    if (giveup) atomicOr(&sc->sort_redo, 1u);
}

int sort_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_sort_passes, cudaFuncAttributeMaxDynamicSharedMemorySize, kSortTile * 12));
    int per_sm = 0;
    BH_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sort_passes, kSortThreads, kSortTile * 12));
    int coop = 0;
    BH_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device));
    if (!coop || per_sm < 1) return BH_ERR_CUDA;
    c->sort_grid = per_sm * c->sm_count;
    return BH_OK;
}

// ------------------------------------------------------------------------------------------ S3
__global__ void __launch_bounds__(256) k_reorder(const uint32_t* __restrict__ perm, int n,
                                                 const float4* __restrict__ pos_in, const float4* __restrict__ vel_in,
                                                 const uint32_t* __restrict__ id_in,
                                                 float4* __restrict__ pos_out, float4* __restrict__ vel_out, uint32_t* __restrict__ id_out) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const uint32_t src = perm[j];
    pos_out[j] = pos_in[src];
    vel_out[j] = vel_in[src];
    id_out[j] = id_in[src];
}

// ------------------------------------------------------------------------------------------ host side
int stage_iota(bh_ctx* c, uint32_t* dst, int64_t n, cudaStream_t s) {
    BH_LAUNCH(c, k_iota, (unsigned)div_up(n, 256), 256, 0, s, dst, (int)n);
    return BH_OK;
}

int stage_bbox_keys(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    BH_LAUNCH(c, k_reset_build, 1, 32, 0, s, c->ws.sc, c->front_full ? 0 : 1);
    // sort bookkeeping (digit histograms, tile tickets, look-back status words of every pass): one memset per build
    const int tiles = (int)div_up(n, kSortTile);
    BH_CUDA(c, cudaMemsetAsync(c->ws.sort_ghist, 0, sizeof(uint32_t) * sort_words(tiles), s));
    const int grid = (int)std::min<int64_t>(div_up(n, 256 * 4), (int64_t)c->sm_count * 8);
    BH_LAUNCH(c, k_bbox, grid, 256, 0, s, c->ws.pos[c->cur], n, c->ws.sc);
    BH_LAUNCH(c, k_domain, 1, 32, 0, s, c->ws.sc);
    if (c->timing) stage_mark(c, 1, s);
    const int kgrid = (int)std::min<int64_t>(div_up(n, 256), (int64_t)c->sm_count * 8);
    BH_LAUNCH(c, k_keys, kgrid, 256, 0, s, c->ws.pos[c->cur], n, c->ws.sc, c->ws.key[0], c->ws.key[1], c->ws.val[0], c->ws.val[1], c->ws.sort_ghist, 0);
    return BH_OK;
}

// The first sort (as many passes as k_reset_build decided, in one cooperative launch, then the fix-up), and the launches of
// the full re-sort, which return at once unless the fix-up asked for it: the sequence of launches does not depend on the data
// (no host round trip; capturable), and the result is in buffer 0 either way.
static int launch_sort_passes(bh_ctx* c, int redo, cudaStream_t s) {
    const Ws& w = c->ws;
    int n = (int)c->n, tiles = (int)div_up(c->n, kSortTile);
    uint64_t *k0 = w.key[0], *k1 = w.key[1];
    uint32_t *v0 = w.val[0], *v1 = w.val[1];
    const uint32_t* gh = w.sort_ghist;
    uint32_t* ticket = w.sort_ticket + redo * kSortPasses;
    uint32_t* status = w.sort_status + (size_t)redo * kSortPasses * kRadix * tiles;
    DevScalars* sc = w.sc;
    uint32_t* bar = w.front_ctl + 5;
    void* args[] = {&k0, &k1, &v0, &v1, &n, &tiles, &redo, &gh, &ticket, &status, &sc, &bar};
    const int grid = std::min(c->sort_grid, tiles);
    cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_sort_passes, dim3(grid), dim3(kSortThreads), args, (size_t)kSortTile * 12, s);
    c->launches += 1;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return BH_ERR_CUDA; }
    return BH_OK;
}

int stage_sort(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    const int tiles = (int)div_up(n, kSortTile);
    const Ws& w = c->ws;
    int rc = launch_sort_passes(c, 0, s);
    if (rc != BH_OK) return rc;
    BH_LAUNCH(c, k_sort_fix, tiles, kSortThreads, 0, s, w.key[1], w.val[1], n, w.key[0], w.val[0], w.sc);
    const int kgrid = (int)std::min<int64_t>(div_up(n, 256), (int64_t)c->sm_count * 8);
    BH_LAUNCH(c, k_keys, kgrid, 256, 0, s, w.pos[c->cur], n, w.sc, w.key[0], w.key[1], w.val[0], w.val[1], w.sort_ghist, 1);
    if ((rc = launch_sort_passes(c, 1, s)) != BH_OK) return rc;
    c->sorted = 0;
    return BH_OK;
}

int stage_reorder(bh_ctx* c, cudaStream_t s) {
    const int n = (int)c->n;
    const int a = c->cur, b = c->cur ^ 1;
    BH_LAUNCH(c, k_reorder, (unsigned)div_up(n, 256), 256, 0, s, c->ws.val[c->sorted], n, c->ws.pos[a], c->ws.vel[a],
              c->ws.idb[a], c->ws.pos[b], c->ws.vel[b], c->ws.idb[b]);
    c->cur = b;
    return BH_OK;
}

}  // namespace bh
