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
//   * accepted cells are staged in a shared-memory ring; opened leaves contribute their particles to a second ring;
//     whenever a ring holds 32 entries the warp sweeps them.
//   * the group's own particles are skipped while staging and handled by a final self block with j != i (A19).
//
// Evaluation layout (what differs from the paper's one-thread-per-particle sweep, and why):
//   (1) Lane use.  A group holds n <= 64 targets (mean ~19), so "one target per lane" idles ~half of the warp.  The
//       paper's remedy is up to 4 threads per particle (L81, L97); here it is taken to its end: n is rounded up to a
//       multiple of 4 and split in binary, 64 | 32 + 16 + 8 + 4 -> "slots" of T = 2^K targets.  In a slot a lane serves
//       TWO targets, (l mod T/2) and (l mod T/2) + T/2, and sub-list (l div T/2): the 64 / T sub-lists interleave the ring
//       entries, and a butterfly of shuffles adds the sub-list sums at the end of the group (>= 93 % useful lanes).
//   (2) FP32 rate.  On sm_100a scalar FFMA issues at half rate; the full 128 lanes/clk/SM needs the packed f32x2 forms
//       (FFMA2/FMUL2/FADD2, measured 71.8 vs 37-45 TFLOP/s).  The rings therefore store PAIRS of entries interleaved
//       (x0, x1, y0, y1, ...), one LDS.128 yields two packed operands, and each lane evaluates two list entries per
//       instruction for each of its targets.
//   (3) Shared-memory delivery.  An LDS.128 moves 512 B into the register file whether or not the lanes share the address,
//       i.e. 4 cycles of the 128 B/clk path: six loads per entry pair for ONE target per lane make the loop smem-bound at
//       ~73 % of the FMA rate (measured 50 TFLOP/s).  Two targets per loaded pair halve that traffic (measured 60 TFLOP/s).
//   Running sums per slot live in shared memory between sweeps (partial sums of a sweep are formed in registers and added
//   once: accuracy, and the kernel stays inside 128 registers at 16 warps/SM).
// Forces: Plummer-softened p-p, and p-c with monopole + quadrupole (second-order expansion of the softened kernel,
// DESIGN.md O10): 35 packed fp32 operations + 2 MUFU.RSQ per PAIR of p-c interactions, 13 + 2 per pair of p-p.
#include <algorithm>
#include <cstdlib>
#include "bh_internal.cuh"

namespace bh {

constexpr int kWalkWarps = 8;
constexpr int kWalkThreads = kWalkWarps * 32;
constexpr int kStackCap = 1024;
constexpr int kStackReserve = 160;   // >= 7 * 20 + 7: room for a pure depth-first descent
constexpr int kRing = 64;            // ring capacity in entries (power of two, >= 63)
constexpr int kRingPairs = kRing / 2;
constexpr int kPcPair = 28;          // floats per p-c pair: 12 fields x 2 + 4 pad (112 B stride: no bank conflict for 8 pairs)
constexpr int kPpPair = 8;           // floats per p-p pair: x0 x1 y0 y1 z0 z1 m0 m1

// p-c pair fields f = 0..11: x y z M | Qm_xx Qm_yy Qm_zz Qm_xy | Qm_xz Qm_yz nTh n3Th, with Qm = -3 Q, nTh = -T/2,
// n3Th = -3T/2; entry e lives in pair e >> 1, half e & 1, at float index pair * kPcPair + 2 f + half.
constexpr int kMaxSlots = 4;         // 32 + 16 + 8 + 4 (or the single 64-target slot)
struct __align__(16) WarpShared {
    float pc[kRingPairs * kPcPair];
    float pp[kRingPairs * kPpPair];
    float4 own[64];                  // the group's particles (targets; sources of the self block)
    float4 tot[kMaxSlots][2][32];    // running sums per slot, target-of-lane, lane: (ax, ay, az, -phi)
    uint32_t stack[kStackCap];
    uint32_t run_begin[32];
    uint32_t run_off[36];
};

typedef unsigned long long f2;   // two fp32 values in one 64-bit register: low word = even entry, high word = odd entry

__device__ __forceinline__ f2 pk(float lo, float hi) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk(f2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ f2 rsqrt2(f2 v) { float lo, hi; upk(v, lo, hi); return pk(rsqrt_approx(lo), rsqrt_approx(hi)); }

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

struct Consts { f2 e2, mhalf, m2p5; };

// The slots of a group are the set bits K = 6 (alone) or 5..2 of m = roundup4(n): a slot of 2^K targets each.  They are
// enumerated on the fly (slot index = rank of the bit from the top, first target = sum of the higher bits).
struct Acc2 { f2 ax, ay, az, p; };

__device__ __forceinline__ void acc_flush(float4* tot, const Acc2& a) {
    float4 t = *tot;
    float lo, hi;
    upk(a.ax, lo, hi); t.x += lo + hi;
    upk(a.ay, lo, hi); t.y += lo + hi;
    upk(a.az, lo, hi); t.z += lo + hi;
    upk(a.p, lo, hi); t.w += lo + hi;
    *tot = t;
}

// p-c sweep of one slot over `npairs` ring pairs starting at pair `hp`.  Lane: targets t0, t1; pairs sub, sub + S, ...
//   -phi += M/rho + nTh/rho^3 - w/(2 rho^5),                 q = Qm dr = -3 Q dr,  w = dr.q
//   a    += dr (M/rho^3 + n3Th/rho^5 - 5 w/(2 rho^7)) + q/rho^5
__device__ __forceinline__ void pc_one(const ulonglong2& v0, const ulonglong2& v1, const ulonglong2& v2, const ulonglong2& v3,
                                       const ulonglong2& v4, const ulonglong2& v5, f2 ntx, f2 nty, f2 ntz, const Consts& k, Acc2& a) {
    const f2 dx = add2(v0.x, ntx), dy = add2(v0.y, nty), dz = add2(v1.x, ntz);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
    const f2 ri = rsqrt2(r2);
    const f2 ri2 = mul2(ri, ri), ri3 = mul2(ri, ri2), ri5 = mul2(ri3, ri2);
    const f2 qx = fma2(v2.x, dx, fma2(v3.y, dy, mul2(v4.x, dz)));
    const f2 qy = fma2(v3.y, dx, fma2(v2.y, dy, mul2(v4.y, dz)));
    const f2 qz = fma2(v4.x, dx, fma2(v4.y, dy, mul2(v3.x, dz)));
    const f2 w = fma2(dx, qx, fma2(dy, qy, mul2(dz, qz)));
    const f2 t = mul2(w, ri5);
    a.p = fma2(v1.y, ri, fma2(v5.x, ri3, fma2(t, k.mhalf, a.p)));
    const f2 br = fma2(mul2(t, ri2), k.m2p5, fma2(v5.y, ri5, mul2(v1.y, ri3)));
    a.ax = fma2(qx, ri5, fma2(dx, br, a.ax));
    a.ay = fma2(qy, ri5, fma2(dy, br, a.ay));
    a.az = fma2(qz, ri5, fma2(dz, br, a.az));
}

__device__ __forceinline__ void eval_pc_slot(WarpShared* ws, int hp, int npairs, int K, int tbase, int slot, int ng, const Consts& k,
                                             int lane) {
    const int L = 1 << (K - 1), sub = lane >> (K - 1), S = 32 >> (K - 1);
    const int t0 = tbase + (lane & (L - 1)), t1 = t0 + L;
    const float4 T0 = ws->own[min(t0, ng - 1)], T1 = ws->own[min(t1, ng - 1)];   // idle targets shadow the last particle
    const f2 ntx0 = pk(-T0.x, -T0.x), nty0 = pk(-T0.y, -T0.y), ntz0 = pk(-T0.z, -T0.z);
    const f2 ntx1 = pk(-T1.x, -T1.x), nty1 = pk(-T1.y, -T1.y), ntz1 = pk(-T1.z, -T1.z);
    Acc2 a0 = {0ull, 0ull, 0ull, 0ull}, a1 = {0ull, 0ull, 0ull, 0ull};
    for (int p = sub; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ws->pc + ((hp + p) & (kRingPairs - 1)) * kPcPair);
        const ulonglong2 v0 = src[0], v1 = src[1], v2 = src[2], v3 = src[3], v4 = src[4], v5 = src[5];
        pc_one(v0, v1, v2, v3, v4, v5, ntx0, nty0, ntz0, k, a0);
        pc_one(v0, v1, v2, v3, v4, v5, ntx1, nty1, ntz1, k, a1);
    }
    acc_flush(&ws->tot[slot][0][lane], a0);
    acc_flush(&ws->tot[slot][1][lane], a1);
}

// p-p sweep.  kSelf: the ring holds the group's own `ng` particles from entry 0 and entry j is target index j: skip j == t
// and the massless pad entry j >= ng (it sits ON the last own particle: r = 0 would give 0 * inf when eps = 0).
template <bool kSelf>
__device__ __forceinline__ void pp_one(const ulonglong2& v0, const ulonglong2& v1, f2 ntx, f2 nty, f2 ntz, const Consts& k, Acc2& a,
                                       int j0, int tidx, int ng) {
    const f2 dx = add2(v0.x, ntx), dy = add2(v0.y, nty), dz = add2(v1.x, ntz);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
    f2 ri;
    if (kSelf) {
        float lo, hi;
        upk(r2, lo, hi);
        lo = (j0 == tidx) ? 0.0f : rsqrt_approx(lo);
        hi = (j0 + 1 == tidx || j0 + 1 >= ng) ? 0.0f : rsqrt_approx(hi);
        ri = pk(lo, hi);
    } else {
        ri = rsqrt2(r2);
    }
    const f2 ri2 = mul2(ri, ri);
    const f2 mr = mul2(v1.y, ri);
    const f2 mr3 = mul2(mr, ri2);
    a.p = add2(a.p, mr);
    a.ax = fma2(dx, mr3, a.ax);
    a.ay = fma2(dy, mr3, a.ay);
    a.az = fma2(dz, mr3, a.az);
}

template <bool kSelf>
__device__ __forceinline__ void eval_pp_slot(WarpShared* ws, int hp, int npairs, int K, int tbase, int slot, int ng, const Consts& k,
                                             int lane) {
    const int L = 1 << (K - 1), sub = lane >> (K - 1), S = 32 >> (K - 1);
    const int t0 = tbase + (lane & (L - 1)), t1 = t0 + L;
    const float4 T0 = ws->own[min(t0, ng - 1)], T1 = ws->own[min(t1, ng - 1)];
    const f2 ntx0 = pk(-T0.x, -T0.x), nty0 = pk(-T0.y, -T0.y), ntz0 = pk(-T0.z, -T0.z);
    const f2 ntx1 = pk(-T1.x, -T1.x), nty1 = pk(-T1.y, -T1.y), ntz1 = pk(-T1.z, -T1.z);
    Acc2 a0 = {0ull, 0ull, 0ull, 0ull}, a1 = {0ull, 0ull, 0ull, 0ull};
    for (int p = sub; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ws->pp + ((hp + p) & (kRingPairs - 1)) * kPpPair);
        const ulonglong2 v0 = src[0], v1 = src[1];
        pp_one<kSelf>(v0, v1, ntx0, nty0, ntz0, k, a0, 2 * p, t0, ng);
        pp_one<kSelf>(v0, v1, ntx1, nty1, ntz1, k, a1, 2 * p, t1, ng);
    }
    acc_flush(&ws->tot[slot][0][lane], a0);
    acc_flush(&ws->tot[slot][1][lane], a1);
}

#ifdef BH_WALK_DEBUG   // experiment hook (never in the product build): bit 0 skips p-c sweeps, bit 1 p-p sweeps, bit 2 the record loads
__device__ int g_dbg = 0;
#define BH_DBG(bit) (g_dbg & (bit))
#else
#define BH_DBG(bit) false
#endif
__device__ __forceinline__ void eval_pc_all(WarpShared* ws, int hp, int npairs, int m, int ng, const Consts& k, int lane) {
    if (BH_DBG(1)) return;
    int slot = 0, base = 0;
#pragma unroll
    for (int K = 6; K >= 2; --K)
        if (m & (1 << K)) { eval_pc_slot(ws, hp, npairs, K, base, slot, ng, k, lane); ++slot; base += 1 << K; }
}
template <bool kSelf>
__device__ __forceinline__ void eval_pp_all(WarpShared* ws, int hp, int npairs, int m, int ng, const Consts& k, int lane) {
    if (BH_DBG(2)) return;
    int slot = 0, base = 0;
#pragma unroll
    for (int K = 6; K >= 2; --K)
        if (m & (1 << K)) { eval_pp_slot<kSelf>(ws, hp, npairs, K, base, slot, ng, k, lane); ++slot; base += 1 << K; }
}

// Add the sub-list sums of a slot (lanes that share l mod T/2) and store its targets.
__device__ __forceinline__ void slot_finish(WarpShared* ws, int slot, int K, int tbase, int lane, int ng, uint32_t gb,
                                            float4* __restrict__ acc_out) {
    const int L = 1 << (K - 1);
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        float4 t = ws->tot[slot][r][lane];
        for (int o = L; o < 32; o <<= 1) {
            t.x += __shfl_xor_sync(0xFFFFFFFFu, t.x, o);
            t.y += __shfl_xor_sync(0xFFFFFFFFu, t.y, o);
            t.z += __shfl_xor_sync(0xFFFFFFFFu, t.z, o);
            t.w += __shfl_xor_sync(0xFFFFFFFFu, t.w, o);
        }
        const int idx = tbase + r * L + lane;
        if (lane < L && idx < ng) acc_out[gb + idx] = make_float4(t.x, t.y, t.z, -t.w);
    }
}

__device__ __forceinline__ void pc_store(float* ring, int e, float x, float y, float z, float M, float qxx, float qyy, float qzz,
                                         float qxy, float qxz, float qyz, float nth, float n3th) {
    float* d = ring + (e >> 1) * kPcPair + (e & 1);
    d[0] = x; d[2] = y; d[4] = z; d[6] = M; d[8] = qxx; d[10] = qyy; d[12] = qzz; d[14] = qxy; d[16] = qxz; d[18] = qyz;
    d[20] = nth; d[22] = n3th;
}
__device__ __forceinline__ void pp_store(float* ring, int e, float x, float y, float z, float m) {
    float* d = ring + (e >> 1) * kPpPair + (e & 1);
    d[0] = x; d[2] = y; d[4] = z; d[6] = m;
}
// An odd tail gets a massless partner at the position of the last real entry (a position no target can coincide with).
__device__ __forceinline__ void pc_pad(float* ring, int e_last) {
    const float* s = ring + (e_last >> 1) * kPcPair + (e_last & 1);
    pc_store(ring, (e_last + 1) & (kRing - 1), s[0], s[2], s[4], 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f);
}
__device__ __forceinline__ void pp_pad(float* ring, int e_last) {
    const float* s = ring + (e_last >> 1) * kPpPair + (e_last & 1);
    pp_store(ring, (e_last + 1) & (kRing - 1), s[0], s[2], s[4], 0.f);
}

__device__ __noinline__ void walk_group(WarpShared* ws, const int lane, const uint32_t g, const uint32_t gb, const uint32_t ge,
                                        const float4* __restrict__ pos, const float4* __restrict__ rec, const size_t rstride, float eps2,
                                        float4* __restrict__ acc_out, uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp,
                                        DevScalars* sc) {
    const uint32_t lt = (1u << lane) - 1u;
    const int ng = (int)(ge - gb);
    Consts k;
    k.e2 = pk(eps2, eps2);
    k.mhalf = pk(-0.5f, -0.5f);
    k.m2p5 = pk(-2.5f, -2.5f);

    // ---- the group's own particles (shared memory) and tight box (A13)
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        const float4 p = __ldg(pos + gb + min(idx, ng - 1));
        if (idx < ng) ws->own[idx] = p;
        mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
        mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
        mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            mn[a] = fminf(mn[a], __shfl_xor_sync(0xFFFFFFFFu, mn[a], o));
            mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xFFFFFFFFu, mx[a], o));
        }

    // ---- slots: n rounded up to a multiple of 4, split as 64 | 32 + 16 + 8 + 4
    const int m = (ng + 3) & ~3;
#pragma unroll
    for (int i = 0; i < kMaxSlots; ++i) {
        ws->tot[i][0][lane] = make_float4(0.f, 0.f, 0.f, 0.f);
        ws->tot[i][1][lane] = make_float4(0.f, 0.f, 0.f, 0.f);
    }

    int sp = 1;
    if (lane == 0) ws->stack[0] = 0u;   // the root (A17)
    __syncwarp();
    int pc_head = 0, pc_cnt = 0, pp_head = 0, pp_cnt = 0;   // heads are even (entries are consumed 32 at a time)
    uint32_t npc = 0, npp = 0, nmac = 0;

    // The batch under test is loaded ONE ITERATION AHEAD: its 64 B records are requested right after the previous
    // batch has been classified, and full rings are evaluated while those loads are in flight.
    int kcur = 0;
    bool valid = false;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0, r3 = r0;
    auto pop_and_load = [&]() {
        kcur = 0;
        valid = false;
        if (sp > 0) {
            int kpop = (kStackCap - kStackReserve - sp) / 7;
            kpop = max(1, min(kpop, 32));
            kpop = min(kpop, sp);
            valid = lane < kpop;
            if (valid) {
                const float4* rp = rec + ws->stack[sp - 1 - lane];
                r0 = __ldg(rp); r1 = __ldg(rp + rstride); r2 = __ldg(rp + 2 * rstride); r3 = __ldg(rp + 3 * rstride);
            }
            sp -= kpop;
            nmac += (uint32_t)kpop;
            kcur = kpop;
        }
        __syncwarp();
    };
    pop_and_load();

    while (kcur > 0) {
        bool accept = false, isleaf = false, isnode = false;
        uint32_t first = 0, cnt = 0;
        if (valid) {
            const float dx = fmaxf(fmaxf(__fsub_rn(mn[0], r0.x), __fsub_rn(r0.x, mx[0])), 0.0f);
            const float dy = fmaxf(fmaxf(__fsub_rn(mn[1], r0.y), __fsub_rn(r0.y, mx[1])), 0.0f);
            const float dz = fmaxf(fmaxf(__fsub_rn(mn[2], r0.z), __fsub_rn(r0.z, mx[2])), 0.0f);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            accept = d2 > r0.w;
            if (!accept) {
                first = __float_as_uint(r3.x);
                cnt = __float_as_uint(r3.y);
                isleaf = __float_as_uint(r3.z) != 0u;
                isnode = !isleaf;
            }
        }
        // ---- accepted cells -> p-c ring (the record is already in the ring's units: a plain copy)
        const uint32_t amask = __ballot_sync(0xFFFFFFFFu, accept);
        if (amask) {
            if (accept) {
                const int e = (pc_head + pc_cnt + __popc(amask & lt)) & (kRing - 1);
                pc_store(ws->pc, e, r0.x, r0.y, r0.z, r1.x, r1.y, r1.z, r1.w, r2.x, r2.y, r2.z, r2.w, r3.w);
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
            if (sp + total > kStackCap) {            // cannot happen (see header); never write out of bounds
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
                    eval_pp_all<false>(ws, pp_head >> 1, 16, m, ng, k, lane);
                    pp_head = (pp_head + 32) & (kRing - 1);
                    pp_cnt -= 32;
                    __syncwarp();
                }
            }
            __syncwarp();
        }
        // ---- request the next batch, then sweep a full p-c ring while those loads are in flight
        pop_and_load();
        if (pc_cnt >= 32) {
            eval_pc_all(ws, pc_head >> 1, 16, m, ng, k, lane);
            pc_head = (pc_head + 32) & (kRing - 1);
            pc_cnt -= 32;
            __syncwarp();
        }
    }
    // ---- flush the rings (an odd tail gets a massless partner)
    if (pc_cnt > 0) {
        if ((pc_cnt & 1) && lane == 0) pc_pad(ws->pc, (pc_head + pc_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pc_all(ws, pc_head >> 1, (pc_cnt + 1) >> 1, m, ng, k, lane);
    }
    if (pp_cnt > 0) {
        if ((pp_cnt & 1) && lane == 0) pp_pad(ws->pp, (pp_head + pp_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pp_all<false>(ws, pp_head >> 1, (pp_cnt + 1) >> 1, m, ng, k, lane);
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
    eval_pp_all<true>(ws, 0, (ng + 1) >> 1, m, ng, k, lane);
    __syncwarp();
    // ---- add the sub-list sums and store
    {
        int slot = 0, base = 0;
#pragma unroll
        for (int K = 6; K >= 2; --K)
            if (m & (1 << K)) { slot_finish(ws, slot, K, base, lane, ng, gb, acc_out); ++slot; base += 1 << K; }
    }
    __syncwarp();
    if (lane == 0) {
        g_npc[g] = npc;
        g_npp[g] = npp;
        atomicAdd(&sc->sum_pc, (unsigned long long)npc * (unsigned long long)ng);
        atomicAdd(&sc->sum_pp, (unsigned long long)npp * (unsigned long long)ng);
        atomicAdd(&sc->sum_mac, (unsigned long long)nmac);
    }
}

__global__ void __launch_bounds__(kWalkThreads, 2) k_walk(DevScalars* sc, const float4* __restrict__ pos, const float4* __restrict__ rec, size_t rstride,
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
        walk_group(ws, lane, g, gb, ge, pos, rec, rstride, eps2, acc_out, g_npc, g_npp, sc);
        __syncwarp();
    }
}

__global__ void k_reset_counters(DevScalars* sc) {
    if (threadIdx.x == 0) { sc->walk_next = 0; sc->sum_pc = 0; sc->sum_pp = 0; sc->sum_mac = 0; }
}

int walk_init(bh_ctx* c) {
#ifdef BH_WALK_DEBUG
    { const char* e = getenv("BH_WALK_DBG"); int v = e ? atoi(e) : 0; cudaMemcpyToSymbol(g_dbg, &v, sizeof(int)); }
#endif
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
    BH_LAUNCH(c, k_walk, grid, kWalkThreads, smem, s, c->ws.sc, c->ws.pos[c->cur], c->ws.rec, (size_t)c->max_cells, c->ws.g_begin, eps * eps, c->ws.acc,
              c->ws.g_npc, c->ws.g_npp);
    if (c->timing) cudaEventRecord(c->ev[10], s);
    return BH_OK;
}

}  // namespace bh
