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
//       multiple of 4 and split in binary, 32 + 32 + 16 + 8 + 4 -> "slots" with T = 2^K targets each.  In a slot,
//       lane l serves target (l mod T) and sub-list (l div T): the 32 / T sub-lists interleave the ring entries, and a
//       butterfly of shuffles adds the sub-list sums at the end of the group.  Every lane does useful work (>= 93 %).
//   (2) FP32 rate.  On sm_100a scalar FFMA issues at half rate; the full 128 lanes/clk/SM needs the packed f32x2 forms
//       (FFMA2/FMUL2/FADD2, measured 71.8 vs 37-45 TFLOP/s).  The rings therefore store PAIRS of entries interleaved
//       (x0, x1, y0, y1, ...), one LDS.128 yields two packed operands, and each lane evaluates two list entries per
//       instruction for its target.  Partial sums per 32-entry batch are added to the running totals (accuracy).
// Forces: Plummer-softened p-p, and p-c with monopole + quadrupole (second-order expansion of the softened kernel,
// DESIGN.md O10): 35 packed fp32 operations + 2 MUFU.RSQ per PAIR of p-c interactions, 13 + 2 per pair of p-p.
#include <algorithm>
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
struct __align__(16) WarpShared {
    float pc[kRingPairs * kPcPair];
    float pp[kRingPairs * kPpPair];
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

// One slot: T = 2^K targets; this lane's target position and running sums (acceleration, MINUS the potential).
struct Slot { float tx, ty, tz, ax, ay, az, p; };

struct Consts { f2 e2, mhalf, m2p5; };

// p-c over `npairs` ring pairs starting at pair `hp`; lane takes pairs sub, sub + S, ...  (S = 32 >> K sub-lists).
//   -phi += M/rho + nTh/rho^3 - w/(2 rho^5),                 q = Qm dr = -3 Q dr,  w = dr.q
//   a    += dr (M/rho^3 + n3Th/rho^5 - 5 w/(2 rho^7)) + q/rho^5
template <int K>
__device__ __forceinline__ void eval_pc(const WarpShared* ws, int hp, int npairs, Slot& s, const Consts& k, int lane) {
    constexpr int S = 32 >> K;
    const f2 ntx = pk(-s.tx, -s.tx), nty = pk(-s.ty, -s.ty), ntz = pk(-s.tz, -s.tz);
    f2 ax = 0ull, ay = 0ull, az = 0ull, P = 0ull;
#pragma unroll 2
    for (int p = lane >> K; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ws->pc + ((hp + p) & (kRingPairs - 1)) * kPcPair);
        const ulonglong2 v0 = src[0], v1 = src[1], v2 = src[2], v3 = src[3], v4 = src[4], v5 = src[5];
        const f2 dx = add2(v0.x, ntx), dy = add2(v0.y, nty), dz = add2(v1.x, ntz);
        const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
        const f2 ri = rsqrt2(r2);
        const f2 ri2 = mul2(ri, ri), ri3 = mul2(ri, ri2), ri5 = mul2(ri3, ri2);
        const f2 qx = fma2(v2.x, dx, fma2(v3.y, dy, mul2(v4.x, dz)));
        const f2 qy = fma2(v3.y, dx, fma2(v2.y, dy, mul2(v4.y, dz)));
        const f2 qz = fma2(v4.x, dx, fma2(v4.y, dy, mul2(v3.x, dz)));
        const f2 w = fma2(dx, qx, fma2(dy, qy, mul2(dz, qz)));
        const f2 t = mul2(w, ri5);
        P = fma2(v1.y, ri, fma2(v5.x, ri3, fma2(t, k.mhalf, P)));
        const f2 br = fma2(mul2(t, ri2), k.m2p5, fma2(v5.y, ri5, mul2(v1.y, ri3)));
        ax = fma2(qx, ri5, fma2(dx, br, ax));
        ay = fma2(qy, ri5, fma2(dy, br, ay));
        az = fma2(qz, ri5, fma2(dz, br, az));
    }
    float lo, hi;
    upk(ax, lo, hi); s.ax += lo + hi;
    upk(ay, lo, hi); s.ay += lo + hi;
    upk(az, lo, hi); s.az += lo + hi;
    upk(P, lo, hi); s.p += lo + hi;
}

// p-p.  kSelf: the ring holds the group's own `nself` particles from entry 0; entry j is target index j: skip j == tidx
// and the massless pad entry j >= nself (it sits ON the last own particle: r = 0 would give 0 * inf when eps = 0).
template <int K, bool kSelf>
__device__ __forceinline__ void eval_pp(const WarpShared* ws, int hp, int npairs, Slot& s, const Consts& k, int lane, int tidx, int nself) {
    constexpr int S = 32 >> K;
    const f2 ntx = pk(-s.tx, -s.tx), nty = pk(-s.ty, -s.ty), ntz = pk(-s.tz, -s.tz);
    f2 ax = 0ull, ay = 0ull, az = 0ull, P = 0ull;
#pragma unroll 2
    for (int p = lane >> K; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ws->pp + ((hp + p) & (kRingPairs - 1)) * kPpPair);
        const ulonglong2 v0 = src[0], v1 = src[1];
        const f2 dx = add2(v0.x, ntx), dy = add2(v0.y, nty), dz = add2(v1.x, ntz);
        const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
        f2 ri;
        if (kSelf) {
            float lo, hi;
            upk(r2, lo, hi);
            lo = (2 * p == tidx) ? 0.0f : rsqrt_approx(lo);
            hi = (2 * p + 1 == tidx || 2 * p + 1 >= nself) ? 0.0f : rsqrt_approx(hi);
            ri = pk(lo, hi);
        } else {
            ri = rsqrt2(r2);
        }
        const f2 ri2 = mul2(ri, ri);
        const f2 mr = mul2(v1.y, ri);
        const f2 mr3 = mul2(mr, ri2);
        P = add2(P, mr);
        ax = fma2(dx, mr3, ax);
        ay = fma2(dy, mr3, ay);
        az = fma2(dz, mr3, az);
    }
    float lo, hi;
    upk(ax, lo, hi); s.ax += lo + hi;
    upk(ay, lo, hi); s.ay += lo + hi;
    upk(az, lo, hi); s.az += lo + hi;
    upk(P, lo, hi); s.p += lo + hi;
}

// The five slots of a group: A, B (32 targets each), C (16), D (8), E (4).
struct Slots {
    Slot a, b, c, d, e;
    bool hasA, hasB, hasC, hasD, hasE;
    int baseC, baseD, baseE;
};

__device__ __forceinline__ void eval_pc_all(const WarpShared* ws, int hp, int npairs, Slots& S, const Consts& k, int lane) {
    if (S.hasA) eval_pc<5>(ws, hp, npairs, S.a, k, lane);
    if (S.hasB) eval_pc<5>(ws, hp, npairs, S.b, k, lane);
    if (S.hasC) eval_pc<4>(ws, hp, npairs, S.c, k, lane);
    if (S.hasD) eval_pc<3>(ws, hp, npairs, S.d, k, lane);
    if (S.hasE) eval_pc<2>(ws, hp, npairs, S.e, k, lane);
}

template <bool kSelf>
__device__ __forceinline__ void eval_pp_all(const WarpShared* ws, int hp, int npairs, Slots& S, const Consts& k, int lane, int nself) {
    if (S.hasA) eval_pp<5, kSelf>(ws, hp, npairs, S.a, k, lane, lane, nself);
    if (S.hasB) eval_pp<5, kSelf>(ws, hp, npairs, S.b, k, lane, 32 + lane, nself);
    if (S.hasC) eval_pp<4, kSelf>(ws, hp, npairs, S.c, k, lane, S.baseC + (lane & 15), nself);
    if (S.hasD) eval_pp<3, kSelf>(ws, hp, npairs, S.d, k, lane, S.baseD + (lane & 7), nself);
    if (S.hasE) eval_pp<2, kSelf>(ws, hp, npairs, S.e, k, lane, S.baseE + (lane & 3), nself);
}

__device__ __forceinline__ void slot_init(Slot& s, const float4* __restrict__ pos, uint32_t gb, int ng, int tidx) {
    const float4 p = __ldg(pos + gb + min(tidx, ng - 1));   // idle target slots shadow the last particle (results discarded)
    s.tx = p.x; s.ty = p.y; s.tz = p.z;
    s.ax = s.ay = s.az = s.p = 0.0f;
}

// Add the sub-list sums of a slot (lanes that share l mod T) and store the T targets.
template <int K>
__device__ __forceinline__ void slot_finish(Slot& s, int lane, int tbase, int ng, uint32_t gb, float4* __restrict__ acc_out) {
#pragma unroll
    for (int o = 1 << K; o < 32; o <<= 1) {
        s.ax += __shfl_xor_sync(0xFFFFFFFFu, s.ax, o);
        s.ay += __shfl_xor_sync(0xFFFFFFFFu, s.ay, o);
        s.az += __shfl_xor_sync(0xFFFFFFFFu, s.az, o);
        s.p += __shfl_xor_sync(0xFFFFFFFFu, s.p, o);
    }
    const int idx = tbase + lane;
    if (lane < (1 << K) && idx < ng) acc_out[gb + idx] = make_float4(s.ax, s.ay, s.az, -s.p);
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
                                        const float4* __restrict__ pos, const float4* __restrict__ rec, float eps2,
                                        float4* __restrict__ acc_out, uint32_t* __restrict__ g_npc, uint32_t* __restrict__ g_npp,
                                        DevScalars* sc) {
    const uint32_t lt = (1u << lane) - 1u;
    const int ng = (int)(ge - gb);
    Consts k;
    k.e2 = pk(eps2, eps2);
    k.mhalf = pk(-0.5f, -0.5f);
    k.m2p5 = pk(-2.5f, -2.5f);

    // ---- the group's tight box (A13) and its own particles
    float4 own[2];
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        own[t] = __ldg(pos + gb + min(lane + 32 * t, ng - 1));
        mn[0] = fminf(mn[0], own[t].x); mx[0] = fmaxf(mx[0], own[t].x);
        mn[1] = fminf(mn[1], own[t].y); mx[1] = fmaxf(mx[1], own[t].y);
        mn[2] = fminf(mn[2], own[t].z); mx[2] = fmaxf(mx[2], own[t].z);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            mn[a] = fminf(mn[a], __shfl_xor_sync(0xFFFFFFFFu, mn[a], o));
            mx[a] = fmaxf(mx[a], __shfl_xor_sync(0xFFFFFFFFu, mx[a], o));
        }

    // ---- slots: n rounded up to a multiple of 4, split as 32 + 32 + 16 + 8 + 4
    Slots S;
    {
        const int m = (ng + 3) & ~3;
        const int full = m >> 5, rem = m & 31;
        S.hasA = full >= 1; S.hasB = full == 2;
        S.hasC = (rem & 16) != 0; S.hasD = (rem & 8) != 0; S.hasE = (rem & 4) != 0;
        int base = 32 * full;
        S.baseC = base; base += S.hasC ? 16 : 0;
        S.baseD = base; base += S.hasD ? 8 : 0;
        S.baseE = base;
        slot_init(S.a, pos, gb, ng, lane);
        slot_init(S.b, pos, gb, ng, 32 + lane);
        slot_init(S.c, pos, gb, ng, S.baseC + (lane & 15));
        slot_init(S.d, pos, gb, ng, S.baseD + (lane & 7));
        slot_init(S.e, pos, gb, ng, S.baseE + (lane & 3));
    }

    int sp = 1;
    if (lane == 0) ws->stack[0] = 0u;   // the root (A17)
    __syncwarp();
    int pc_head = 0, pc_cnt = 0, pp_head = 0, pp_cnt = 0;   // heads are even (entries are consumed 32 at a time)
    uint32_t npc = 0, npp = 0, nmac = 0;

    while (sp > 0) {
        int kpop = (kStackCap - kStackReserve - sp) / 7;
        kpop = max(1, min(kpop, 32));
        kpop = min(kpop, sp);
        const bool valid = lane < kpop;
        uint32_t cell = 0;
        if (valid) cell = ws->stack[sp - 1 - lane];
        sp -= kpop;
        nmac += (uint32_t)kpop;
        __syncwarp();
        bool accept = false, isleaf = false, isnode = false;
        float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0, r3 = r0;
        uint32_t first = 0, cnt = 0;
        if (valid) {
            const float4* rp = rec + 4 * (size_t)cell;     // the whole 64 B record in one round trip
            r0 = __ldg(rp); r1 = __ldg(rp + 1); r2 = __ldg(rp + 2); r3 = __ldg(rp + 3);
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
        // ---- accepted cells -> p-c ring
        const uint32_t amask = __ballot_sync(0xFFFFFFFFu, accept);
        if (amask) {
            if (accept) {
                const float T = (r1.y + r1.z) + r1.w;
                const int e = (pc_head + pc_cnt + __popc(amask & lt)) & (kRing - 1);
                pc_store(ws->pc, e, r0.x, r0.y, r0.z, r1.x, -3.0f * r1.y, -3.0f * r1.z, -3.0f * r1.w, -3.0f * r2.x, -3.0f * r2.y,
                         -3.0f * r2.z, -0.5f * T, -1.5f * T);
            }
            const int na = __popc(amask);
            pc_cnt += na;
            npc += (uint32_t)na;
            __syncwarp();
            if (pc_cnt >= 32) {
                eval_pc_all(ws, pc_head >> 1, 16, S, k, lane);
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
                if (keep) {
                    const float4 p = __ldg(pos + src);
                    pp_store(ws->pp, (pp_head + pp_cnt + __popc(kmask & lt)) & (kRing - 1), p.x, p.y, p.z, p.w);
                }
                pp_cnt += __popc(kmask);
                __syncwarp();
                if (pp_cnt >= 32) {
                    eval_pp_all<false>(ws, pp_head >> 1, 16, S, k, lane, 0);
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
    // ---- flush the rings (an odd tail gets a massless partner)
    if (pc_cnt > 0) {
        if ((pc_cnt & 1) && lane == 0) pc_pad(ws->pc, (pc_head + pc_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pc_all(ws, pc_head >> 1, (pc_cnt + 1) >> 1, S, k, lane);
    }
    if (pp_cnt > 0) {
        if ((pp_cnt & 1) && lane == 0) pp_pad(ws->pp, (pp_head + pp_cnt - 1) & (kRing - 1));
        __syncwarp();
        eval_pp_all<false>(ws, pp_head >> 1, (pp_cnt + 1) >> 1, S, k, lane, 0);
    }
    __syncwarp();
    // ---- self block: the group's own particles, entry j = target index j, j != i
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        if (idx < ng) pp_store(ws->pp, idx, own[t].x, own[t].y, own[t].z, own[t].w);
    }
    __syncwarp();
    if ((ng & 1) && lane == 0) pp_pad(ws->pp, ng - 1);
    __syncwarp();
    eval_pp_all<true>(ws, 0, (ng + 1) >> 1, S, k, lane, ng);
    __syncwarp();
    // ---- add the sub-list sums and store
    if (S.hasA) slot_finish<5>(S.a, lane, 0, ng, gb, acc_out);
    if (S.hasB) slot_finish<5>(S.b, lane, 32, ng, gb, acc_out);
    if (S.hasC) slot_finish<4>(S.c, lane, S.baseC, ng, gb, acc_out);
    if (S.hasD) slot_finish<3>(S.d, lane, S.baseD, ng, gb, acc_out);
    if (S.hasE) slot_finish<2>(S.e, lane, S.baseE, ng, gb, acc_out);
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
        walk_group(ws, lane, g, gb, ge, pos, rec, eps2, acc_out, g_npc, g_npp, sc);
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
