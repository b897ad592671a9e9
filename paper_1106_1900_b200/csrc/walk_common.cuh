// walk_common.cuh -- what the walk kernels share: packed-fp32 helpers, the group box, the MAC tests (Eq.1 and the
// minimum-distance variant), and the ring / slot force evaluation of the fused fallback kernel (walk.cu).  The
// list-driven evaluation kernel (walk_eval.cu) has its own, later layout: two targets per 64-bit register.
//
// Evaluation layout of the fused kernel (what differs from the paper's one-thread-per-particle sweep):
//   (1) Lane use.  A group holds n <= 64 targets (mean ~19), so "one target per lane" idles ~half of the warp.  The
//       paper's remedy is up to 4 threads per particle (L81, L97); here it is taken to its end: n is rounded up to a
//       multiple of 4 and split in binary, 64 | 32 + 16 + 8 + 4 -> "slots" of T = 2^K targets.  In a slot a lane serves
//       TWO targets, (l mod T/2) and (l mod T/2) + T/2, and sub-list (l div T/2): the 64 / T sub-lists interleave the ring
//       entries, and a butterfly of shuffles adds the sub-list sums at the end of the group (>= 93 % useful lanes).
//   (2) FP32 rate.  The packed f32x2 forms (FFMA2/FMUL2/FADD2) get nearer to the 128 lanes/clk/SM than scalar FFMA
//       (measured 71.8 vs 37-45 TFLOP/s; both are bounded by register-file bandwidth).  The rings therefore store PAIRS of entries interleaved
//       (x0, x1, y0, y1, ...), one LDS.128 yields two packed operands, and each lane evaluates two list entries per
//       instruction for each of its targets.
//   (3) Shared-memory delivery.  An LDS.128 moves 512 B into the register file whether or not the lanes share the address,
//       i.e. 4 cycles of the 128 B/clk path: six loads per entry pair for ONE target per lane make the loop smem-bound at
//       ~73 % of the FMA rate (measured 50 TFLOP/s).  Two targets per loaded pair halve that traffic (measured 60 TFLOP/s).
//   Running sums per slot live in shared memory between sweeps (partial sums of a sweep are formed in registers and added
//   once: accuracy, and the kernels stay inside 128 registers at 16 warps/SM).
// Forces: Plummer-softened p-p, and p-c with monopole + quadrupole (second-order expansion of the softened kernel,
// DESIGN.md O10): 33 packed fp32 operations + 2 MUFU.RSQ per PAIR of p-c interactions, 13 + 2 per pair of p-p.
#pragma once
#include "bh_internal.cuh"

namespace bh {

constexpr int kPcPair = 28;          // floats per p-c pair: 12 fields x 2 + 4 pad (112 B stride: no bank conflict for 8 pairs)
constexpr int kPpPair = 8;           // floats per p-p pair: x0 x1 y0 y1 z0 z1 m0 m1
constexpr int kMaxSlots = 4;         // 32 + 16 + 8 + 4 (or the single 64-target slot)

// p-c pair fields f = 0..11: x y z M | Qm_xx Qm_yy Qm_zz Qm_xy | Qm_xz Qm_yz nTh n3Th, with Qm = -3 Q, nTh = -T/2,
// n3Th = -3T/2; the two entries of a pair sit at float index pair * kPcPair + 2 f + half.
typedef float4 SlotTotals[2][32];    // running sums of one slot: [target-of-lane][lane] = (ax, ay, az, -phi)

typedef unsigned long long f2;   // two fp32 values in one 64-bit register: low word = first entry, high word = second entry

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
__device__ __forceinline__ Consts make_consts(float eps2) {
    Consts k;
    k.e2 = pk(eps2, eps2);
    k.mhalf = pk(-0.5f, -0.5f);
    k.m2p5 = pk(-2.5f, -2.5f);
    return k;
}

struct Acc2 { f2 ax, ay, az, p; };

// ---- the force bodies of the list evaluation (walk_eval.cu; also timed on their own by probe.cu)
__device__ __forceinline__ f2 bc(float s) { return pk(s, s); }   // ptxas folds this into the broadcast operand form

// One p-c entry on one packed pair of targets.  Record: v0 = (com, M), v1 = (Qm_xx, Qm_yy, Qm_zz, Qm_xy),
// v2 = (Qm_xz, Qm_yz, nTh, n3Th) with Qm = -3 Q, nTh = -T/2, n3Th = -3T/2.  rho^2 = |dr|^2 + eps^2, u = 1/rho^2,
// q = Qm dr, w = dr.q:   -phi += (1/rho) (M + u (nTh - w u / 2)),   a += (1/rho^5) (q + dr (M rho^2 + n3Th - 5 w u / 2)).
__device__ __forceinline__ void pc_bc(const float4& v0, const float4& v1, const float4& v2, f2 ntx, f2 nty, f2 ntz, const Consts& k, Acc2& a) {
    const f2 dx = add2(bc(v0.x), ntx), dy = add2(bc(v0.y), nty), dz = add2(bc(v0.z), ntz);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
    const f2 ri = rsqrt2(r2);
    const f2 u = mul2(ri, ri), uu = mul2(u, u), ri5 = mul2(ri, uu);
    const f2 qx = fma2(bc(v1.x), dx, fma2(bc(v1.w), dy, mul2(bc(v2.x), dz)));
    const f2 qy = fma2(bc(v1.w), dx, fma2(bc(v1.y), dy, mul2(bc(v2.y), dz)));
    const f2 qz = fma2(bc(v2.x), dx, fma2(bc(v2.y), dy, mul2(bc(v1.z), dz)));
    const f2 w = fma2(dx, qx, fma2(dy, qy, mul2(dz, qz)));
    const f2 wu = mul2(w, u);
    a.p = fma2(ri, fma2(u, fma2(wu, k.mhalf, bc(v2.z)), bc(v0.w)), a.p);
    const f2 c = fma2(bc(v0.w), r2, fma2(wu, k.m2p5, bc(v2.w)));
    a.ax = fma2(fma2(dx, c, qx), ri5, a.ax);
    a.ay = fma2(fma2(dy, c, qy), ri5, a.ay);
    a.az = fma2(fma2(dz, c, qz), ri5, a.az);
}

// One p-p entry on one packed pair of targets tA, tA + 1.  kSelf: the entry is particle `e` of the group itself: skip
// e == target (A19) and the shadow targets >= ng (they sit ON a real particle: r = 0 would give 0 * inf when eps = 0).
template <bool kSelf>
__device__ __forceinline__ void pp_bc(const float4& v, f2 ntx, f2 nty, f2 ntz, const Consts& k, Acc2& a, int e, int tA, int ng) {
    const f2 dx = add2(bc(v.x), ntx), dy = add2(bc(v.y), nty), dz = add2(bc(v.z), ntz);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
    f2 ri;
    if (kSelf) {
        float lo, hi;
        upk(r2, lo, hi);
        lo = (e == tA || tA >= ng) ? 0.0f : rsqrt_approx(lo);
        hi = (e == tA + 1 || tA + 1 >= ng) ? 0.0f : rsqrt_approx(hi);
        ri = pk(lo, hi);
    } else {
        ri = rsqrt2(r2);
    }
    const f2 ri2 = mul2(ri, ri);
    const f2 mr = mul2(bc(v.w), ri);
    const f2 mr3 = mul2(mr, ri2);
    a.p = add2(a.p, mr);
    a.ax = fma2(dx, mr3, a.ax);
    a.ay = fma2(dy, mr3, a.ay);
    a.az = fma2(dz, mr3, a.az);
}



// One pair of p-c entries on one target.  With rho^2 = |dr|^2 + eps^2, u = 1/rho^2, q = Qm dr = -3 Q dr, w = dr.q:
//   -phi += (1/rho)   (M + u (nTh - w u / 2))
//   a    += (1/rho^5) (q + dr (M rho^2 + n3Th - 5 w u / 2))
// which is O10's  -phi = M/rho - T/(2 rho^3) + 3 (dr Q dr)/(2 rho^5),  a = dr (M/rho^3 - 3T/(2 rho^5) + 15 (dr Q dr)/(2 rho^7)) - 3 Q dr/rho^5.
__device__ __forceinline__ void pc_one(const ulonglong2& v0, const ulonglong2& v1, const ulonglong2& v2, const ulonglong2& v3,
                                       const ulonglong2& v4, const ulonglong2& v5, f2 ntx, f2 nty, f2 ntz, const Consts& k, Acc2& a) {
    const f2 dx = add2(v0.x, ntx), dy = add2(v0.y, nty), dz = add2(v1.x, ntz);
    const f2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, k.e2)));
    const f2 ri = rsqrt2(r2);
    const f2 u = mul2(ri, ri), uu = mul2(u, u), ri5 = mul2(ri, uu);
    const f2 qx = fma2(v2.x, dx, fma2(v3.y, dy, mul2(v4.x, dz)));
    const f2 qy = fma2(v3.y, dx, fma2(v2.y, dy, mul2(v4.y, dz)));
    const f2 qz = fma2(v4.x, dx, fma2(v4.y, dy, mul2(v3.x, dz)));
    const f2 w = fma2(dx, qx, fma2(dy, qy, mul2(dz, qz)));
    const f2 wu = mul2(w, u);
    a.p = fma2(ri, fma2(u, fma2(wu, k.mhalf, v5.x), v1.y), a.p);
    const f2 c = fma2(v1.y, r2, fma2(wu, k.m2p5, v5.y));
    a.ax = fma2(fma2(dx, c, qx), ri5, a.ax);
    a.ay = fma2(fma2(dy, c, qy), ri5, a.ay);
    a.az = fma2(fma2(dz, c, qz), ri5, a.az);
}

// Running sums <-> packed accumulators: a sweep starts from (total, 0) and stores low + high, so the only extra
// arithmetic per slot and sweep is one add per component.
__device__ __forceinline__ Acc2 acc_load(const float4* tot) {
    const float4 t = *tot;
    Acc2 a;
    a.ax = pk(t.x, 0.f); a.ay = pk(t.y, 0.f); a.az = pk(t.z, 0.f); a.p = pk(t.w, 0.f);
    return a;
}
__device__ __forceinline__ void acc_store(float4* tot, const Acc2& a) {
    float4 t;
    float lo, hi;
    upk(a.ax, lo, hi); t.x = lo + hi;
    upk(a.ay, lo, hi); t.y = lo + hi;
    upk(a.az, lo, hi); t.z = lo + hi;
    upk(a.p, lo, hi); t.w = lo + hi;
    *tot = t;
}

// p-c sweep of one slot over `npairs` ring pairs starting at pair `hp` of a ring of `kPairs` pairs (power of two; the
// ring never wraps when kWrap is false).  Lane: targets t0, t1; pairs sub, sub + S, ...  kUnroll2: two pairs per
// iteration (four independent interaction chains per lane hide the rsqrt and FMA latencies with few resident warps).
template <int kPairs, bool kWrap, bool kUnroll2>
__device__ __forceinline__ void eval_pc_slot(const float* ring, const float4* own, SlotTotals* tot, int hp, int npairs, int K, int tbase,
                                             int slot, int ng, const Consts& k, int lane) {
    const int L = 1 << (K - 1), sub = lane >> (K - 1), S = 32 >> (K - 1);
    const int t0 = tbase + (lane & (L - 1)), t1 = t0 + L;
    const float4 T0 = own[min(t0, ng - 1)], T1 = own[min(t1, ng - 1)];   // idle targets shadow the last particle
    const f2 ntx0 = pk(-T0.x, -T0.x), nty0 = pk(-T0.y, -T0.y), ntz0 = pk(-T0.z, -T0.z);
    const f2 ntx1 = pk(-T1.x, -T1.x), nty1 = pk(-T1.y, -T1.y), ntz1 = pk(-T1.z, -T1.z);
    Acc2 a0 = acc_load(&tot[slot][0][lane]), a1 = acc_load(&tot[slot][1][lane]);
    int p = sub;
    if (kUnroll2) {
        for (; p + S < npairs; p += 2 * S) {
            const ulonglong2* sa = reinterpret_cast<const ulonglong2*>(ring + (kWrap ? ((hp + p) & (kPairs - 1)) : (hp + p)) * kPcPair);
            const ulonglong2* sb = reinterpret_cast<const ulonglong2*>(ring + (kWrap ? ((hp + p + S) & (kPairs - 1)) : (hp + p + S)) * kPcPair);
            const ulonglong2 v0 = sa[0], v1 = sa[1], v2 = sa[2], v3 = sa[3], v4 = sa[4], v5 = sa[5];
            const ulonglong2 w0 = sb[0], w1 = sb[1], w2 = sb[2], w3 = sb[3], w4 = sb[4], w5 = sb[5];
            pc_one(v0, v1, v2, v3, v4, v5, ntx0, nty0, ntz0, k, a0);
            pc_one(v0, v1, v2, v3, v4, v5, ntx1, nty1, ntz1, k, a1);
            pc_one(w0, w1, w2, w3, w4, w5, ntx0, nty0, ntz0, k, a0);
            pc_one(w0, w1, w2, w3, w4, w5, ntx1, nty1, ntz1, k, a1);
        }
    }
    for (; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ring + (kWrap ? ((hp + p) & (kPairs - 1)) : (hp + p)) * kPcPair);
        const ulonglong2 v0 = src[0], v1 = src[1], v2 = src[2], v3 = src[3], v4 = src[4], v5 = src[5];
        pc_one(v0, v1, v2, v3, v4, v5, ntx0, nty0, ntz0, k, a0);
        pc_one(v0, v1, v2, v3, v4, v5, ntx1, nty1, ntz1, k, a1);
    }
    acc_store(&tot[slot][0][lane], a0);
    acc_store(&tot[slot][1][lane], a1);
}

// p-p, one pair of entries on one target.  kSelf: the ring holds the group's own `ng` particles from entry 0 and entry j is
// target index j: skip j == t and the massless pad entry j >= ng (it sits ON the last own particle: r = 0 would give
// 0 * inf when eps = 0).
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

template <bool kSelf, int kPairs, bool kWrap>
__device__ __forceinline__ void eval_pp_slot(const float* ring, const float4* own, SlotTotals* tot, int hp, int npairs, int K, int tbase,
                                             int slot, int ng, const Consts& k, int lane) {
    const int L = 1 << (K - 1), sub = lane >> (K - 1), S = 32 >> (K - 1);
    const int t0 = tbase + (lane & (L - 1)), t1 = t0 + L;
    const float4 T0 = own[min(t0, ng - 1)], T1 = own[min(t1, ng - 1)];
    const f2 ntx0 = pk(-T0.x, -T0.x), nty0 = pk(-T0.y, -T0.y), ntz0 = pk(-T0.z, -T0.z);
    const f2 ntx1 = pk(-T1.x, -T1.x), nty1 = pk(-T1.y, -T1.y), ntz1 = pk(-T1.z, -T1.z);
    Acc2 a0 = acc_load(&tot[slot][0][lane]), a1 = acc_load(&tot[slot][1][lane]);
    for (int p = sub; p < npairs; p += S) {
        const ulonglong2* src = reinterpret_cast<const ulonglong2*>(ring + (kWrap ? ((hp + p) & (kPairs - 1)) : (hp + p)) * kPpPair);
        const ulonglong2 v0 = src[0], v1 = src[1];
        pp_one<kSelf>(v0, v1, ntx0, nty0, ntz0, k, a0, 2 * p, t0, ng);
        pp_one<kSelf>(v0, v1, ntx1, nty1, ntz1, k, a1, 2 * p, t1, ng);
    }
    acc_store(&tot[slot][0][lane], a0);
    acc_store(&tot[slot][1][lane], a1);
}

// The slots of a group are the set bits K = 6 (alone) or 5..2 of m = roundup4(n): a slot of 2^K targets each.  They are
// enumerated on the fly (slot index = rank of the bit from the top, first target = sum of the higher bits).
template <int kPairs, bool kWrap, bool kUnroll2>
__device__ __forceinline__ void eval_pc_all(const float* ring, const float4* own, SlotTotals* tot, int hp, int npairs, int m, int ng,
                                            const Consts& k, int lane) {
    int slot = 0, base = 0;
#pragma unroll
    for (int K = 6; K >= 2; --K)
        if (m & (1 << K)) { eval_pc_slot<kPairs, kWrap, kUnroll2>(ring, own, tot, hp, npairs, K, base, slot, ng, k, lane); ++slot; base += 1 << K; }
}
template <bool kSelf, int kPairs, bool kWrap>
__device__ __forceinline__ void eval_pp_all(const float* ring, const float4* own, SlotTotals* tot, int hp, int npairs, int m, int ng,
                                            const Consts& k, int lane) {
    int slot = 0, base = 0;
#pragma unroll
    for (int K = 6; K >= 2; --K)
        if (m & (1 << K)) { eval_pp_slot<kSelf, kPairs, kWrap>(ring, own, tot, hp, npairs, K, base, slot, ng, k, lane); ++slot; base += 1 << K; }
}

__device__ __forceinline__ void totals_clear(SlotTotals* tot, int lane) {
#pragma unroll
    for (int i = 0; i < kMaxSlots; ++i) {
        tot[i][0][lane] = make_float4(0.f, 0.f, 0.f, 0.f);
        tot[i][1][lane] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
}

// Add the sub-list sums of every slot (lanes that share l mod T/2) and store the group's accelerations + potentials.
__device__ __forceinline__ void totals_finish(SlotTotals* tot, int m, int lane, int ng, uint32_t gb, float4* __restrict__ acc_out) {
    int slot = 0, base = 0;
#pragma unroll
    for (int K = 6; K >= 2; --K) {
        if (!(m & (1 << K))) continue;
        const int L = 1 << (K - 1);
#pragma unroll
        for (int r = 0; r < 2; ++r) {
            float4 t = tot[slot][r][lane];
            for (int o = L; o < 32; o <<= 1) {
                t.x += __shfl_xor_sync(0xFFFFFFFFu, t.x, o);
                t.y += __shfl_xor_sync(0xFFFFFFFFu, t.y, o);
                t.z += __shfl_xor_sync(0xFFFFFFFFu, t.z, o);
                t.w += __shfl_xor_sync(0xFFFFFFFFu, t.w, o);
            }
            const int idx = base + r * L + lane;
            if (lane < L && idx < ng) acc_out[gb + idx] = make_float4(t.x, t.y, t.z, -t.w);
        }
        ++slot;
        base += 1 << K;
    }
}

// Scalar stores of one entry into a pair-interleaved ring: entry e lives in pair e >> 1, half e & 1.
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

// Group box (A13): exact per-axis min / max of the group's particles, which are also copied to `own`.
__device__ __forceinline__ void group_box(const float4* __restrict__ pos, uint32_t gb, int ng, int lane, float4* own, float mn[3], float mx[3]) {
    mn[0] = mn[1] = mn[2] = INFINITY;
    mx[0] = mx[1] = mx[2] = -INFINITY;
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int idx = lane + 32 * t;
        const float4 p = __ldg(pos + gb + min(idx, ng - 1));
        if (own && idx < ng) own[idx] = p;
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
}

// Eq.1 in exactly the fp32 operations of DESIGN.md O9: accept iff d^2 > r2open.
__device__ __forceinline__ bool mac_accept(const float mn[3], const float mx[3], const float4& com_r2) {
    const float dx = fmaxf(fmaxf(__fsub_rn(mn[0], com_r2.x), __fsub_rn(com_r2.x, mx[0])), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(mn[1], com_r2.y), __fsub_rn(com_r2.y, mx[1])), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(mn[2], com_r2.z), __fsub_rn(com_r2.z, mx[2])), 0.0f);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    return d2 > com_r2.w;
}

// The minimum-distance MAC the paper also implemented ([31]; reading A28): the distance is taken
// between the group's box and the cell's tight BOX, and compared with l / theta: accept iff d^2 > r2open, with
// d_k = max(max(gmin_k - cmax_k, cmin_k - gmax_k), 0) in the same single fp32 operations as Eq.1's test.
constexpr int kMacEq1 = 0, kMacMinDist = 1;
struct CellBox { float2 a, b, c; };        // (min x, min y) (min z, max x) (max y, max z): the row of `box` as three 8-byte loads
__device__ __forceinline__ CellBox load_cell_box(const float* __restrict__ box, uint32_t cell) {
    const float2* p = reinterpret_cast<const float2*>(box + 6 * (size_t)cell);
    CellBox r;
    r.a = __ldg(p); r.b = __ldg(p + 1); r.c = __ldg(p + 2);
    return r;
}
__device__ __forceinline__ bool mac_accept_box(const float mn[3], const float mx[3], const CellBox& cb, float r2open) {
    const float dx = fmaxf(fmaxf(__fsub_rn(mn[0], cb.b.y), __fsub_rn(cb.a.x, mx[0])), 0.0f);
    const float dy = fmaxf(fmaxf(__fsub_rn(mn[1], cb.c.x), __fsub_rn(cb.a.y, mx[1])), 0.0f);
    const float dz = fmaxf(fmaxf(__fsub_rn(mn[2], cb.c.y), __fsub_rn(cb.b.x, mx[2])), 0.0f);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    return d2 > r2open;
}

}  // namespace bh
