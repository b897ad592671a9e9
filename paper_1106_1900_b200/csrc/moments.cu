// moments.cu -- S6: monopole + quadrupole moments and tight boxes, bottom-up, in binary64 with a fixed operation
// order ("performed in double precision ... converted back to single precision"; Fig.4), and the
// fp32 walk / evaluation records with the opening radius of Eq.1.
// Every fp64 operation is an explicit round-to-nearest intrinsic so that no multiply-add is ever fused: the fp32
// roundings of these values feed the MAC, and a one-ulp difference would flip an opening decision somewhere.
//
// The paper goes level by level, one launch per level (~20 dependent launches, nearly all tiny).  Here ONE launch:
//   * a block owns a contiguous range of P particles and with it every cell that lies entirely inside the range.  It
//     computes its leaves (one thread each, particles in ascending order) and then its nodes level by level from the
//     deepest one, separated by __syncthreads only: a node's children lie inside the same range.  A node is computed by
//     EIGHT LANES, one child each: the lanes load their child at once, and the sums run over the children in ascending
//     order through shuffles -- the same sequence of roundings as a sequential loop (bit-identical);
//   * the cells that straddle a range boundary (at most one per level and block) are left to k_moments_span, a second
//     launch of ONE cluster of eight blocks, which computes them level by level in the same way: their children are
//     either owned cells (all published by the first launch: read from L2) or straddling cells of the level below, which
//     the cluster keeps in (distributed) shared memory -- the dependent chain over the levels of the tree never leaves it.
// No thread ever waits for another block of k_moments.  Cells of the same level are numbered in ascending first particle, so the
// owned cells of a block are one index range per level, read off the per-tile scans of tree.cu.
// The fp32 records (what the walk tests and what the force loop consumes) are written in the same pass when the caller
// knows theta (bh_leapfrog_step, or the theta of the last bh_compute_forces as a hint); k_cell_record writes them alone
// when theta changes on an existing tree.
#include <algorithm>
#include <cstdio>
#include <cooperative_groups.h>
#include "bh_internal.cuh"

namespace cg = cooperative_groups;


namespace bh {

struct Mom {
    double M, com[3], Q[6];
    float bmin[3], bmax[3];
};

struct RecOut {
    float4* trec;
    uint2* tlink;
    float4* erec;
    float theta;
    int mac_kind;
    int enabled;
};

// fp32 records of one cell: trec = (com, r2open), tlink = (first child | first particle, count | leaf << 31),
// erec (48 B) = (com, M) (Qm_xx, Qm_yy, Qm_zz, Qm_xy) (Qm_xz, Qm_yz, -T/2, -3T/2), Qm = -3 Q, T = trace Q;
// Eq.1: l = longest side of the tight box (A14), delta = |com - box centre|, r2open = (l / theta + delta)^2; the
// minimum-distance MAC (A28): r2open = (l / theta)^2.  All in single fp32 operations (O8).
struct Rec { float4 t; uint2 link; float4 e0, e1, e2; };
__device__ __forceinline__ Rec make_record(const Mom& m, float theta, int mac_kind, uint32_t pb, uint32_t pe, uint32_t cb, uint32_t ce) {
    Rec r;
    const float M = (float)m.M;
    const float cx = (float)m.com[0], cy = (float)m.com[1], cz = (float)m.com[2];
    float l = fmaxf(fmaxf(__fsub_rn(m.bmax[0], m.bmin[0]), __fsub_rn(m.bmax[1], m.bmin[1])), __fsub_rn(m.bmax[2], m.bmin[2]));
    l = fmaxf(l, 0.0f);
    const float ux = __fsub_rn(cx, __fmul_rn(0.5f, __fadd_rn(m.bmin[0], m.bmax[0])));
    const float uy = __fsub_rn(cy, __fmul_rn(0.5f, __fadd_rn(m.bmin[1], m.bmax[1])));
    const float uz = __fsub_rn(cz, __fmul_rn(0.5f, __fadd_rn(m.bmin[2], m.bmax[2])));
    const float s2 = __fadd_rn(__fadd_rn(__fmul_rn(ux, ux), __fmul_rn(uy, uy)), __fmul_rn(uz, uz));
    const float delta = __fsqrt_rn(s2);
    const float ropen = mac_kind == 1 ? __fdiv_rn(l, theta) : __fadd_rn(__fdiv_rn(l, theta), delta);   // A28 / Eq.1
    const float r2open = __fmul_rn(ropen, ropen);
    const bool leaf = (ce == cb);
    r.link.x = leaf ? pb : cb;
    r.link.y = leaf ? ((pe - pb) | 0x80000000u) : (ce - cb);
    const float qxx = (float)m.Q[0], qyy = (float)m.Q[1], qzz = (float)m.Q[2], qxy = (float)m.Q[3], qxz = (float)m.Q[4], qyz = (float)m.Q[5];
    const float T = __fadd_rn(__fadd_rn(qxx, qyy), qzz);
    r.t = make_float4(cx, cy, cz, r2open);
    r.e0 = make_float4(cx, cy, cz, M);
    r.e1 = make_float4(__fmul_rn(-3.0f, qxx), __fmul_rn(-3.0f, qyy), __fmul_rn(-3.0f, qzz), __fmul_rn(-3.0f, qxy));
    r.e2 = make_float4(__fmul_rn(-3.0f, qxz), __fmul_rn(-3.0f, qyz), __fmul_rn(-0.5f, T), __fmul_rn(-1.5f, T));
    return r;
}

__device__ __forceinline__ void mom_store(const Mom& m, double* mom64, float* box, uint32_t c) {
    double2* o = reinterpret_cast<double2*>(mom64 + 10 * (size_t)c);
    o[0] = make_double2(m.M, m.com[0]);
    o[1] = make_double2(m.com[1], m.com[2]);
    o[2] = make_double2(m.Q[0], m.Q[1]);
    o[3] = make_double2(m.Q[2], m.Q[3]);
    o[4] = make_double2(m.Q[4], m.Q[5]);
    float2* b = reinterpret_cast<float2*>(box + 6 * (size_t)c);
    b[0] = make_float2(m.bmin[0], m.bmin[1]);
    b[1] = make_float2(m.bmin[2], m.bmax[0]);
    b[2] = make_float2(m.bmax[1], m.bmax[2]);
}

__device__ __forceinline__ void rec_store(const Rec& r, const RecOut& o, uint32_t c) {
    o.trec[c] = r.t;
    o.tlink[c] = r.link;
    o.erec[3 * (size_t)c] = r.e0;
    o.erec[3 * (size_t)c + 1] = r.e1;
    o.erec[3 * (size_t)c + 2] = r.e2;
}

// Leaf: M = sum m; S = sum m x; com = S / M; Q_jk = sum (m r_j) r_k, r = x - com; particles in ascending order.
// `ld(i)` returns particle i (from the block's shared-memory copy where it has one).
template <typename Loader>
__device__ __forceinline__ void leaf_moments(Mom& m, Loader ld, uint32_t b, uint32_t e) {
    double S[3] = {0.0, 0.0, 0.0};
    m.M = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) { m.bmin[k] = INFINITY; m.bmax[k] = -INFINITY; }
#pragma unroll
    for (int k = 0; k < 6; ++k) m.Q[k] = 0.0;
    for (uint32_t i0 = b; i0 < e; i0 += 4) {                  // four loads in flight; the sums stay in ascending particle order
        float4 q[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) q[u] = ld(min(i0 + u, e - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (i0 + u >= e) break;
            const float4 p = q[u];
            const double w = (double)p.w;
            m.M = __dadd_rn(m.M, w);
            S[0] = __dadd_rn(S[0], __dmul_rn(w, (double)p.x));
            S[1] = __dadd_rn(S[1], __dmul_rn(w, (double)p.y));
            S[2] = __dadd_rn(S[2], __dmul_rn(w, (double)p.z));
            m.bmin[0] = fminf(m.bmin[0], p.x); m.bmax[0] = fmaxf(m.bmax[0], p.x);
            m.bmin[1] = fminf(m.bmin[1], p.y); m.bmax[1] = fmaxf(m.bmax[1], p.y);
            m.bmin[2] = fminf(m.bmin[2], p.z); m.bmax[2] = fmaxf(m.bmax[2], p.z);
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) m.com[k] = __ddiv_rn(S[k], m.M);
    for (uint32_t i = b; i < e; ++i) {
        const float4 p = ld(i);
        const double w = (double)p.w;
        const double rx = __dsub_rn((double)p.x, m.com[0]);
        const double ry = __dsub_rn((double)p.y, m.com[1]);
        const double rz = __dsub_rn((double)p.z, m.com[2]);
        const double tx = __dmul_rn(w, rx), ty = __dmul_rn(w, ry), tz = __dmul_rn(w, rz);
        m.Q[0] = __dadd_rn(m.Q[0], __dmul_rn(tx, rx));
        m.Q[1] = __dadd_rn(m.Q[1], __dmul_rn(ty, ry));
        m.Q[2] = __dadd_rn(m.Q[2], __dmul_rn(tz, rz));
        m.Q[3] = __dadd_rn(m.Q[3], __dmul_rn(tx, ry));
        m.Q[4] = __dadd_rn(m.Q[4], __dmul_rn(tx, rz));
        m.Q[5] = __dadd_rn(m.Q[5], __dmul_rn(ty, rz));
    }
}


// What a parent reads of a child.
struct Child {
    double M, c[3], Q[6];
    float bn[3], bx[3];
};
__device__ __forceinline__ void child_clear(Child& ch) {
    ch.M = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) { ch.c[k] = 0.0; ch.bn[k] = INFINITY; ch.bx[k] = -INFINITY; }
#pragma unroll
    for (int k = 0; k < 6; ++k) ch.Q[k] = 0.0;
}
// from the cell arrays, written earlier in this launch or the one before (possibly by another block): read from L2 (ld.global.cg)
__device__ __forceinline__ void child_load_global(Child& ch, const double* mom64, const float* box, uint32_t c) {
    const double2* mc = reinterpret_cast<const double2*>(mom64 + 10 * (size_t)c);
    const float2* bc = reinterpret_cast<const float2*>(box + 6 * (size_t)c);
    const double2 a0 = __ldcg(mc), a1 = __ldcg(mc + 1), a2 = __ldcg(mc + 2), a3 = __ldcg(mc + 3), a4 = __ldcg(mc + 4);
    const float2 b0 = __ldcg(bc), b1 = __ldcg(bc + 1), b2 = __ldcg(bc + 2);
    ch.M = a0.x; ch.c[0] = a0.y; ch.c[1] = a1.x; ch.c[2] = a1.y;
    ch.Q[0] = a2.x; ch.Q[1] = a2.y; ch.Q[2] = a3.x; ch.Q[3] = a3.y; ch.Q[4] = a4.x; ch.Q[5] = a4.y;
    ch.bn[0] = b0.x; ch.bn[1] = b0.y; ch.bn[2] = b1.x; ch.bx[0] = b1.y; ch.bx[1] = b2.x; ch.bx[2] = b2.y;
}
// the shared-memory copy of a straddling node (k_moments_span): 10 doubles, 6 floats
struct __align__(16) SpanCell { double m[10]; float b[6]; float pad[2]; };
__device__ __forceinline__ void child_load_shared(Child& ch, const SpanCell& sc) {
    ch.M = sc.m[0]; ch.c[0] = sc.m[1]; ch.c[1] = sc.m[2]; ch.c[2] = sc.m[3];
#pragma unroll
    for (int k = 0; k < 6; ++k) ch.Q[k] = sc.m[4 + k];
#pragma unroll
    for (int k = 0; k < 3; ++k) { ch.bn[k] = sc.b[k]; ch.bx[k] = sc.b[3 + k]; }
}

// Scratch of one lane group (eight lanes = one node): the children's terms, transposed through shared memory so that lane q
// sums quantity q over the children in ascending order.
struct NodeScratch { double a[8][4]; double q[8][6]; double p[8][6]; };     // (M, M cx, M cy, M cz), Q_c, (M d_j) d_k

// Node: M = sum M_c; S = sum M_c com_c; com = S / M; Q_jk = sum_c ((Q + Q_c,jk) + (M_c d_j) d_k), d = com_c - com; children
// in ascending order -- the same sequence of roundings as a sequential loop over the children.  Eight consecutive lanes
// (sub = 0..7) hold one child each in `ch` (cleared where sub >= nch; nch = 0: the lane group has no node).  Products are
// formed by the child's lane (one rounding each); the sums run in lane q < 4 (M, S) and lane q < 6 (Q) over scratch rows
// 0..nch-1.  On return every lane holds the whole result in `m`.
__device__ __forceinline__ void node_moments8(Mom& m, const Child& ch, int nch, int sub, NodeScratch& sx) {
    float bn[3], bx[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) { bn[k] = ch.bn[k]; bx[k] = ch.bx[k]; }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1)          // box: min / max are exact in any order
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bn[k] = fminf(bn[k], __shfl_xor_sync(0xFFFFFFFFu, bn[k], o, 8));
            bx[k] = fmaxf(bx[k], __shfl_xor_sync(0xFFFFFFFFu, bx[k], o, 8));
        }
#pragma unroll
    for (int k = 0; k < 3; ++k) { m.bmin[k] = bn[k]; m.bmax[k] = bx[k]; }
    sx.a[sub][0] = ch.M;
    sx.a[sub][1] = __dmul_rn(ch.M, ch.c[0]);
    sx.a[sub][2] = __dmul_rn(ch.M, ch.c[1]);
    sx.a[sub][3] = __dmul_rn(ch.M, ch.c[2]);
#pragma unroll
    for (int k = 0; k < 6; ++k) sx.q[sub][k] = ch.Q[k];
    __syncwarp();
    double acc = 0.0;
    if (sub < 4)
        for (int k = 0; k < nch; ++k) acc = __dadd_rn(acc, sx.a[k][sub]);
    const double M = __shfl_sync(0xFFFFFFFFu, acc, 0, 8);
    double com = 0.0;
    if (sub >= 1 && sub < 4 && nch > 0) com = __ddiv_rn(acc, M);
    m.M = M;
    m.com[0] = __shfl_sync(0xFFFFFFFFu, com, 1, 8);
    m.com[1] = __shfl_sync(0xFFFFFFFFu, com, 2, 8);
    m.com[2] = __shfl_sync(0xFFFFFFFFu, com, 3, 8);
    const double dx = __dsub_rn(ch.c[0], m.com[0]), dy = __dsub_rn(ch.c[1], m.com[1]), dz = __dsub_rn(ch.c[2], m.com[2]);
    const double tx = __dmul_rn(ch.M, dx), ty = __dmul_rn(ch.M, dy), tz = __dmul_rn(ch.M, dz);
    sx.p[sub][0] = __dmul_rn(tx, dx); sx.p[sub][1] = __dmul_rn(ty, dy); sx.p[sub][2] = __dmul_rn(tz, dz);
    sx.p[sub][3] = __dmul_rn(tx, dy); sx.p[sub][4] = __dmul_rn(tx, dz); sx.p[sub][5] = __dmul_rn(ty, dz);
    __syncwarp();
    double Q = 0.0;
    if (sub < 6)
        for (int k = 0; k < nch; ++k) Q = __dadd_rn(__dadd_rn(Q, sx.q[k][sub]), sx.p[k][sub]);
#pragma unroll
    for (int k = 0; k < 6; ++k) m.Q[k] = __shfl_sync(0xFFFFFFFFu, Q, k, 8);
    __syncwarp();                            // the scratch may be rewritten
}

constexpr int kMomThreads = 1024;
constexpr int kMomGroups = kMomThreads / 8;      // nodes in flight per block step
constexpr int kMomStage = 8192;                  // particles a block can stage in the shared memory of its node scratch
constexpr int kMomMaxBlocks = kMomBlockCap;      // straddling nodes per level (at most one per block)
constexpr int kSpanCtas = 8;                     // CTAs of the cluster that computes the straddling nodes
constexpr int kSpanThreads = 256;
constexpr int kSpanGroups = kSpanThreads / 8;
constexpr int kSpanSlots = (kMomMaxBlocks + kSpanCtas - 1) / kSpanCtas;

struct SpanShared {
    NodeScratch sx[kSpanGroups];
    SpanCell cell[2][kSpanSlots];                // this CTA's straddling nodes of the level being computed / the level below
    uint32_t list[kLevels][kMomMaxBlocks];       // the straddling nodes of every level: cell indices, ascending
    uint4 topo[kLevels][kMomMaxBlocks];          // ... and their topology
    uint32_t cnt[kLevels + 1];
};

// The owned nodes [lo, hi) of one level: eight lanes per node, the next node's topology is requested before the current
// node's children are summed.
__device__ __forceinline__ void node_pass(uint32_t lo, uint32_t hi, const uint4* __restrict__ topo, double* mom64, float* box, const RecOut& ro,
                                          NodeScratch* sx, uint8_t* dirty, bool partial) {
    const int tid = threadIdx.x, grp = tid >> 3, sub = tid & 7;
    const uint32_t cnt = hi - lo;
    uint4 tp = make_uint4(0u, 0u, 0u, 0u);
    if ((uint32_t)grp < cnt) tp = __ldg(topo + lo + grp);
    for (uint32_t q0 = 0; q0 < cnt; q0 += kMomGroups) {
        const uint32_t q = q0 + grp;
        const uint4 t = tp;
        if (q + kMomGroups < cnt) tp = __ldg(topo + lo + q + kMomGroups);
        bool node = q < cnt && t.w != t.z;
        if (partial) {                                                // a node whose children are all clean keeps what it holds
            uint32_t d = 0;
            if (node && (uint32_t)sub < t.w - t.z) d = __ldcg(dirty + t.z + sub);
            d |= __shfl_xor_sync(0xFFFFFFFFu, d, 1, 8); d |= __shfl_xor_sync(0xFFFFFFFFu, d, 2, 8); d |= __shfl_xor_sync(0xFFFFFFFFu, d, 4, 8);
            if (node && sub == 0) dirty[lo + q] = (uint8_t)(d ? 1 : 0);
            node = node && d != 0;
        }
        if (!__any_sync(0xFFFFFFFFu, node)) continue;                 // (warp-uniform) none of this warp's four cells is a node to compute
        const int nch = node ? (int)(t.w - t.z) : 0;
        Child ch;
        child_clear(ch);
        if (sub < nch) child_load_global(ch, mom64, box, t.z + sub);
        Mom m;
        node_moments8(m, ch, nch, sub, sx[grp]);
        if (node) {
            const uint32_t c = lo + q;
            if (sub == 0) mom_store(m, mom64, box, c);
            if (ro.enabled && sub == 1) rec_store(make_record(m, ro.theta, ro.mac_kind, t.x, t.y, t.z, t.w), ro, c);
        }
    }
}

// Leaves that START inside the block's particle range (a leaf that reaches into the next range is still computed here:
// it depends on nothing but the particles) and the nodes that lie entirely inside it.
__global__ void __launch_bounds__(kMomThreads, 1) k_moments(const DevScalars* __restrict__ sc, const float4* __restrict__ pos, int n, int P, int tiles,
                                                            const uint32_t* __restrict__ tile_base, const uint4* __restrict__ topo,
                                                            double* mom64, float* box, uint32_t* span, const RecOut ro,
                                                            const uint8_t* __restrict__ active, uint8_t* dirty) {
    extern __shared__ __align__(16) unsigned char mom_smem[];
    NodeScratch* sx = reinterpret_cast<NodeScratch*>(mom_smem);
    const bool partial = active != nullptr;                   // block time-steps (L266): only cells with an updated particle below them
    __shared__ uint32_t s_lo[kLevels], s_hi[kLevels], s_hin[kLevels], s_pre[kLevels + 1];
    const int tid = threadIdx.x;
    const uint32_t b = blockIdx.x, nb = gridDim.x;
    const int nlev = (int)sc->n_levels;                       // 0: capacity overflow, the tree is empty
    // ---- the cells that start inside this block's particle range [b P, (b + 1) P): one index range per level
    if (tid < kLevels) {
        const int L = tid;
        uint32_t lo = 0, hi = 0, hin = 0, sp = kNone;
        if (L < nlev) {
            const uint32_t off = sc->level_offset[L];
            const int64_t tb0 = (int64_t)b * P / kTreeTile, tb1 = (int64_t)(b + 1) * P / kTreeTile;
            lo = off + tile_base[(size_t)L * tiles + tb0];
            hi = tb1 < tiles ? off + tile_base[(size_t)L * tiles + tb1] : sc->level_offset[L + 1];
            hin = hi;
            if (hi > lo) {
                const uint4 t = topo[hi - 1];
                if ((int64_t)t.y > (int64_t)(b + 1) * P && t.w != t.z) { sp = hi - 1; hin = hi - 1; }   // the last one is a node that straddles the boundary
            }
        }
        s_lo[L] = lo; s_hi[L] = hi; s_hin[L] = hin;
        span[(size_t)L * nb + b] = sp;
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t run = 0;
        for (int L = 0; L < kLevels; ++L) { s_pre[L] = run; run += s_hi[L] - s_lo[L]; }
        s_pre[kLevels] = run;
    }
    __syncthreads();
    // ---- the block's particles, once, coalesced, into shared memory (the node scratch is not in use yet) when they fit
    float4* spos = reinterpret_cast<float4*>(mom_smem);
    const uint32_t p0 = b * (uint32_t)P;
    const uint32_t staged = P <= kMomStage ? min((uint32_t)P, (uint32_t)n - min((uint32_t)n, p0)) : 0u;
    // one contiguous run of up to 128 KB: a 1-D bulk copy (TMA, cp.async.bulk) issued by one thread and completed on an
    // mbarrier, instead of seven 16-byte loads and stores per thread (measured against plain loads: profiles/r2_tma_ab.md)
    __shared__ __align__(8) unsigned long long s_bar;
    const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0 && staged) {
        const uint32_t bytes = staged * 16u;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
        for (uint32_t off = 0; off < bytes; off += 32768u) {
            const uint32_t len = min(32768u, bytes - off);
            const uint32_t dst = (uint32_t)__cvta_generic_to_shared(mom_smem + off);
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(dst), "l"(reinterpret_cast<const unsigned char*>(pos + p0) + off), "r"(len), "r"(bar) : "memory");
        }
    }
    if (staged) {
        uint32_t done = 0;
        while (!done)
            asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(bar) : "memory");
    }
    auto ld = [&](uint32_t i) -> float4 { return (i - p0 < staged) ? spos[i - p0] : __ldg(pos + i); };
    // ---- leaves: one thread each
    const uint32_t total = s_pre[kLevels];
    for (uint32_t f = tid; f < total; f += kMomThreads) {
        int L = 0;
#pragma unroll
        for (int k = 1; k < kLevels; ++k) L += (f >= s_pre[k]) ? 1 : 0;       // s_pre is non-decreasing
        const uint32_t c = s_lo[L] + (f - s_pre[L]);
        const uint4 t = __ldg(topo + c);
        if (t.w != t.z) continue;
        if (partial) {
            uint32_t any = 0;
            for (uint32_t i = t.x; i < t.y; ++i) any |= __ldg(active + i);
            dirty[c] = (uint8_t)(any ? 1 : 0);
            if (!any) continue;
        }
        Mom m;
        leaf_moments(m, ld, t.x, t.y);
        mom_store(m, mom64, box, c);
        if (ro.enabled) rec_store(make_record(m, ro.theta, ro.mac_kind, t.x, t.y, t.z, t.w), ro, c);
    }
    __syncthreads();
    // ---- owned nodes, deepest level first
    for (int L = nlev - 2; L >= 0; --L) {
        if (s_hin[L] == s_lo[L]) continue;                    // (uniform over the block)
        node_pass(s_lo[L], s_hin[L], topo, mom64, box, ro, sx, dirty, partial);
        __syncthreads();
    }
}

// The straddling nodes, level by level from the deepest one, by ONE THREAD-BLOCK CLUSTER of eight CTAs that keeps them in
// (distributed) shared memory: node q of a level belongs to CTA q mod 8, which stores the result in its own shared memory
// (and in the cell arrays); a child that straddles a boundary itself was computed one level ago and is read from the shared
// memory of the CTA that owns it (DSMEM), any other child is a cell of k_moments (L2).  cluster.sync() separates the
// levels, so the dependent chain over the levels of the tree never goes through global memory, and the fp64 work of a
// level is spread over eight SMs.
__global__ void __cluster_dims__(kSpanCtas, 1, 1) __launch_bounds__(kSpanThreads, 1)
k_moments_span(const DevScalars* __restrict__ sc, const uint4* __restrict__ topo, double* mom64, float* box,
               const uint32_t* __restrict__ span, uint32_t nb, const RecOut ro, uint8_t* dirty, int partial) {
    extern __shared__ __align__(16) unsigned char mom_smem[];
    SpanShared& sh = *reinterpret_cast<SpanShared*>(mom_smem);
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t rank = cluster.block_rank();
    const int tid = threadIdx.x, lane = tid & 31;
    const int nlev = (int)sc->n_levels;
    const int grp = tid >> 3, sub = tid & 7;
    // the straddling nodes of every level, in ascending order (= block order), and their topology (every CTA builds the
    // same lists): warp w takes levels w, w + 8, ...
    for (int L = tid >> 5; L < nlev; L += kSpanThreads / 32) {
        uint32_t run = 0;
        for (uint32_t b0 = 0; b0 < nb; b0 += 32) {
            uint32_t sp = kNone;
            if (b0 + lane < nb) sp = __ldg(span + (size_t)L * nb + b0 + lane);
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, sp != kNone);
            if (sp != kNone) {
                const uint32_t at = run + __popc(bal & ((1u << lane) - 1u));
                sh.list[L][at] = sp;
                sh.topo[L][at] = __ldg(topo + sp);
            }
            run += __popc(bal);
        }
        if (lane == 0) sh.cnt[L] = run;
    }
    if (tid == 0) sh.cnt[nlev] = 0;
    __syncthreads();
    // A node's children are (a) cells that k_moments finished before this kernel started, or (b) straddling nodes of the
    // level below.  (a) does not depend on anything computed here: while the cluster barrier of level L is pending (between
    // its arrive and its wait), the lanes work out where the children of their node of level L - 1 are (binary search) and
    // request the (a)-children, so that the chain over the levels holds only the shared-memory reads of the (b)-children,
    // the sums and the barrier.  With at most kMomMaxBlocks straddling nodes per level a CTA has at most one node per lane
    // group and level: node q = rank + kSpanCtas * grp.
    struct Desc { bool have; uint32_t c; uint4 t; int nch; int src; };
    auto describe = [&](int L) {
        Desc d;
        d.have = false; d.c = 0; d.t = make_uint4(0u, 0u, 0u, 0u); d.nch = 0; d.src = -1;
        if (L < 0) return d;
        const uint32_t q = rank + kSpanCtas * (uint32_t)grp;
        if (q >= sh.cnt[L]) return d;
        d.have = true;
        d.c = sh.list[L][q];
        d.t = sh.topo[L][q];
        d.nch = (int)(d.t.w - d.t.z);
        if (sub < d.nch) {
            const uint32_t cc = d.t.z + sub;
            const uint32_t* listb = sh.list[L + 1 < kLevels ? L + 1 : L];
            const int cntb = (int)sh.cnt[L + 1];
            int lo2 = 0, hi2 = cntb;
            while (lo2 < hi2) {
                const int mid = (lo2 + hi2) >> 1;
                if (listb[mid] < cc) lo2 = mid + 1; else hi2 = mid;
            }
            if (lo2 < cntb && listb[lo2] == cc) d.src = lo2;             // computed one level earlier by CTA lo2 mod 8, kept in its slot lo2 / 8
        }
        return d;
    };
    auto request = [&](const Desc& d, Child& ch, Child& own, uint32_t& dflag) {
        child_clear(ch);
        child_clear(own);
        dflag = 0;
        if (d.have && sub < d.nch && d.src < 0) {
            child_load_global(ch, mom64, box, d.t.z + sub);
            if (partial) dflag = __ldcg(dirty + d.t.z + sub);
        }
        if (partial && d.have && sub == 0) child_load_global(own, mom64, box, d.c);   // (handed on unchanged when no child is dirty)
    };
    int Lc = nlev - 1;
    while (Lc >= 0 && sh.cnt[Lc] == 0u) --Lc;                              // (levels without a straddling node: the same for every CTA)
    Desc cur_d = describe(Lc);
    Child cur_ch, cur_own;
    uint32_t cur_df;
    request(cur_d, cur_ch, cur_own, cur_df);
    while (Lc >= 0) {
        const int L = Lc;
        const int cur = L & 1, below = cur ^ 1;
        int Ln = L - 1;
        while (Ln >= 0 && sh.cnt[Ln] == 0u) --Ln;
        const bool have = cur_d.have;
        const uint4 t = cur_d.t;
        const uint32_t c = cur_d.c;
        int nch = cur_d.nch;
        Child ch = cur_ch;
        uint32_t d = cur_df;
        if (cur_d.src >= 0) {                                              // (b): from the shared memory of the CTA that owns it (DSMEM)
            const SpanCell* remote = cluster.map_shared_rank(&sh.cell[below][cur_d.src / kSpanCtas], cur_d.src % kSpanCtas);
            child_load_shared(ch, *remote);
            d = __float_as_uint(remote->pad[0]);
        }
        bool clean = false;
        if (partial) {                                                     // all children clean: hand on what the cell arrays hold
            d |= __shfl_xor_sync(0xFFFFFFFFu, d, 1, 8); d |= __shfl_xor_sync(0xFFFFFFFFu, d, 2, 8); d |= __shfl_xor_sync(0xFFFFFFFFu, d, 4, 8);
            if (have && sub == 0) dirty[c] = (uint8_t)(d ? 1 : 0);
            clean = have && d == 0;
            if (clean) { nch = 0; child_clear(ch); }
        }
        Mom m;
        node_moments8(m, ch, nch, sub, sh.sx[grp]);
        if (have && sub == 0) {
            SpanCell& o = sh.cell[cur][grp];
            if (clean) {
                o.m[0] = cur_own.M; o.m[1] = cur_own.c[0]; o.m[2] = cur_own.c[1]; o.m[3] = cur_own.c[2];
#pragma unroll
                for (int k = 0; k < 6; ++k) o.m[4 + k] = cur_own.Q[k];
#pragma unroll
                for (int k = 0; k < 3; ++k) { o.b[k] = cur_own.bn[k]; o.b[3 + k] = cur_own.bx[k]; }
            } else {
                o.m[0] = m.M; o.m[1] = m.com[0]; o.m[2] = m.com[1]; o.m[3] = m.com[2];
#pragma unroll
                for (int k = 0; k < 6; ++k) o.m[4 + k] = m.Q[k];
#pragma unroll
                for (int k = 0; k < 3; ++k) { o.b[k] = m.bmin[k]; o.b[3 + k] = m.bmax[k]; }
            }
            o.pad[0] = __uint_as_float(partial ? (d ? 1u : 0u) : 1u);
        }
        cluster.barrier_arrive();                                          // this CTA's part of the level is in its shared memory
        // while the barrier is pending: the stores to the cell arrays (the peers only need the shared-memory copy) and
        // everything about the next level that does not depend on this one
        if (have && !clean) {
            if (sub == 0) mom_store(m, mom64, box, c);
            if (ro.enabled && sub == 1) rec_store(make_record(m, ro.theta, ro.mac_kind, t.x, t.y, t.z, t.w), ro, c);
        }
        cur_d = describe(Ln);
        request(cur_d, cur_ch, cur_own, cur_df);
        cluster.barrier_wait();                                            // ... and so is everybody else's
        Lc = Ln;
    }
}

// fp32 records alone (theta or the MAC changed on an existing tree).
__global__ void __launch_bounds__(256) k_cell_record(const DevScalars* __restrict__ sc, const uint4* __restrict__ topo,
                                                     const double* __restrict__ mom64, const float* __restrict__ box, const RecOut ro) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const double* s = mom64 + 10 * (size_t)c;
        const float* bb = box + 6 * (size_t)c;
        Mom m;
        m.M = s[0]; m.com[0] = s[1]; m.com[1] = s[2]; m.com[2] = s[3];
#pragma unroll
        for (int k = 0; k < 6; ++k) m.Q[k] = s[4 + k];
#pragma unroll
        for (int k = 0; k < 3; ++k) { m.bmin[k] = bb[k]; m.bmax[k] = bb[3 + k]; }
        const uint4 t = topo[c];
        rec_store(make_record(m, ro.theta, ro.mac_kind, t.x, t.y, t.z, t.w), ro, c);
    }
}

static RecOut rec_out(bh_ctx* c, float theta, bool enabled) {
    RecOut ro;
    ro.trec = c->ws.trec; ro.tlink = c->ws.tlink; ro.erec = c->ws.erec;
    ro.theta = theta; ro.mac_kind = c->mac_kind; ro.enabled = enabled ? 1 : 0;
    return ro;
}

int moments_init(bh_ctx* c) {
    BH_CUDA(c, cudaFuncSetAttribute(k_moments_span, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SpanShared)));
    BH_CUDA(c, cudaFuncSetAttribute(k_moments, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(NodeScratch) * kMomGroups)));
    return BH_OK;
}

// theta > 0: the fp32 records are written in the same pass (c->rec_theta / rec_mac remember for which criterion).
int stage_moments(bh_ctx* c, float theta, const uint8_t* d_active, cudaStream_t s) {
    const int64_t n = c->n;
    // particles per block: a multiple of the tree tile; one block per SM (one wave), at most kMomMaxBlocks blocks
    const int64_t nb_target = std::min<int64_t>(c->sm_count, kMomMaxBlocks);
    const int64_t P = div_up(div_up(n + 1, nb_target), kTreeTile) * kTreeTile;
    const int nb = (int)div_up(n + 1, P);
    const int tiles = (int)div_up(n + 1, kTreeTile);
    const bool rec = theta > 0.0f;
    // A partial refresh rewrites the fp32 records of the dirty cells only; the others keep what they hold, which is good only
    // if that was written for this same criterion.  Otherwise the records are not valid as a whole and stage_walk redoes them.
    const bool partial = d_active != nullptr;
    const bool kept = c->rec_valid && c->rec_theta == theta && c->rec_mac == c->mac_kind;
    BH_LAUNCH(c, k_moments, nb, kMomThreads, sizeof(NodeScratch) * kMomGroups, s, c->ws.sc, c->ws.pos[c->cur], (int)n, (int)P, tiles, c->ws.tile_cnt, c->ws.c_topo,
              c->ws.mom64, c->ws.box, c->ws.mom_span, rec_out(c, theta, rec), d_active, c->ws.c_dirty);
    BH_LAUNCH(c, k_moments_span, kSpanCtas, kSpanThreads, sizeof(SpanShared), s, c->ws.sc, c->ws.c_topo, c->ws.mom64, c->ws.box,
              c->ws.mom_span, (uint32_t)nb, rec_out(c, theta, rec), c->ws.c_dirty, d_active ? 1 : 0);
    c->rec_valid = rec && (!partial || kept);
    c->rec_theta = theta;
    c->rec_mac = c->mac_kind;
    return BH_OK;
}

int stage_cell_record(bh_ctx* c, float theta, cudaStream_t s) {
    const int grid = (int)std::min<int64_t>(div_up(c->max_cells, 256), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_cell_record, grid, 256, 0, s, c->ws.sc, c->ws.c_topo, c->ws.mom64, c->ws.box, rec_out(c, theta, true));
    c->rec_valid = true;
    c->rec_theta = theta;
    c->rec_mac = c->mac_kind;
    return BH_OK;
}

}  // namespace bh
