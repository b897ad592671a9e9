// moments.cu -- S6: monopole + quadrupole moments and tight boxes, bottom-up, in binary64 with a fixed operation
// order ("performed in double precision ... converted back to single precision"; Fig.4), then the
// fp32 walk record with the opening radius of Eq.1.
// Every fp64 operation is an explicit round-to-nearest intrinsic so that no multiply-add is ever fused: the fp32
// roundings of these values feed the MAC, and a one-ulp difference would flip an opening decision somewhere.
#include <algorithm>
#include "bh_internal.cuh"

namespace bh {

struct Mom {
    double M, S[3], com[3], Q[6];
    float bmin[3], bmax[3];
};

__device__ __forceinline__ void mom_store(const Mom& m, double* __restrict__ mom64, float* __restrict__ box, uint32_t c) {
    double* o = mom64 + 10 * (size_t)c;
    o[0] = m.M; o[1] = m.com[0]; o[2] = m.com[1]; o[3] = m.com[2];
#pragma unroll
    for (int k = 0; k < 6; ++k) o[4 + k] = m.Q[k];
    float* b = box + 6 * (size_t)c;
#pragma unroll
    for (int k = 0; k < 3; ++k) { b[k] = m.bmin[k]; b[3 + k] = m.bmax[k]; }
}

// Leaf: M = sum m; S = sum m x; com = S / M; Q_jk = sum (m r_j) r_k, r = x - com; particles in ascending order.
__device__ __forceinline__ void leaf_moments(Mom& m, const float4* __restrict__ pos, uint32_t b, uint32_t e) {
    m.M = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) { m.S[k] = 0.0; m.bmin[k] = INFINITY; m.bmax[k] = -INFINITY; }
#pragma unroll
    for (int k = 0; k < 6; ++k) m.Q[k] = 0.0;
    for (uint32_t i = b; i < e; ++i) {
        const float4 p = __ldg(pos + i);
        const double w = (double)p.w;
        m.M = __dadd_rn(m.M, w);
        m.S[0] = __dadd_rn(m.S[0], __dmul_rn(w, (double)p.x));
        m.S[1] = __dadd_rn(m.S[1], __dmul_rn(w, (double)p.y));
        m.S[2] = __dadd_rn(m.S[2], __dmul_rn(w, (double)p.z));
        m.bmin[0] = fminf(m.bmin[0], p.x); m.bmax[0] = fmaxf(m.bmax[0], p.x);
        m.bmin[1] = fminf(m.bmin[1], p.y); m.bmax[1] = fmaxf(m.bmax[1], p.y);
        m.bmin[2] = fminf(m.bmin[2], p.z); m.bmax[2] = fmaxf(m.bmax[2], p.z);
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) m.com[k] = __ddiv_rn(m.S[k], m.M);
    for (uint32_t i = b; i < e; ++i) {
        const float4 p = __ldg(pos + i);
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

// Node: M = sum M_c; S = sum M_c com_c; com = S / M; Q_jk = sum_c ((Q + Q_c,jk) + (M_c d_j) d_k), d = com_c - com; children
// in ascending order.  The children were written by other threads of this launch: read them from L2 (ld.global.cg).
__device__ __forceinline__ void node_moments(Mom& m, const double* mom64, const float* box, uint32_t cb, uint32_t ce) {
    m.M = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) { m.S[k] = 0.0; m.bmin[k] = INFINITY; m.bmax[k] = -INFINITY; }
#pragma unroll
    for (int k = 0; k < 6; ++k) m.Q[k] = 0.0;
    for (uint32_t k2 = cb; k2 < ce; ++k2) {
        const double* mc = mom64 + 10 * (size_t)k2;
        const float* bc = box + 6 * (size_t)k2;
        const double Mc = __ldcg(mc);
        m.M = __dadd_rn(m.M, Mc);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            m.S[k] = __dadd_rn(m.S[k], __dmul_rn(Mc, __ldcg(mc + 1 + k)));
            m.bmin[k] = fminf(m.bmin[k], __ldcg(bc + k));
            m.bmax[k] = fmaxf(m.bmax[k], __ldcg(bc + 3 + k));
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) m.com[k] = __ddiv_rn(m.S[k], m.M);
    for (uint32_t k2 = cb; k2 < ce; ++k2) {
        const double* mc = mom64 + 10 * (size_t)k2;
        const double Mc = __ldcg(mc);
        const double dx = __dsub_rn(__ldcg(mc + 1), m.com[0]);
        const double dy = __dsub_rn(__ldcg(mc + 2), m.com[1]);
        const double dz = __dsub_rn(__ldcg(mc + 3), m.com[2]);
        const double tx = __dmul_rn(Mc, dx), ty = __dmul_rn(Mc, dy), tz = __dmul_rn(Mc, dz);
        m.Q[0] = __dadd_rn(__dadd_rn(m.Q[0], __ldcg(mc + 4)), __dmul_rn(tx, dx));
        m.Q[1] = __dadd_rn(__dadd_rn(m.Q[1], __ldcg(mc + 5)), __dmul_rn(ty, dy));
        m.Q[2] = __dadd_rn(__dadd_rn(m.Q[2], __ldcg(mc + 6)), __dmul_rn(tz, dz));
        m.Q[3] = __dadd_rn(__dadd_rn(m.Q[3], __ldcg(mc + 7)), __dmul_rn(tx, dy));
        m.Q[4] = __dadd_rn(__dadd_rn(m.Q[4], __ldcg(mc + 8)), __dmul_rn(tx, dz));
        m.Q[5] = __dadd_rn(__dadd_rn(m.Q[5], __ldcg(mc + 9)), __dmul_rn(ty, dz));
    }
}

// The whole bottom-up pass in ONE launch (the paper goes level by level: one launch per level, ~20
// dependent launches that are nearly all empty).  A thread computes a leaf, publishes it (store, fence) and counts itself
// in at the parent (c_arrive, zeroed by k_emit_cells); whoever arrives last at a node finds all of its children
// published, computes the node and climbs on.  Nobody waits, so the launch cannot deadlock; every node is still computed
// from its children in ascending order, so the values are bit-identical to the level-by-level pass.
__global__ void __launch_bounds__(128) k_moments(const DevScalars* __restrict__ sc, const float4* __restrict__ pos,
                                                 const uint32_t* __restrict__ c_pbegin, const uint32_t* __restrict__ c_pend,
                                                 const uint32_t* __restrict__ c_cbegin, const uint32_t* __restrict__ c_cend,
                                                 const uint32_t* __restrict__ c_parent, uint32_t* __restrict__ c_arrive,
                                                 double* mom64, float* box) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        if (c_cend[c] != c_cbegin[c]) continue;   // node: computed by its last child
        Mom m;
        leaf_moments(m, pos, c_pbegin[c], c_pend[c]);
        mom_store(m, mom64, box, c);
        uint32_t cur = c;
        for (;;) {
            const uint32_t par = c_parent[cur];
            if (par == kNone) break;
            const uint32_t cb = c_cbegin[par], ce = c_cend[par];
            __threadfence();                                   // publish `cur` before counting in
            if (atomicAdd(c_arrive + par, 1u) != ce - cb - 1u) break;
            c_arrive[par] = 0u;                                // ready for the next pass (bh_refresh_moments runs without k_emit_cells)
            __threadfence();                                   // all children are published; do not read them early
            node_moments(m, mom64, box, cb, ce);
            mom_store(m, mom64, box, par);
            cur = par;
        }
    }
}

// fp32 records per cell: what the walk tests (trec: com, r2open; tlink: first child / particle, count | leaf << 31) and what
// the force loop consumes (erec, 48 B: (com, M) (Qm_xx, Qm_yy, Qm_zz, Qm_xy) (Qm_xz, Qm_yz, nTh, n3Th)),
// with the opening radius of Eq.1:  l = longest side of the tight box (A14),
// delta = |com - box centre|, r2open = (l / theta + delta)^2, all in single fp32 operations (O8).
__global__ void __launch_bounds__(256) k_cell_record(const DevScalars* __restrict__ sc, float theta, int mac_kind,
                                                     const uint32_t* __restrict__ c_pbegin, const uint32_t* __restrict__ c_pend,
                                                     const uint32_t* __restrict__ c_cbegin, const uint32_t* __restrict__ c_cend,
                                                     const double* __restrict__ mom64, const float* __restrict__ box,
                                                     float4* __restrict__ trec, uint2* __restrict__ tlink, float4* __restrict__ erec) {
    const uint32_t nc = sc->n_cells;
    for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < nc; c += gridDim.x * blockDim.x) {
        const double* m = mom64 + 10 * (size_t)c;
        const float* b = box + 6 * (size_t)c;
        const float M = (float)m[0];
        const float cx = (float)m[1], cy = (float)m[2], cz = (float)m[3];
        float l = fmaxf(fmaxf(__fsub_rn(b[3], b[0]), __fsub_rn(b[4], b[1])), __fsub_rn(b[5], b[2]));
        l = fmaxf(l, 0.0f);
        const float ux = __fsub_rn(cx, __fmul_rn(0.5f, __fadd_rn(b[0], b[3])));
        const float uy = __fsub_rn(cy, __fmul_rn(0.5f, __fadd_rn(b[1], b[4])));
        const float uz = __fsub_rn(cz, __fmul_rn(0.5f, __fadd_rn(b[2], b[5])));
        const float s2 = __fadd_rn(__fadd_rn(__fmul_rn(ux, ux), __fmul_rn(uy, uy)), __fmul_rn(uz, uz));
        const float delta = __fsqrt_rn(s2);
        const float ropen = mac_kind == 1 ? __fdiv_rn(l, theta) : __fadd_rn(__fdiv_rn(l, theta), delta);   // A28 / Eq.1
        const float r2open = __fmul_rn(ropen, ropen);
        const uint32_t cb = c_cbegin[c], ce = c_cend[c];
        const bool leaf = (ce == cb);
        uint2 link;
        link.x = leaf ? c_pbegin[c] : cb;
        link.y = leaf ? ((c_pend[c] - c_pbegin[c]) | 0x80000000u) : (ce - cb);
        // evaluation record, pre-scaled once: Qm = -3 Q, nTh = -T/2, n3Th = -3T/2 (T = trace of Q)
        const float qxx = (float)m[4], qyy = (float)m[5], qzz = (float)m[6], qxy = (float)m[7], qxz = (float)m[8], qyz = (float)m[9];
        const float T = (qxx + qyy) + qzz;
        trec[c] = make_float4(cx, cy, cz, r2open);
        tlink[c] = link;
        erec[3 * (size_t)c] = make_float4(cx, cy, cz, M);
        erec[3 * (size_t)c + 1] = make_float4(-3.0f * qxx, -3.0f * qyy, -3.0f * qzz, -3.0f * qxy);
        erec[3 * (size_t)c + 2] = make_float4(-3.0f * qxz, -3.0f * qyz, -0.5f * T, -1.5f * T);
    }
}

int stage_moments(bh_ctx* c, cudaStream_t s) {
    const int grid = (int)std::min<int64_t>(div_up(std::min<int64_t>(c->max_cells, c->n + c->n / 2 + 1), 128), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_moments, grid, 128, 0, s, c->ws.sc, c->ws.pos[c->cur], c->ws.c_pbegin, c->ws.c_pend, c->ws.c_cbegin,
              c->ws.c_cend, c->ws.c_parent, c->ws.c_arrive, c->ws.mom64, c->ws.box);
    return BH_OK;
}

int stage_cell_record(bh_ctx* c, float theta, cudaStream_t s) {
    const int grid = (int)std::min<int64_t>(div_up(c->max_cells, 256), (int64_t)c->sm_count * 16);
    BH_LAUNCH(c, k_cell_record, grid, 256, 0, s, c->ws.sc, theta, c->mac_kind, c->ws.c_pbegin, c->ws.c_pend, c->ws.c_cbegin, c->ws.c_cend,
              c->ws.mom64, c->ws.box, c->ws.trec, c->ws.tlink, c->ws.erec);
    return BH_OK;
}

}  // namespace bh
