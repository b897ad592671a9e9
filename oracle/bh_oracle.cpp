// bh_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct CPU statement of the per-step Barnes-Hut force
// pipeline of arxiv/paper_1106_1900 (Bedorf, Gaburov & Portegies Zwart), written from
// /root/reference/PAPER.md ("L<n>" below = PAPER.md line n) and the readings recorded in
// DESIGN.md ("A<n>").  It shares no code with the CUDA path under
// paper_1106_1900_b200/; only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.
//
// The method is an approximation (tree + multipoles), so the oracle follows the algorithm
// step by step, in the paper's order:
//   O1 domain (L374)  O2 grid coords (L374)  O3 Morton key (L376, L392)  O4 stable sort (L59, L352, L362)
//   O5 reorder (L174) O6 sparse octree (L63, L65, Fig.1-2)  O7 groups (L75)
//   O8 moments + boxes, binary64, fixed order (L109-115, L127, L266)
//   O9 group walk with Eq.1 (L83, L87, L125)  O10 p-p / p-c forces, binary64 (L85, L109)
//   O11 leapfrog (L105)   plus an O(N^2) binary64 direct sum (L131: theta -> 0 limit), and the block time-step
//   scheme of L101 / L105 / L264-266 in the reading A29 (orc_rungs, orc_block_*).
//
// Pins (tests/ -m "not gpu"): dilate worked example L376, mask example L67, List 1 (L380-390) as an
// independent dilate, numpy stable argsort, a second tree construction (the paper's literal
// per-level mask/flag loop, tests/level_loop_tree.py), structural tree invariants, direct-sum root
// moments, the parallel-axis identity, closed-form two-mass quadrupole, (s/R)^3 convergence,
// brute force O(N^2), theta -> 0, analytic Plummer potential, two-body orbit, reversibility;
// Eq.1's l, delta, r_open: hand-built cells with closed-form values and a target one ulp on either side of the
// threshold, plus a numpy-float32 restatement over every cell and a root-to-leaf walk with it; block time-steps: rung
// closed forms and thresholds, commensurate times, the one-rung case against the shared-step leapfrog, second order on a
// two-body orbit with unequal steps, energy over a macro-step; group boxes (orc_group_boxes): numpy min / max over every
// group's slice, equality with the cell's box for whole-cell groups, overflow-leaf chunks.
// Parity unpinned against the paper: magnitudes of the interaction counts (Fig.6 inset is an image).
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
// -ffp-contract=off: every "+f", "*f", "+d", "*d" below is ONE IEEE operation; fmaf() only where written.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <vector>

namespace {

constexpr int KEY_BITS = 20;   // bits per axis (L392: 60-bit key, 20 levels)
constexpr int MAXLEVEL = 20;

struct Cell {
    int32_t level;
    uint64_t prefix;   // key >> (60 - 3*level)
    int64_t pbegin, pcount;
    int64_t parent_tmp;           // index in creation order
    std::vector<int64_t> kids;    // creation-order indices, ascending octant
};

inline uint64_t level_prefix(uint64_t key, int level) {
    return level == 0 ? 0 : key >> (60 - 3 * level);
}

// O6: direct recursion on a run [b, e) of sorted keys that share their level-L prefix.
int64_t build_rec(const uint64_t* keys, int64_t b, int64_t e, int level, int nleaf,
                  int64_t parent, std::vector<Cell>& cells) {
    const int64_t me = (int64_t)cells.size();
    cells.push_back(Cell{level, level_prefix(keys[b], level), b, e - b, parent, {}});
    if (e - b <= nleaf || level == MAXLEVEL) return me;   // leaf (A7: "up-to Nleaf"; A9: max depth)
    int64_t s = b;
    while (s < e) {   // split by the next three key bits
        const uint64_t p = level_prefix(keys[s], level + 1);
        int64_t t = s + 1;
        while (t < e && level_prefix(keys[t], level + 1) == p) ++t;
        const int64_t kid = build_rec(keys, s, t, level + 1, nleaf, me, cells);
        cells[me].kids.push_back(kid);
        s = t;
    }
    return me;
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------------------------
// O1 (L374 "shifting the reference frame to the lower left corner of the domain"; A2):
// lo_k = min_i x_ik, hi_k = max_i x_ik; ext = max_k (hi_k -f lo_k), 1 if 0;
// frexpf(ext) = (mu, e), mu in [0.5, 1): cube side 2^e > ext.
// pos4: float[n][4] = (x, y, z, m).  Returns 0, or -1 on a non-finite position / mass <= 0 (A27).
int orc_domain(int64_t n, const float* pos4, float lo[3], float hi[3], int32_t* e_out) {
    for (int k = 0; k < 3; ++k) { lo[k] = INFINITY; hi[k] = -INFINITY; }
    int bad = 0;
    for (int64_t i = 0; i < n; ++i) {
        for (int k = 0; k < 3; ++k) {
            const float x = pos4[4 * i + k];
            if (!std::isfinite(x)) bad = 1;
            lo[k] = std::min(lo[k], x);
            hi[k] = std::max(hi[k], x);
        }
        const float m = pos4[4 * i + 3];
        if (!(m > 0.0f) || !std::isfinite(m)) bad = 1;
    }
    float ext = 0.0f;
    for (int k = 0; k < 3; ++k) ext = std::max(ext, hi[k] - lo[k]);
    if (ext == 0.0f) ext = 1.0f;
    int e = 0;
    (void)frexpf(ext, &e);
    *e_out = e;
    return bad ? -1 : 0;
}

// O2 + O3 (L374-392; A3, A4): ix = min(trunc((x -f lo_x) * 2^(20-e)), 2^20 - 1), likewise iy, iz;
// key = sum_b bit_b(ix) 2^(3b+2) + bit_b(iy) 2^(3b+1) + bit_b(iz) 2^(3b)   -- a plain per-bit loop.
// Scaling by a power of two is exact (ldexpf), so the only rounding is the subtraction.
void orc_keys(int64_t n, const float* pos4, const float lo[3], int32_t e, uint64_t* keys) {
    for (int64_t i = 0; i < n; ++i) {
        uint32_t g[3];
        for (int k = 0; k < 3; ++k) {
            const float d = pos4[4 * i + k] - lo[k];
            const float s = ldexpf(d, KEY_BITS - e);
            const float t = truncf(s);
            uint32_t v = (t <= 0.0f) ? 0u : (uint32_t)t;
            g[k] = std::min<uint32_t>(v, (1u << KEY_BITS) - 1u);
        }
        uint64_t key = 0;
        for (int b = 0; b < KEY_BITS; ++b) {
            key |= (uint64_t)((g[0] >> b) & 1u) << (3 * b + 2);
            key |= (uint64_t)((g[1] >> b) & 1u) << (3 * b + 1);
            key |= (uint64_t)((g[2] >> b) & 1u) << (3 * b);
        }
        keys[i] = key;
    }
}

// The dilate primitive on its own (L376: "converts the first 10 bits of an integer to a 30 bit
// representation"), generalised to `bits` bits, by the per-bit definition.  Pinned by the paper's
// worked example and by List 1 in tests.
uint64_t orc_dilate(uint32_t value, int32_t bits) {
    uint64_t r = 0;
    for (int b = 0; b < bits; ++b) r |= (uint64_t)((value >> b) & 1u) << (3 * b);
    return r;
}

// O4 (L59, L352, L362 "preserves the item ordering"; A6): stable ascending sort; perm[j] = input
// index of the j-th sorted particle.
void orc_sort(int64_t n, const uint64_t* keys, uint32_t* perm) {
    std::vector<uint32_t> p(n);
    std::iota(p.begin(), p.end(), 0u);
    std::stable_sort(p.begin(), p.end(), [&](uint32_t a, uint32_t b) { return keys[a] < keys[b]; });
    std::memcpy(perm, p.data(), sizeof(uint32_t) * n);
}

// O6 (L63, L65, Fig.1-2; A7-A10).  keys sorted.  A cell (L, p) exists iff it holds >= 1 particle and
// every proper ancestor holds > nleaf; leaf iff count <= nleaf or L = 20.  Numbering: level-major,
// ascending pbegin within a level.  Arrays must have room for the worst case; returns the cell count
// (call with null outputs to size).  level_offset has 22 entries.
int64_t orc_build_tree(int64_t n, const uint64_t* keys, int32_t nleaf,
                       int64_t* level_offset, int32_t* level, uint64_t* prefix,
                       int64_t* pbegin, int64_t* pcount, int64_t* child_begin, int32_t* nchild,
                       int64_t* parent) {
    std::vector<Cell> cells;
    cells.reserve((size_t)std::max<int64_t>(16, n / 2));
    // explicit stack instead of deep recursion would be equivalent; depth <= 20 so recursion is fine
    build_rec(keys, 0, n, 0, nleaf, -1, cells);
    const int64_t C = (int64_t)cells.size();
    if (!level) return C;
    std::vector<int64_t> order(C);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int64_t a, int64_t b) {
        if (cells[a].level != cells[b].level) return cells[a].level < cells[b].level;
        return cells[a].pbegin < cells[b].pbegin;
    });
    std::vector<int64_t> newidx(C);
    for (int64_t j = 0; j < C; ++j) newidx[order[j]] = j;
    for (int l = 0; l < MAXLEVEL + 2; ++l) level_offset[l] = 0;
    for (int64_t j = 0; j < C; ++j) level_offset[cells[order[j]].level + 1] += 1;
    for (int l = 1; l < MAXLEVEL + 2; ++l) level_offset[l] += level_offset[l - 1];
    for (int64_t j = 0; j < C; ++j) {
        const Cell& c = cells[order[j]];
        level[j] = c.level;
        prefix[j] = c.prefix;
        pbegin[j] = c.pbegin;
        pcount[j] = c.pcount;
        nchild[j] = (int32_t)c.kids.size();
        child_begin[j] = c.kids.empty() ? -1 : newidx[c.kids[0]];
        parent[j] = c.parent_tmp < 0 ? -1 : newidx[c.parent_tmp];
    }
    return C;
}

// O7 (L75; A12): cell c is a group iff pcount <= ncrit and (root or pcount(parent) > ncrit); a
// level-20 leaf with pcount > ncrit yields ceil(pcount / ncrit) chunks of consecutive particles.
// Groups ordered by pbegin.  Outputs sized n (worst case); returns the number of groups.
int64_t orc_groups(int64_t C, const int32_t* nchild, const int64_t* pbegin, const int64_t* pcount,
                   const int64_t* parent, int32_t ncrit,
                   int64_t* gcell, int64_t* gbegin, int64_t* gcount) {
    struct G { int64_t cell, b, c; };
    std::vector<G> gs;
    for (int64_t c = 0; c < C; ++c) {
        const bool parent_big = parent[c] < 0 || pcount[parent[c]] > ncrit;
        if (!parent_big) continue;
        if (pcount[c] <= ncrit) {
            gs.push_back({c, pbegin[c], pcount[c]});
        } else if (nchild[c] == 0) {   // overflow leaf at the deepest level
            for (int64_t o = 0; o < pcount[c]; o += ncrit)
                gs.push_back({c, pbegin[c] + o, std::min<int64_t>(ncrit, pcount[c] - o)});
        }
    }
    std::sort(gs.begin(), gs.end(), [](const G& a, const G& b) { return a.b < b.b; });
    for (size_t g = 0; g < gs.size(); ++g) { gcell[g] = gs[g].cell; gbegin[g] = gs[g].b; gcount[g] = gs[g].c; }
    return (int64_t)gs.size();
}

// O8 (L109-115 "double precision ... converted back to single precision", L127, L266; A14, A18, A20).
// Leaves: M = sum m_i; S_k = sum m_i * x_ik; com = S / M; Q_jk = sum (m_i r_j) r_k, r = x_i - com.
// Nodes (deepest level first): M = sum M_c; S_k = sum M_c * com_c,k; com = S / M;
//   Q_jk = sum_c (Q_c,jk + (M_c d_j) d_k), d = com_c - com   (parallel-axis shift), children in order.
// Boxes: exact min / max.  All sums sequential in ascending index, binary64, no fusion.
// mom64: double[C][10] = M, com xyz, Qxx, Qyy, Qzz, Qxy, Qxz, Qyz.   box: float[C][6] = min xyz, max xyz.
void orc_moments(int64_t C, const int64_t* level_offset, const int32_t* nchild,
                 const int64_t* child_begin, const int64_t* pbegin, const int64_t* pcount,
                 const float* pos4, double* mom64, float* box) {
    for (int L = MAXLEVEL; L >= 0; --L) {
        for (int64_t c = level_offset[L]; c < level_offset[L + 1]; ++c) {
            double M = 0.0, S[3] = {0.0, 0.0, 0.0}, Q[6] = {0, 0, 0, 0, 0, 0};
            float bmin[3] = {INFINITY, INFINITY, INFINITY}, bmax[3] = {-INFINITY, -INFINITY, -INFINITY};
            double com[3];
            if (nchild[c] == 0) {
                const int64_t b = pbegin[c], e = b + pcount[c];
                for (int64_t i = b; i < e; ++i) {
                    const double m = (double)pos4[4 * i + 3];
                    M = M + m;
                    for (int k = 0; k < 3; ++k) {
                        const float x = pos4[4 * i + k];
                        S[k] = S[k] + m * (double)x;
                        bmin[k] = std::min(bmin[k], x);
                        bmax[k] = std::max(bmax[k], x);
                    }
                }
                for (int k = 0; k < 3; ++k) com[k] = S[k] / M;
                for (int64_t i = b; i < e; ++i) {
                    const double m = (double)pos4[4 * i + 3];
                    double r[3], t[3];
                    for (int k = 0; k < 3; ++k) { r[k] = (double)pos4[4 * i + k] - com[k]; t[k] = m * r[k]; }
                    Q[0] = Q[0] + t[0] * r[0];
                    Q[1] = Q[1] + t[1] * r[1];
                    Q[2] = Q[2] + t[2] * r[2];
                    Q[3] = Q[3] + t[0] * r[1];
                    Q[4] = Q[4] + t[0] * r[2];
                    Q[5] = Q[5] + t[1] * r[2];
                }
            } else {
                const int64_t cb = child_begin[c], ce = cb + nchild[c];
                for (int64_t k2 = cb; k2 < ce; ++k2) {
                    const double* mc = mom64 + 10 * k2;
                    M = M + mc[0];
                    for (int k = 0; k < 3; ++k) {
                        S[k] = S[k] + mc[0] * mc[1 + k];
                        bmin[k] = std::min(bmin[k], box[6 * k2 + k]);
                        bmax[k] = std::max(bmax[k], box[6 * k2 + 3 + k]);
                    }
                }
                for (int k = 0; k < 3; ++k) com[k] = S[k] / M;
                for (int64_t k2 = cb; k2 < ce; ++k2) {
                    const double* mc = mom64 + 10 * k2;
                    double d[3], t[3];
                    for (int k = 0; k < 3; ++k) { d[k] = mc[1 + k] - com[k]; t[k] = mc[0] * d[k]; }
                    Q[0] = (Q[0] + mc[4]) + t[0] * d[0];
                    Q[1] = (Q[1] + mc[5]) + t[1] * d[1];
                    Q[2] = (Q[2] + mc[6]) + t[2] * d[2];
                    Q[3] = (Q[3] + mc[7]) + t[0] * d[1];
                    Q[4] = (Q[4] + mc[8]) + t[0] * d[2];
                    Q[5] = (Q[5] + mc[9]) + t[1] * d[2];
                }
            }
            double* out = mom64 + 10 * c;
            out[0] = M; out[1] = com[0]; out[2] = com[1]; out[3] = com[2];
            for (int k = 0; k < 6; ++k) out[4 + k] = Q[k];
            for (int k = 0; k < 3; ++k) { box[6 * c + k] = bmin[k]; box[6 * c + 3 + k] = bmax[k]; }
        }
    }
}

// O8, float outputs and the MAC inputs (Eq.1; A14-A16):
// l = max_k (bmax_k -f bmin_k); gc_k = 0.5f *f (bmin_k +f bmax_k); u = com~ -f gc;
// delta = sqrtf(((ux*ux) +f (uy*uy)) +f (uz*uz)); r_open = (l /f theta) +f delta; r2_open = r_open *f r_open.
// mom32: float[C][10] (same order as mom64);  mac: float[C][3] = l, delta, r2_open.
// mac_kind 0: Eq.1 (L125), r_open = l / theta + delta.  mac_kind 1: the minimum-distance MAC the paper also implemented
// (L129, [31]; reading A28): r_open = l / theta, to be compared with the distance between the group's box and the
// cell's tight BOX instead of its centre of mass (orc_walk_forces).
void orc_cell_floats(int64_t C, const double* mom64, const float* box, float theta, int32_t mac_kind,
                     float* mom32, float* mac) {
    for (int64_t c = 0; c < C; ++c) {
        for (int k = 0; k < 10; ++k) mom32[10 * c + k] = (float)mom64[10 * c + k];
        float l = 0.0f, u[3];
        for (int k = 0; k < 3; ++k) {
            const float bmin = box[6 * c + k], bmax = box[6 * c + 3 + k];
            l = std::max(l, bmax - bmin);
            const float gc = 0.5f * (bmin + bmax);
            u[k] = mom32[10 * c + 1 + k] - gc;
        }
        const float s2 = ((u[0] * u[0]) + (u[1] * u[1])) + (u[2] * u[2]);
        const float delta = sqrtf(s2);
        const float ropen = mac_kind == 1 ? (l / theta) : (l / theta) + delta;
        mac[3 * c + 0] = l;
        mac[3 * c + 1] = delta;
        mac[3 * c + 2] = ropen * ropen;
    }
}

// Group boxes (A13): exact per-axis min / max of the group's particles.  gbox: float[G][6].
void orc_group_boxes(int64_t G, const int64_t* gbegin, const int64_t* gcount, const float* pos4, float* gbox) {
    for (int64_t g = 0; g < G; ++g) {
        for (int k = 0; k < 3; ++k) { gbox[6 * g + k] = INFINITY; gbox[6 * g + 3 + k] = -INFINITY; }
        for (int64_t i = gbegin[g]; i < gbegin[g] + gcount[g]; ++i)
            for (int k = 0; k < 3; ++k) {
                gbox[6 * g + k] = std::min(gbox[6 * g + k], pos4[4 * i + k]);
                gbox[6 * g + 3 + k] = std::max(gbox[6 * g + 3 + k], pos4[4 * i + k]);
            }
    }
}

// O9 + O10 for a selection of groups (groups are independent, L75).
// O9 (L83, L87, Eq.1; A16, A17): breadth-first from the root;  d_k = max(max(gmin_k -f com_k, com_k -f gmax_k), 0);
//   d2 = fmaf(dz, dz, fmaf(dy, dy, dx *f dx));  d2 > r2_open -> cell list; else leaf -> particle list; else
//   children queued.  n_pc = accepted cells, n_pp = sum of pcount over opened leaves.
//   mac_kind 1 (L129, A28): d_k = max(max(gmin_k -f cmax_k, cmin_k -f gmax_k), 0) with the cell's tight box, r2_open = (l / theta)^2.
// O10 (L85, L109; A18, A19, A22), binary64 from the float inputs, eps2 = eps * eps:
//   p-p (j != i): dr = x_j - x_i, rho2 = |dr|^2 + eps2: phi -= m_j / rho; a += m_j dr / rho^3.
//   p-c: dr = com - x_i, T = Qxx+Qyy+Qzz, q = Q dr, w = dr . q:
//        phi += -M/rho + T/(2 rho^3) - 3 w/(2 rho^5);  a += dr (M/rho^3 - 3T/(2 rho^5) + 15 w/(2 rho^7)) - 3 q/rho^5.
// sel: indices of the groups to process (nsel of them).  npc / npp indexed by group id.  accpot: double[n][4]
// (ax, ay, az, phi), written only for particles of selected groups; may be null (counts only).
// list_cells / list_leaves (optional, for ONE selected group, nsel == 1): receive the lists; caps given.
void orc_walk_forces(int64_t n, const float* pos4,
                     const int32_t* nchild, const int64_t* child_begin,
                     const int64_t* pbegin, const int64_t* pcount,
                     const float* mom32, const float* mac, int32_t mac_kind, const float* box,
                     const int64_t* gbegin, const int64_t* gcount, const float* gbox,
                     int64_t nsel, const int64_t* sel, float eps,
                     int64_t* npc, int64_t* npp, double* accpot,
                     int64_t* list_cells, int64_t cap_cells, int64_t* list_leaves, int64_t cap_leaves) {
    (void)n;
    const double eps2 = (double)eps * (double)eps;
#pragma omp parallel for schedule(dynamic, 8)
    for (int64_t s = 0; s < nsel; ++s) {
        const int64_t g = sel[s];
        const float* gb = gbox + 6 * g;
        std::vector<int64_t> queue, cells_acc, leaves_open;
        queue.push_back(0);
        size_t head = 0;
        int64_t cnt_pp = 0;
        while (head < queue.size()) {
            const int64_t c = queue[head++];
            const float* cm = mom32 + 10 * c + 1;
            float d[3];
            if (mac_kind == 1) {      // A28: per-axis gap between the group's box and the cell's tight box (0 where they overlap)
                const float* cb = box + 6 * c;
                for (int k = 0; k < 3; ++k) d[k] = std::max(std::max(gb[k] - cb[3 + k], cb[k] - gb[3 + k]), 0.0f);
            } else {
                for (int k = 0; k < 3; ++k) d[k] = std::max(std::max(gb[k] - cm[k], cm[k] - gb[3 + k]), 0.0f);
            }
            const float d2 = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
            if (d2 > mac[3 * c + 2]) {
                cells_acc.push_back(c);
            } else if (nchild[c] == 0) {
                leaves_open.push_back(c);
                cnt_pp += pcount[c];
            } else {
                for (int k = 0; k < nchild[c]; ++k) queue.push_back(child_begin[c] + k);
            }
        }
        npc[g] = (int64_t)cells_acc.size();
        npp[g] = cnt_pp;
        if (list_cells && nsel == 1)
            for (size_t k = 0; k < cells_acc.size() && (int64_t)k < cap_cells; ++k) list_cells[k] = cells_acc[k];
        if (list_leaves && nsel == 1)
            for (size_t k = 0; k < leaves_open.size() && (int64_t)k < cap_leaves; ++k) list_leaves[k] = leaves_open[k];
        if (!accpot) continue;
        for (int64_t i = gbegin[g]; i < gbegin[g] + gcount[g]; ++i) {
            const double xi[3] = {(double)pos4[4 * i], (double)pos4[4 * i + 1], (double)pos4[4 * i + 2]};
            double a[3] = {0, 0, 0}, phi = 0;
            for (int64_t lc : leaves_open) {
                for (int64_t j = pbegin[lc]; j < pbegin[lc] + pcount[lc]; ++j) {
                    if (j == i) continue;
                    const double dr[3] = {(double)pos4[4 * j] - xi[0], (double)pos4[4 * j + 1] - xi[1],
                                          (double)pos4[4 * j + 2] - xi[2]};
                    const double rho2 = dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2] + eps2;
                    const double rho = std::sqrt(rho2);
                    const double mj = (double)pos4[4 * j + 3];
                    phi -= mj / rho;
                    const double f = mj / (rho2 * rho);
                    a[0] += f * dr[0]; a[1] += f * dr[1]; a[2] += f * dr[2];
                }
            }
            for (int64_t c : cells_acc) {
                const float* m = mom32 + 10 * c;
                const double M = m[0];
                const double dr[3] = {(double)m[1] - xi[0], (double)m[2] - xi[1], (double)m[3] - xi[2]};
                const double Qxx = m[4], Qyy = m[5], Qzz = m[6], Qxy = m[7], Qxz = m[8], Qyz = m[9];
                const double rho2 = dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2] + eps2;
                const double rho = std::sqrt(rho2);
                const double i1 = 1.0 / rho, i2 = i1 * i1, i3 = i1 * i2, i5 = i3 * i2, i7 = i5 * i2;
                const double T = Qxx + Qyy + Qzz;
                const double q[3] = {Qxx * dr[0] + Qxy * dr[1] + Qxz * dr[2],
                                     Qxy * dr[0] + Qyy * dr[1] + Qyz * dr[2],
                                     Qxz * dr[0] + Qyz * dr[1] + Qzz * dr[2]};
                const double w = dr[0] * q[0] + dr[1] * q[1] + dr[2] * q[2];
                phi += -M * i1 + 0.5 * T * i3 - 1.5 * w * i5;
                const double br = M * i3 - 1.5 * T * i5 + 7.5 * w * i7;
                for (int k = 0; k < 3; ++k) a[k] += dr[k] * br - 3.0 * q[k] * i5;
            }
            accpot[4 * i + 0] = a[0]; accpot[4 * i + 1] = a[1]; accpot[4 * i + 2] = a[2]; accpot[4 * i + 3] = phi;
        }
    }
}

// O(N^2) binary64 softened direct sum (L131: the theta -> 0 limit; L200: the accuracy reference).
// Targets [t0, t1).  accpot: double[n][4].
void orc_direct(int64_t n, const float* pos4, float eps, int64_t t0, int64_t t1, double* accpot) {
    const double eps2 = (double)eps * (double)eps;
#pragma omp parallel for schedule(static)
    for (int64_t i = t0; i < t1; ++i) {
        const double xi[3] = {(double)pos4[4 * i], (double)pos4[4 * i + 1], (double)pos4[4 * i + 2]};
        double a[3] = {0, 0, 0}, phi = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const double dr[3] = {(double)pos4[4 * j] - xi[0], (double)pos4[4 * j + 1] - xi[1],
                                  (double)pos4[4 * j + 2] - xi[2]};
            const double rho2 = dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2] + eps2;
            const double rho = std::sqrt(rho2);
            const double mj = (double)pos4[4 * j + 3];
            phi -= mj / rho;
            const double f = mj / (rho2 * rho);
            a[0] += f * dr[0]; a[1] += f * dr[1]; a[2] += f * dr[2];
        }
        accpot[4 * i + 0] = a[0]; accpot[4 * i + 1] = a[1]; accpot[4 * i + 2] = a[2]; accpot[4 * i + 3] = phi;
    }
}

// O11 (L105; A21), float: kick v = fmaf(a, h, v); drift x = fmaf(v, dt, x).  acc4: float[n][4] (ax, ay, az, phi).
void orc_kick(int64_t n, float* vel4, const float* acc4, float h) {
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < 3; ++k) vel4[4 * i + k] = fmaf(acc4[4 * i + k], h, vel4[4 * i + k]);
}
void orc_drift(int64_t n, float* pos4, const float* vel4, float dt) {
    for (int64_t i = 0; i < n; ++i)
        for (int k = 0; k < 3; ++k) pos4[4 * i + k] = fmaf(vel4[4 * i + k], dt, pos4[4 * i + k]);
}

// ---------------------------------------------------------------------------------------------
// Block time-steps (L45, L101 "time-step calculation ... on the GPU", L105 "... or on a subset of particles in case of
// the block-time step regime", L264-266).  The paper names the ingredients and leaves the criterion open; reading A29
// (DESIGN.md):  every particle i carries (x_i, v_i, a_i) at its own time t_i = tick_i * dt_max / 2^R and a step
// dt_i = dt_max / 2^rung_i (a power-of-two fraction, so times stay commensurate).  One system step goes to
// t_next = min_i (t_i + dt_i); the ACTIVE particles are those with t_i + dt_i = t_next.  Only they are predicted
// (x_i += v_i dt_i + a_i dt_i^2 / 2, the leapfrog predictor of Hut et al. that L105 cites) and, after the accelerations
// of the groups that hold them have been recomputed (moments refreshed on the existing cells, L266), corrected
// (v_i += (a_i + a_new) dt_i / 2, "the velocities are corrected"); inactive particles stay where they were last updated.
// All in float, single operations as written.

// Time-step criterion (A29): tau = eta * sqrt(len / |a|), rung = the smallest r in [0, R] with dt_max / 2^r <= tau (R if
// none); a particle may only move to a longer step at a time that is a multiple of it: rung >= R - ctz(tick) for tick > 0.
// acc4: float[n][4]; only particles with active[i] != 0 get a new rung (active may be null: all).
void orc_rungs(int64_t n, const float* acc4, const uint8_t* active, float len, float eta, float dt_max, int32_t R,
               uint32_t tick, uint8_t* rung) {
    int lowest = 0;                                      // longest step the current time allows
    if (tick != 0) {
        int z = 0;
        while (((tick >> z) & 1u) == 0u) ++z;
        lowest = R - z < 0 ? 0 : R - z;
    }
    for (int64_t i = 0; i < n; ++i) {
        if (active && !active[i]) continue;
        const float ax = acc4[4 * i], ay = acc4[4 * i + 1], az = acc4[4 * i + 2];
        const float a2 = fmaf(az, az, fmaf(ay, ay, ax * ax));
        const float amag = sqrtf(a2);
        const float tau = eta * sqrtf(len / amag);       // |a| = 0: tau = +inf, the longest step
        int r = 0;
        while (r < R && !(ldexpf(dt_max, -r) <= tau)) ++r;
        rung[i] = (uint8_t)(r < lowest ? lowest : r);
    }
}

// tick_next = min_i (tick_i + 2^(R - rung_i)); active_i = (tick_i + 2^(R - rung_i) == tick_next).  Returns tick_next.
uint32_t orc_block_active(int64_t n, const uint32_t* tick, const uint8_t* rung, int32_t R, uint8_t* active) {
    uint32_t next = 0xFFFFFFFFu;
    for (int64_t i = 0; i < n; ++i) next = std::min<uint32_t>(next, tick[i] + (1u << (R - rung[i])));
    for (int64_t i = 0; i < n; ++i) active[i] = (tick[i] + (1u << (R - rung[i])) == next) ? 1 : 0;
    return next;
}

// Predictor of the active particles (L105): h = dt_max / 2^rung; x = fmaf(a, (0.5f * h) * h, fmaf(v, h, x)).
void orc_block_predict(int64_t n, float* pos4, const float* vel4, const float* acc4, const uint8_t* active, const uint8_t* rung,
                       float dt_max) {
    for (int64_t i = 0; i < n; ++i) {
        if (!active[i]) continue;
        const float h = ldexpf(dt_max, -(int)rung[i]);
        const float hh = (0.5f * h) * h;
        for (int k = 0; k < 3; ++k) pos4[4 * i + k] = fmaf(acc4[4 * i + k], hh, fmaf(vel4[4 * i + k], h, pos4[4 * i + k]));
    }
}

// Corrector of the active particles (L105): v = fmaf(a_old + a_new, 0.5f * h, v); the held acceleration (and potential)
// becomes the new one; tick_i = tick_next.
void orc_block_correct(int64_t n, float* vel4, float* accb4, const float* accnew4, const uint8_t* active, const uint8_t* rung,
                       float dt_max, uint32_t tick_next, uint32_t* tick) {
    for (int64_t i = 0; i < n; ++i) {
        if (!active[i]) continue;
        const float h = ldexpf(dt_max, -(int)rung[i]);
        const float hh = 0.5f * h;
        for (int k = 0; k < 3; ++k) vel4[4 * i + k] = fmaf(accb4[4 * i + k] + accnew4[4 * i + k], hh, vel4[4 * i + k]);
        for (int k = 0; k < 4; ++k) accb4[4 * i + k] = accnew4[4 * i + k];
        tick[i] = tick_next;
    }
}

}  // extern "C"
