// =====================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded fp64 CPU implementation of the per-step Barnes-Hut
// gravity pipeline of "Bonsai: A GPU Tree-Code" (arXiv 1204.2280; /root/reference/PAPER.md,
// cited below as P:Lnn).  It exists to define what the CUDA path in
// paper_1204_2280_b200/csrc must compute.  It shares NO code with that path, and only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call it.  The product path never routes through this file.
//
// The paper gives no formula, constant or layout (it defers them to a companion paper that
// is not available); every step below therefore follows the reading fixed in DESIGN.md
// ("Readings of the paper", R1..R21), which restates SURVEY.md section 8(c).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   oracle_box / oracle_keys   hand-worked keys (tests/golden/morton_keys.txt), decode.encode = id,
//                              monotonicity, prefix <=> same cell
//   oracle_sort                bijection, order, stability, numpy lexsort
//   oracle_tree                tiling / leaf / prefix invariants, hand cases (chains, octants)
//   oracle_groups              partition invariants, exact boxes
//   oracle_multipoles          brute-force numpy sums per cell, root = global sums, parallel-axis,
//                              closed forms (cube corners, dumbbell)
//   oracle_walk                theta = 0 equals oracle_direct; error falls with theta; mass
//                              conservation of every group's lists; two-body softened Newton;
//                              dumbbell far-field expansion; independent numpy p-c formula
//   oracle_direct              independent numpy O(N^2) sum; two-body closed form
//   acc/pot of the CUDA path vs oracle_walk: tolerance only (summation order is free) --
//   "parity unpinned" beyond the stated tolerance.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

constexpr int kMaxLevel = 30;  // R1: 30 bits per axis, 90-bit key (BASELINE.json north_star)

struct Key {
    uint32_t hi, mid, lo;  // levels 1-10, 11-20, 21-30; 30 bits each (R1)
};

inline bool key_less(const Key& a, const Key& b) {
    if (a.hi != b.hi) return a.hi < b.hi;
    if (a.mid != b.mid) return a.mid < b.mid;
    return a.lo < b.lo;
}

// Octal digit of the key at level L in 1..30 (most significant first); R2: 4*x + 2*y + z.
inline uint32_t key_digit(const Key& k, int L) {
    uint32_t w = (L <= 10) ? k.hi : (L <= 20) ? k.mid : k.lo;
    int within = (L - 1) % 10;  // 0 = most significant digit of the word
    return (w >> (3 * (9 - within))) & 7u;
}

inline Key load_key(const uint32_t* keys, uint32_t i) {
    return Key{keys[3 * i + 0], keys[3 * i + 1], keys[3 * i + 2]};
}

}  // namespace

extern "C" {

// -------------------------------------------------------------------------------------
// O1a  Bounding box -> root cube (R3).  P:L30 (Results): "Sorting of the particles along a
// Space Filling Curve (Morton (1966))" needs a root cube; the paper is silent on it.
// lo = per-axis minimum (fp32); ext = largest per-axis extent, evaluated in fp64 on the fp32
// values; side = smallest power of two STRICTLY greater than ext; ext = 0 -> side = 1.
// -------------------------------------------------------------------------------------
void oracle_box(const float* pos_mass, uint32_t n, float lo[3], double* side) {
    float mn[3], mx[3];
    for (int a = 0; a < 3; ++a) {
        mn[a] = std::numeric_limits<float>::infinity();
        mx[a] = -std::numeric_limits<float>::infinity();
    }
    for (uint32_t i = 0; i < n; ++i)
        for (int a = 0; a < 3; ++a) {
            float v = pos_mass[4 * i + a];
            if (v < mn[a]) mn[a] = v;
            if (v > mx[a]) mx[a] = v;
        }
    double ext = 0.0;
    for (int a = 0; a < 3; ++a) {
        lo[a] = mn[a];
        double e = (double)mx[a] - (double)mn[a];
        if (e > ext) ext = e;
    }
    if (ext == 0.0) {
        *side = 1.0;
    } else {
        int e;
        std::frexp(ext, &e);  // ext = f * 2^e, f in [0.5, 1)  =>  2^e > ext >= 2^(e-1)
        *side = std::ldexp(1.0, e);
    }
}

// -------------------------------------------------------------------------------------
// O1b  Morton keys (R1, R2, R4).  Per axis, in fp32, round-to-nearest, no contraction:
//   t = x - lo;  u = t * (2^30 / side)  (exact power-of-two scale);  i = trunc(u) clamped to
//   [0, 2^30-1].  Digit at level L = 4*bit(ix) + 2*bit(iy) + bit(iz) with bit index 30-L.
// keys: 3 u32 per particle {hi, mid, lo}.
// -------------------------------------------------------------------------------------
void oracle_keys(const float* pos_mass, uint32_t n, const float lo[3], double side, uint32_t* keys) {
    const float scale = (float)(1073741824.0 / side);
    for (uint32_t i = 0; i < n; ++i) {
        uint32_t q[3];
        for (int a = 0; a < 3; ++a) {
            volatile float t = pos_mass[4 * i + a] - lo[a];
            volatile float u = t * scale;
            float uu = u;
            int64_t v = (uu >= 0.0f) ? (int64_t)uu : 0;  // trunc; negatives cannot occur (x >= lo)
            if (v > 1073741823) v = 1073741823;
            q[a] = (uint32_t)v;
        }
        uint32_t w[3] = {0, 0, 0};
        for (int L = 1; L <= kMaxLevel; ++L) {
            int bit = kMaxLevel - L;
            uint32_t d = 4u * ((q[0] >> bit) & 1u) + 2u * ((q[1] >> bit) & 1u) + ((q[2] >> bit) & 1u);
            int word = (L - 1) / 10;
            w[word] = (w[word] << 3) | d;
        }
        keys[3 * i + 0] = w[0];
        keys[3 * i + 1] = w[1];
        keys[3 * i + 2] = w[2];
    }
}

// Inverse of the interleave: integer coordinates from a key (used by oracle_multipoles for the
// geometric cell centre, and by the tests for decode(encode) = id).
void oracle_decode_key(const uint32_t key[3], uint32_t q[3]) {
    Key k{key[0], key[1], key[2]};
    q[0] = q[1] = q[2] = 0;
    for (int L = 1; L <= kMaxLevel; ++L) {
        uint32_t d = key_digit(k, L);
        q[0] = (q[0] << 1) | ((d >> 2) & 1u);
        q[1] = (q[1] << 1) | ((d >> 1) & 1u);
        q[2] = (q[2] << 1) | (d & 1u);
    }
}

// -------------------------------------------------------------------------------------
// O2  Sort (R5): order by (key, load index) ascending = a stable sort by key.
// perm[i] = load index of the i-th sorted particle.   P:L30 "sorting".
// -------------------------------------------------------------------------------------
void oracle_sort(const uint32_t* keys, uint32_t n, uint32_t* perm) {
    for (uint32_t i = 0; i < n; ++i) perm[i] = i;
    std::stable_sort(perm, perm + n, [&](uint32_t a, uint32_t b) {
        return key_less(load_key(keys, a), load_key(keys, b));
    });
}

// -------------------------------------------------------------------------------------
// O3  Reorder ("moving"): sorted_x[i] = x[perm[i]] for the particle properties.
// -------------------------------------------------------------------------------------
void oracle_reorder(const float* pos_mass, const uint32_t* keys, const uint32_t* perm, uint32_t n,
                    float* sorted_pos_mass, uint32_t* sorted_keys) {
    for (uint32_t i = 0; i < n; ++i) {
        uint32_t j = perm[i];
        for (int c = 0; c < 4; ++c) sorted_pos_mass[4 * i + c] = pos_mass[4 * j + c];
        for (int c = 0; c < 3; ++c) sorted_keys[3 * i + c] = keys[3 * j + c];
    }
}

// -------------------------------------------------------------------------------------
// O4  Octree (R7).  P:L22 fn.1 "we use an octree data-structure"; "construction of the
// tree-datastructure".  Root = level 0 over [0, n).  A cell at level L over [b, e) is a LEAF iff
// e-b <= nleaf or L = 30; otherwise it has one child per distinct level-(L+1) digit in [b, e)
// (sparse, chains kept), in ascending digit order.  Numbering: breadth-first, so children are
// consecutive (first_child, n_child).  Leaves have n_child = 0, first_child = 0.
// level_offsets[L] = index of the first cell of level L, L = 0..30; level_offsets[31] = n_cells.
// Returns n_cells, or 0xFFFFFFFF if more than cap_cells would be needed.
// -------------------------------------------------------------------------------------
uint32_t oracle_tree(const uint32_t* sorted_keys, uint32_t n, uint32_t nleaf, uint32_t cap_cells,
                     uint32_t* level, uint32_t* first, uint32_t* count, uint32_t* first_child,
                     uint32_t* n_child, uint32_t* parent, uint32_t level_offsets[32]) {
    if (n == 0 || cap_cells == 0) return 0xFFFFFFFFu;
    uint32_t n_cells = 1;
    level[0] = 0; first[0] = 0; count[0] = n; parent[0] = 0xFFFFFFFFu;
    uint32_t lvl_begin = 0, lvl_end = 1;
    for (int L = 0; L <= kMaxLevel; ++L) {
        level_offsets[L] = lvl_begin;
        for (uint32_t c = lvl_begin; c < lvl_end; ++c) {
            first_child[c] = 0;
            n_child[c] = 0;
            if (count[c] <= nleaf || L == kMaxLevel) continue;  // leaf
            uint32_t b = first[c], e = first[c] + count[c];
            uint32_t run_start = b;
            first_child[c] = n_cells;
            for (uint32_t i = b + 1; i <= e; ++i) {
                bool boundary = (i == e) ||
                    key_digit(load_key(sorted_keys, i), L + 1) != key_digit(load_key(sorted_keys, i - 1), L + 1);
                if (!boundary) continue;
                if (n_cells >= cap_cells) return 0xFFFFFFFFu;
                level[n_cells] = (uint32_t)(L + 1);
                first[n_cells] = run_start;
                count[n_cells] = i - run_start;
                parent[n_cells] = c;
                ++n_cells;
                ++n_child[c];
                run_start = i;
            }
        }
        lvl_begin = lvl_end;
        lvl_end = n_cells;
    }
    level_offsets[31] = n_cells;
    return n_cells;
}

// -------------------------------------------------------------------------------------
// O5  Groups (R13).  P:L30: "the method used for tree-traversion on vector machines
// (Barnes 1990)": one shared traversal per group of neighbouring particles.
// active_sorted: NULL = all active, else u8[n] indexed by SORTED particle index.
// active_list[k] = sorted index of the k-th active particle (ascending); groups index into it.
//   mode 0 (tree-cell): cells with count <= ncrit whose parent has count > ncrit (the root if
//       n <= ncrit; a level-30 leaf may exceed ncrit), in key order; a group keeps only its active
//       members and is dropped if none remain.
//   mode 1 (sorted-chunk): consecutive runs of ncrit active particles (last one shorter).
//   mode 2 (cell-chunk): the "container" cells are the mode-0 cells at threshold group_cell (count <=
//       group_cell, parent count > group_cell; childless cells always qualify); the active members of each
//       container, in sorted order, are cut into consecutive runs of ncrit (last one shorter).  A group
//       therefore never straddles the boundary of a cell holding more than group_cell particles.
//       group_cell = ncrit gives mode 0 for every cell with <= ncrit particles, group_cell >= n gives mode 1.
// bmin/bmax: exact fp32 per-axis min/max over the group's members (3 floats per group each).
// Returns n_groups; *n_active_out = number of active particles.
// -------------------------------------------------------------------------------------
uint32_t oracle_groups(uint32_t mode, uint32_t ncrit, uint32_t group_cell, uint32_t n, const float* sorted_pos_mass,
                       uint32_t n_cells, const uint32_t* first, const uint32_t* count,
                       const uint32_t* first_child, const uint32_t* n_child,
                       const uint8_t* active_sorted, uint32_t* active_list, uint32_t* n_active_out,
                       uint32_t* gfirst, uint32_t* gcount, float* gbmin, float* gbmax) {
    std::vector<uint32_t> rank(n + 1);  // rank[i] = number of active particles with sorted index < i
    uint32_t na = 0;
    for (uint32_t i = 0; i < n; ++i) {
        rank[i] = na;
        if (!active_sorted || active_sorted[i]) active_list[na++] = i;
    }
    rank[n] = na;
    *n_active_out = na;
    uint32_t ng = 0;
    auto emit = [&](uint32_t f, uint32_t c) {
        if (c == 0) return;
        gfirst[ng] = f; gcount[ng] = c;
        for (int a = 0; a < 3; ++a) {
            float mn = std::numeric_limits<float>::infinity(), mx = -mn;
            for (uint32_t k = f; k < f + c; ++k) {
                float v = sorted_pos_mass[4 * active_list[k] + a];
                if (v < mn) mn = v;
                if (v > mx) mx = v;
            }
            gbmin[3 * ng + a] = mn; gbmax[3 * ng + a] = mx;
        }
        ++ng;
    };
    if (mode == 1) {
        for (uint32_t f = 0; f < na; f += ncrit) emit(f, std::min(ncrit, na - f));
    } else {
        // depth-first in key order: descend while count > ncrit and the cell has children
        std::vector<uint32_t> stack;
        stack.push_back(0);
        (void)n_cells;
        const uint32_t limit = (mode == 2) ? group_cell : ncrit;
        while (!stack.empty()) {
            uint32_t c = stack.back(); stack.pop_back();
            if (count[c] <= limit || n_child[c] == 0) {
                const uint32_t r0 = rank[first[c]], a = rank[first[c] + count[c]] - r0;
                if (mode == 2) {
                    for (uint32_t f = 0; f < a; f += ncrit) emit(r0 + f, std::min(ncrit, a - f));
                } else {
                    emit(r0, a);
                }
            } else {
                for (uint32_t k = n_child[c]; k-- > 0;) stack.push_back(first_child[c] + k);
            }
        }
    }
    return ng;
}

// -------------------------------------------------------------------------------------
// O6  Multipole moments (R8).  P:L20 "computation of the tree-properties (multipole moments)";
// BASELINE.json north_star: monopole + quadrupole.  For each cell, directly from its particle
// range, in fp64:  M = sum m;  COM = sum m x / M;  Q_ab = sum m (x_a-COM_a)(x_b-COM_b) in the order
// (xx, yy, zz, xy, xz, yz) -- raw second moments about the COM, not trace-free.
// Geometric centre g_a = lo_a + (c_a + 1/2) l, l = side / 2^L, c_a = the cell's integer coordinate
// (top L bits of the quantised coordinate);  delta = |COM - g|.  All stored rounded once to fp32.
// A cell whose mass is 0 takes COM = g and Q = 0.
// -------------------------------------------------------------------------------------
void oracle_multipoles(const float* sorted_pos_mass, const uint32_t* sorted_keys, uint32_t n,
                       const float lo[3], double side, uint32_t n_cells, const uint32_t* level,
                       const uint32_t* first, const uint32_t* count, float* com_m, float* quad,
                       float* delta, float* lside) {
    (void)n;
    for (uint32_t c = 0; c < n_cells; ++c) {
        uint32_t b = first[c], e = first[c] + count[c];
        int L = (int)level[c];
        double l = std::ldexp(side, -L);
        uint32_t q[3];
        oracle_decode_key(&sorted_keys[3 * b], q);
        double g[3];
        for (int a = 0; a < 3; ++a) {
            uint32_t ca = (L == 0) ? 0u : (q[a] >> (kMaxLevel - L));
            g[a] = (double)lo[a] + ((double)ca + 0.5) * l;
        }
        double M = 0.0, S[3] = {0, 0, 0};
        for (uint32_t i = b; i < e; ++i) {
            double m = sorted_pos_mass[4 * i + 3];
            M += m;
            for (int a = 0; a < 3; ++a) S[a] += m * (double)sorted_pos_mass[4 * i + a];
        }
        double com[3];
        for (int a = 0; a < 3; ++a) com[a] = (M > 0.0) ? S[a] / M : g[a];
        double Q[6] = {0, 0, 0, 0, 0, 0};
        if (M > 0.0)
            for (uint32_t i = b; i < e; ++i) {
                double m = sorted_pos_mass[4 * i + 3];
                double dx = (double)sorted_pos_mass[4 * i + 0] - com[0];
                double dy = (double)sorted_pos_mass[4 * i + 1] - com[1];
                double dz = (double)sorted_pos_mass[4 * i + 2] - com[2];
                Q[0] += m * dx * dx; Q[1] += m * dy * dy; Q[2] += m * dz * dz;
                Q[3] += m * dx * dy; Q[4] += m * dx * dz; Q[5] += m * dy * dz;
            }
        double d2 = 0.0;
        for (int a = 0; a < 3; ++a) d2 += (com[a] - g[a]) * (com[a] - g[a]);
        for (int a = 0; a < 3; ++a) com_m[4 * c + a] = (float)com[a];
        com_m[4 * c + 3] = (float)M;
        for (int k = 0; k < 6; ++k) quad[6 * c + k] = (float)Q[k];
        delta[c] = (float)std::sqrt(d2);
        lside[c] = (float)l;
    }
}

// -------------------------------------------------------------------------------------
// O7  Tree walk (R9, R10, R11, R12, R14, R19).  P:L30: MAC = "a combination of the method introduced
// by Barnes (1994) and the method used for tree-traversion on vector machines (Barnes 1990)";
// "particle-cell interactions", "particle-particle", theta = 0.75.
//
// For each selected group G (sel = NULL: all), depth-first from the root.  For cell c -- the MAC is
// DEFINED in fp32, each operation rounded to nearest, in exactly this order:
//   d_a = max(0, max(bmin_a - COM_a, COM_a - bmax_a));  d2 = fma(dz,dz, fma(dy,dy, dx*dx));
//   rc = fma(l, inv_theta, delta), inv_theta = 1.0f / theta;  rc2 = rc*rc;  accept iff d2 > rc2.
// accepted -> p-c list;  rejected leaf -> p-p list;  rejected internal -> visit children.
// Every active particle i of G then sums, in fp64 with e2 = eps^2:
//   p-p (j != i by sorted index): dr = x_j - x_i; r2 = |dr|^2 + e2; pot -= m_j r^-1; acc += m_j r^-3 dr
//   p-c: dr = COM - x_i; r2 = |dr|^2 + e2; tr = Qxx+Qyy+Qzz; Qr = Q dr; q = dr.Qr;
//        pot -= M r^-1 - 1/2 tr r^-3 + 3/2 q r^-5
//        acc += dr (M r^-3 - 3/2 tr r^-5 + 15/2 q r^-7) - 3 r^-5 Qr
// Outputs are indexed by SORTED particle index (only entries of walked particles are written):
//   acc[3*i..], pot[i], n_pp[i] = (sum of leaf counts in G's p-p list) - 1, n_pc[i] = |p-c list|.
// order = 1 (R29): a p-c term is  pot -= M r^-1;  acc += M r^-3 dr  only.
// Per selected group k (position in sel): g_ntests[k] = number of MAC tests; g_borderline[k] = 1 if
// any test had |d2 - rc2| <= 1e-5 rc2 (fp64 on the fp32 inputs).
// -------------------------------------------------------------------------------------
void oracle_walk(float theta, float eps, const float* sorted_pos_mass, uint32_t n,
                 const uint32_t* first, const uint32_t* count, const uint32_t* first_child,
                 const uint32_t* n_child, const float* com_m, const float* quad, const float* delta,
                 const float* lside, const uint32_t* active_list, const uint32_t* gfirst,
                 const uint32_t* gcount, const float* gbmin, const float* gbmax, uint32_t n_sel,
                 const uint32_t* sel, double* acc, double* pot, uint32_t* n_pp, uint32_t* n_pc,
                 uint32_t* g_ntests, uint8_t* g_borderline, uint32_t order) {
    // order: 1 = accepted cells act as monopoles only (R29, oracle/mac_oracle.cpp); anything else = monopole +
    // quadrupole (R8, the default).
    (void)n;
    volatile float inv_theta_v = 1.0f / theta;
    const float inv_theta = inv_theta_v;
    const double e2 = (double)eps * (double)eps;
    std::vector<uint32_t> stack, pc, pp;
    for (uint32_t s = 0; s < n_sel; ++s) {
        uint32_t G = sel ? sel[s] : s;
        const float* bmin = &gbmin[3 * G];
        const float* bmax = &gbmax[3 * G];
        pc.clear(); pp.clear(); stack.clear();
        stack.push_back(0);
        uint32_t ntests = 0;
        bool borderline = false;
        while (!stack.empty()) {
            uint32_t c = stack.back(); stack.pop_back();
            ++ntests;
            float d[3];
            for (int a = 0; a < 3; ++a) {
                float com = com_m[4 * c + a];
                volatile float below = bmin[a] - com;
                volatile float above = com - bmax[a];
                float m = std::fmax((float)below, (float)above);
                d[a] = std::fmax(0.0f, m);
            }
            volatile float xx = d[0] * d[0];
            float d2 = std::fmaf(d[2], d[2], std::fmaf(d[1], d[1], (float)xx));
            float rc = std::fmaf(lside[c], inv_theta, delta[c]);
            volatile float rc2v = rc * rc;
            float rc2 = rc2v;
            bool accept = d2 > rc2;
            if (std::fabs((double)d2 - (double)rc2) <= 1e-5 * (double)rc2) borderline = true;
            if (accept) {
                pc.push_back(c);
            } else if (n_child[c] == 0) {
                pp.push_back(c);
            } else {
                for (uint32_t k = n_child[c]; k-- > 0;) stack.push_back(first_child[c] + k);
            }
        }
        if (g_ntests) g_ntests[s] = ntests;
        if (g_borderline) g_borderline[s] = borderline ? 1 : 0;
        uint32_t npp_total = 0;
        for (uint32_t c : pp) npp_total += count[c];
        for (uint32_t k = gfirst[G]; k < gfirst[G] + gcount[G]; ++k) {
            uint32_t i = active_list[k];
            double xi = sorted_pos_mass[4 * i + 0], yi = sorted_pos_mass[4 * i + 1], zi = sorted_pos_mass[4 * i + 2];
            double ax = 0, ay = 0, az = 0, ph = 0;
            for (uint32_t c : pp)
                for (uint32_t j = first[c]; j < first[c] + count[c]; ++j) {
                    if (j == i) continue;
                    double dx = (double)sorted_pos_mass[4 * j + 0] - xi;
                    double dy = (double)sorted_pos_mass[4 * j + 1] - yi;
                    double dz = (double)sorted_pos_mass[4 * j + 2] - zi;
                    double m = sorted_pos_mass[4 * j + 3];
                    double r2 = dx * dx + dy * dy + dz * dz + e2;
                    double rinv = 1.0 / std::sqrt(r2);
                    double rinv3 = rinv * rinv * rinv;
                    ph -= m * rinv;
                    ax += m * rinv3 * dx; ay += m * rinv3 * dy; az += m * rinv3 * dz;
                }
            for (uint32_t c : pc) {
                double dx = (double)com_m[4 * c + 0] - xi;
                double dy = (double)com_m[4 * c + 1] - yi;
                double dz = (double)com_m[4 * c + 2] - zi;
                double M = com_m[4 * c + 3];
                if (order == 1) {
                    double r2 = dx * dx + dy * dy + dz * dz + e2;
                    double rinv = 1.0 / std::sqrt(r2);
                    double rinv3 = rinv * rinv * rinv;
                    ph -= M * rinv;
                    ax += M * rinv3 * dx; ay += M * rinv3 * dy; az += M * rinv3 * dz;
                    continue;
                }
                double Qxx = quad[6 * c + 0], Qyy = quad[6 * c + 1], Qzz = quad[6 * c + 2];
                double Qxy = quad[6 * c + 3], Qxz = quad[6 * c + 4], Qyz = quad[6 * c + 5];
                double r2 = dx * dx + dy * dy + dz * dz + e2;
                double rinv = 1.0 / std::sqrt(r2);
                double rinv2 = rinv * rinv;
                double rinv3 = rinv * rinv2, rinv5 = rinv3 * rinv2, rinv7 = rinv5 * rinv2;
                double tr = Qxx + Qyy + Qzz;
                double Qrx = Qxx * dx + Qxy * dy + Qxz * dz;
                double Qry = Qxy * dx + Qyy * dy + Qyz * dz;
                double Qrz = Qxz * dx + Qyz * dy + Qzz * dz;
                double q = dx * Qrx + dy * Qry + dz * Qrz;
                ph -= M * rinv - 0.5 * tr * rinv3 + 1.5 * q * rinv5;
                double f = M * rinv3 - 1.5 * tr * rinv5 + 7.5 * q * rinv7;
                ax += dx * f - 3.0 * rinv5 * Qrx;
                ay += dy * f - 3.0 * rinv5 * Qry;
                az += dz * f - 3.0 * rinv5 * Qrz;
            }
            acc[3 * i + 0] = ax; acc[3 * i + 1] = ay; acc[3 * i + 2] = az;
            pot[i] = ph;
            n_pp[i] = npp_total - 1;
            n_pc[i] = (uint32_t)pc.size();
        }
    }
}

// Lists of one group (for the mass-conservation pin and for debugging): returns the number of
// accepted cells / opened leaves and writes up to cap ids of each.
void oracle_walk_lists(float theta, const uint32_t* first_child, const uint32_t* n_child,
                       const float* com_m, const float* delta, const float* lside, const float bmin[3],
                       const float bmax[3], uint32_t cap, uint32_t* pc_ids, uint32_t* n_pc_out,
                       uint32_t* pp_ids, uint32_t* n_pp_out) {
    volatile float inv_theta_v = 1.0f / theta;
    const float inv_theta = inv_theta_v;
    std::vector<uint32_t> stack;
    stack.push_back(0);
    uint32_t npc = 0, npp = 0;
    while (!stack.empty()) {
        uint32_t c = stack.back(); stack.pop_back();
        float d[3];
        for (int a = 0; a < 3; ++a) {
            float com = com_m[4 * c + a];
            volatile float below = bmin[a] - com;
            volatile float above = com - bmax[a];
            d[a] = std::fmax(0.0f, std::fmax((float)below, (float)above));
        }
        volatile float xx = d[0] * d[0];
        float d2 = std::fmaf(d[2], d[2], std::fmaf(d[1], d[1], (float)xx));
        float rc = std::fmaf(lside[c], inv_theta, delta[c]);
        volatile float rc2 = rc * rc;
        if (d2 > (float)rc2) {
            if (npc < cap) pc_ids[npc] = c;
            ++npc;
        } else if (n_child[c] == 0) {
            if (npp < cap) pp_ids[npp] = c;
            ++npp;
        } else {
            for (uint32_t k = n_child[c]; k-- > 0;) stack.push_back(first_child[c] + k);
        }
    }
    *n_pc_out = npc;
    *n_pp_out = npp;
}

// -------------------------------------------------------------------------------------
// O8  Direct summation (ground truth; "brute force methods").  For each sink s (an index
// into pos_mass), over ALL j != s:  pot = -sum m_j (|x_j-x_s|^2 + eps^2)^-1/2,  acc likewise.  fp64.
// -------------------------------------------------------------------------------------
void oracle_direct(const float* pos_mass, uint32_t n, float eps, uint32_t n_sinks,
                   const uint32_t* sinks, double* acc, double* pot) {
    const double e2 = (double)eps * (double)eps;
    for (uint32_t s = 0; s < n_sinks; ++s) {
        uint32_t i = sinks ? sinks[s] : s;
        double xi = pos_mass[4 * i + 0], yi = pos_mass[4 * i + 1], zi = pos_mass[4 * i + 2];
        double ax = 0, ay = 0, az = 0, ph = 0;
        for (uint32_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = (double)pos_mass[4 * j + 0] - xi;
            double dy = (double)pos_mass[4 * j + 1] - yi;
            double dz = (double)pos_mass[4 * j + 2] - zi;
            double m = pos_mass[4 * j + 3];
            double r2 = dx * dx + dy * dy + dz * dz + e2;
            double rinv = 1.0 / std::sqrt(r2);
            double rinv3 = rinv * rinv * rinv;
            ph -= m * rinv;
            ax += m * rinv3 * dx; ay += m * rinv3 * dy; az += m * rinv3 * dz;
        }
        acc[3 * s + 0] = ax; acc[3 * s + 1] = ay; acc[3 * s + 2] = az;
        pot[s] = ph;
    }
}

}  // extern "C"
