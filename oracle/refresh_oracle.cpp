// =====================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY (see bonsai_oracle.cpp for the rules that apply).
//
// Row f1 of DESIGN.md section 0: re-using the sorted order and the tree after the particles have moved.
// P:L52 (Discussion): sorting, moving and tree-construction "do not have to be executed during each time-step
// when using the block time-step method.  It is sufficient to only recompute the multipole moments of tree-cells
// that have updated child particles, and only when the tree-traverse shows a considerable decline in performance
// does the complete tree-structure has to be rebuild.  This decline is the result of ... an increase of the average
// number of particle-cell and particle-particle interactions.  This quantity increases because the tree-cell size
// increases, which causes more cells to be opened by the MAC."  No formula is given.  Reading taken (R25):
//
//   R25  A refreshed tree keeps the permutation, the keys, the cells and their links, the geometric centres g and
//        the group membership of the last full build.  The particles are re-gathered through the old permutation,
//        group boxes and multipoles (R8) are recomputed from the new positions, and the cell size that enters the
//        opening test (R9) grows so that the cell still contains its members:
//            l' = max( l,  2 max_i max_a |x_ia - g_a| )      (fp64, rounded once to fp32),
//        l = side / 2^L the geometric side.  delta = |COM - g| as before.  With no motion l' = l except where the
//        fp32 quantisation of R4 placed a particle a rounding error outside its nominal cell.
//
// This file only supplies l'; everything else of a refreshed step is the unchanged oracle applied to the
// re-gathered positions (oracle/__init__.py: refresh()).
//
// Pins (tests/test_oracle_refresh.py): every member lies inside the cube of side l' about g and l' is minimal
// (numpy brute force); zero motion reproduces the fresh build; theta = 0 on a refreshed tree equals direct
// summation at the new positions; the force error against direct summation stays of the order of a fresh tree's
// while the interaction count grows with the drift (the paper's stated behaviour).
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>

extern "C" {

void oracle_decode_key(const uint32_t key[3], uint32_t q[3]);  // bonsai_oracle.cpp (R1, R2)

// lside[c] <- (float) max(side / 2^L, 2 max_i max_a |x_ia - g_a|) over the cell's particle range, g as in O6.
void oracle_extent_side(const float* sorted_pos_mass, const uint32_t* sorted_keys, const float lo[3], double side,
                        uint32_t n_cells, const uint32_t* level, const uint32_t* first, const uint32_t* count,
                        float* lside) {
    const int kMaxLevel = 30;
    for (uint32_t c = 0; c < n_cells; ++c) {
        const uint32_t b = first[c], e = first[c] + count[c];
        const int L = (int)level[c];
        const double l = std::ldexp(side, -L);
        uint32_t q[3];
        oracle_decode_key(&sorted_keys[3 * b], q);
        double ext = 0.0;
        for (int a = 0; a < 3; ++a) {
            const uint32_t ca = (L == 0) ? 0u : (q[a] >> (kMaxLevel - L));
            const double g = (double)lo[a] + ((double)ca + 0.5) * l;
            for (uint32_t i = b; i < e; ++i) ext = std::max(ext, std::fabs((double)sorted_pos_mass[4 * i + a] - g));
        }
        lside[c] = (float)std::max(l, 2.0 * ext);
    }
}

}  // extern "C"
