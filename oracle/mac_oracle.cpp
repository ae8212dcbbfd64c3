// =====================================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY (see bonsai_oracle.cpp for the rules that apply).
//
// Row f3 of DESIGN.md section 0: variants of the multipole acceptance criterion.  P:L30 (Results): "the multipole
// acceptance critera (MAC) (theta) which sets the trade-off between speed and accuracy"; the MAC itself is "a
// combination of the method introduced by Barnes (1994) and the method used for tree-traversion on vector machines
// (Barnes (1990))" -- no formula.  R9 reads it as  d > l / theta + delta  with l the GEOMETRIC side of the cell and
// delta the distance of the centre of mass from the GEOMETRIC centre.  SURVEY.md section 8(c) A9b leaves the other
// natural reading for this row:
//
//   R28  tight MAC (mac_mode = 1): the cell's size and centre are those of the exact bounding box of its particles,
//            bmin_a = min_i x_ia,  bmax_a = max_i x_ia              (fp32 values, exact),
//            l_t   = max_a (bmax_a - bmin_a)                        (fp64, rounded once to fp32),
//            c_t   = (bmin + bmax) / 2                              (fp64),
//            delta_t = |COM - c_t|                                  (fp64 COM of O6, rounded once to fp32),
//        and the opening test is R9 unchanged with (l_t, delta_t) in place of (l, delta).  A cell with one particle
//        (or coincident particles) has l_t = delta_t = 0 and is accepted from any distance > 0 -- exact, its
//        quadrupole vanishes.  A cell that contains a sink still has d <= |x - COM| <= (sqrt(3)/2) l_t + delta_t, so
//        the bound theta < 2/sqrt(3) of R9/R11 carries over.
//   R29  monopole-only walk (order = 1): accepted cells act through M and COM alone,
//            phi_i -= M r^-1,   a_i += M r^-3 dr,   r^2 = |dr|^2 + eps^2;
//        lists, counts and the p-p part are unchanged (implemented in oracle_walk, bonsai_oracle.cpp).
//
// This file supplies (l_t, delta_t); everything else is the unchanged oracle.
//
// Pins (tests/test_oracle_mac.py): every member inside the box and the box minimal (numpy brute force); l_t <= l
// (up to the rounding of the key quantisation R4) -- so at equal theta the tight MAC accepts a superset of cells;
// theta = 0 is direct summation for both MACs and both orders; a monopole p-c term converges as (s/d)^2 where
// the quadrupole term converges as (s/d)^3; mass accounting of the lists; error against direct summation falls
// monotonically with theta for every variant.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>

extern "C" {

// For every cell c over the sorted particle range [first, first + count):
//   lside[c] <- (float) l_t,  delta[c] <- (float) delta_t,  box[6c..6c+5] <- bmin xyz, bmax xyz (may be NULL).
void oracle_tight_mac(const float* sorted_pos_mass, uint32_t n_cells, const uint32_t* first, const uint32_t* count,
                      float* lside, float* delta, float* box) {
    for (uint32_t c = 0; c < n_cells; ++c) {
        const uint32_t b = first[c], e = first[c] + count[c];
        float mn[3], mx[3];
        for (int a = 0; a < 3; ++a) mn[a] = mx[a] = sorted_pos_mass[4 * b + a];
        double M = 0.0, S[3] = {0, 0, 0};
        for (uint32_t i = b; i < e; ++i) {
            const double m = sorted_pos_mass[4 * i + 3];
            M += m;
            for (int a = 0; a < 3; ++a) {
                const float x = sorted_pos_mass[4 * i + a];
                mn[a] = std::min(mn[a], x);
                mx[a] = std::max(mx[a], x);
                S[a] += m * (double)x;  // the same sums, in the same order, as O6 (oracle_multipoles)
            }
        }
        double l = 0.0, d2 = 0.0;
        for (int a = 0; a < 3; ++a) {
            l = std::max(l, (double)mx[a] - (double)mn[a]);
            const double centre = 0.5 * ((double)mn[a] + (double)mx[a]);
            const double com = (M > 0.0) ? S[a] / M : centre;  // massless cell: COM := centre (cf. O6)
            d2 += (com - centre) * (com - centre);
        }
        lside[c] = (float)l;
        delta[c] = (float)std::sqrt(d2);
        if (box)
            for (int a = 0; a < 3; ++a) {
                box[6 * c + a] = mn[a];
                box[6 * c + 3 + a] = mx[a];
            }
    }
}

}  // extern "C"
