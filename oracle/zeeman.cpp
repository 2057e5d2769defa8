// oracle/zeeman.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// Zeeman pattern of a line in LS coupling, computed once per run (Table 1
// PAPER.md:37-43 gives g_eff = 1.667 for 6301.5 A (5P2 - 5D2) and 2.500 for 6302.5 A (5P1 - 5D0);
// PAPER.md:351 "four contributions ... to each of the three Zeeman components" for 6301.5).
// Reading F8: shift of a component in Lorentz units = g_l M_l - g_u M_u (> 0 = red);
// kind by Delta M = M_u - M_l: +1 -> sigma_blue, 0 -> pi, -1 -> sigma_red; relative strengths are the
// standard dipole ones (Landi Degl'Innocenti & Landolfi 2004, Table 3.1), normalised to 1 per kind.
#include "oracle.hpp"
#include <cmath>

namespace orc {

double lande_g(double S, double L, double J) {
    if (J == 0.0) return 0.0;
    return 1.5 + (S * (S + 1.0) - L * (L + 1.0)) / (2.0 * J * (J + 1.0));
}

double g_eff(double gl, double Jl, double gu, double Ju) {
    return 0.5 * (gl + gu) + 0.25 * (gl - gu) * (Jl * (Jl + 1.0) - Ju * (Ju + 1.0));
}

static double strength(double Jl, double Ju, double Ml, int dM) {
    double J = Jl, M = Ml;
    int dJ = (int)std::lround(Ju - Jl);
    if (dJ == 0) {
        if (dM == 0) return M * M;
        if (dM == +1) return (J - M) * (J + M + 1.0);
        return (J + M) * (J - M + 1.0);
    } else if (dJ == 1) {
        if (dM == 0) return (J + 1.0) * (J + 1.0) - M * M;
        if (dM == +1) return (J + M + 1.0) * (J + M + 2.0);
        return (J - M + 1.0) * (J - M + 2.0);
    } else {
        if (dM == 0) return J * J - M * M;
        if (dM == +1) return (J - M) * (J - M - 1.0);
        return (J + M) * (J + M - 1.0);
    }
}

std::vector<Component> zeeman_pattern(double Sl, double Ll, double Jl, double Su, double Lu, double Ju) {
    double gl = lande_g(Sl, Ll, Jl), gu = lande_g(Su, Lu, Ju);
    std::vector<Component> out;
    for (int dM = -1; dM <= 1; ++dM) {            // dM = M_u - M_l
        std::vector<Component> k;
        double tot = 0.0;
        for (double Ml = -Jl; Ml <= Jl + 1e-9; Ml += 1.0) {
            double Mu = Ml + dM;
            if (std::fabs(Mu) > Ju + 1e-9) continue;
            double s = strength(Jl, Ju, Ml, dM);
            if (s <= 0.0) continue;                 // zero-strength components (e.g. M = 0 -> 0 for dJ = 0) are dropped
            Component c;
            c.shift = gl * Ml - gu * Mu;
            c.weight = s;
            c.kind = -dM;                           // dM = +1 -> sigma_blue (-1); dM = -1 -> sigma_red (+1)
            k.push_back(c);
            tot += s;
        }
        for (auto& c : k) { c.weight /= tot; out.push_back(c); }
    }
    return out;
}

std::vector<Component> zeeman_triplet(double geff) {
    return { Component{0.0, 1.0, 0}, Component{-geff, 1.0, -1}, Component{+geff, 1.0, +1} };
}

}  // namespace orc
