// oracle/faddeeva.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// w(z) = exp(-z^2) erfc(-iz) = (i/pi) * Integral exp(-t^2)/(z - t) dt  for Im z > 0.
// The paper evaluates H = Re w and F = Im w with the Hui, Armstrong & Wray (1978) rational
// approximation whose coefficient table is not printed; the oracle instead writes
// out the integral definition with the trapezoid rule, which for this integrand converges
// geometrically (Matta & Reichel 1971; Hunter & Regan 1972):
//
//   w(z) = (i h / pi) * sum_n exp(-(n h)^2) / (z - n h)
//          + [ 2 exp(-z^2) / (1 - exp(-2 pi i z / h))   if Im z < pi / h ]      (pole correction)
//          + O(exp(-pi^2 / h^2)).
//
// h = 0.5 gives a remainder of 7e-18; nodes n = -13..13 leave exp(-42) outside the sum.
// Valid for Im z > 0; documented for Im z >= 1e-3 (closer to the real axis the node term and the
// correction cancel and digits are lost when Re z sits on a node).
#include "oracle.hpp"
#include <cmath>

namespace orc {

cplx faddeeva(cplx z) {
    const double h = 0.5;
    const int nmax = 13;
    const cplx I(0.0, 1.0);
    cplx sum(0.0, 0.0);
    for (int n = -nmax; n <= nmax; ++n) {
        double t = n * h;
        sum += std::exp(-t * t) / (z - t);
    }
    cplx w = I * h / M_PI * sum;
    if (z.imag() < M_PI / h) {
        cplx e = std::exp(-2.0 * M_PI * I * z / h);
        w += 2.0 * std::exp(-z * z) / (1.0 - e);
    }
    return w;
}

}  // namespace orc
