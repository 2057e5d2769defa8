// oracle/sobol.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// Sobol' quasi-random sequence, generated the way Bratley & Fox (1988, ACM TOMS Algorithm 659) do it, which is what the
// paper uses for the initial population and for restarts: direction numbers v_i = m_i 2^(32-i) from
// a primitive polynomial per dimension and the recurrence
//     m_i = 2 a_1 m_(i-1) xor 2^2 a_2 m_(i-2) xor ... xor 2^(s-1) a_(s-1) m_(i-s+1) xor 2^s m_(i-s) xor m_(i-s),
// points in Gray-code order (Antonov & Saleev): x_n = xor of v_(b+1) over the set bits b of n xor (n >> 1).
// The initial m_i are those of Joe & Kuo's table (the first 11 dimensions; reading V1 of DESIGN.md: the paper does
// not say which initial numbers it took).  Pinned against scipy.stats.qmc.Sobol in tests/test_oracle_ga_binary.py.
#include "oracle.hpp"

namespace orc {

namespace {
struct Dim { int s; unsigned a; unsigned m[5]; };
// dimension 1 is the van der Corput sequence (all m_i = 1); dimensions 2..11:
const Dim DIMS[10] = {
    { 1, 0, { 1, 0, 0, 0, 0 } },  { 2, 1, { 1, 3, 0, 0, 0 } },  { 3, 1, { 1, 3, 1, 0, 0 } },  { 3, 2, { 1, 1, 1, 0, 0 } },
    { 4, 1, { 1, 1, 3, 3, 0 } },  { 4, 4, { 1, 3, 5, 13, 0 } }, { 5, 2, { 1, 1, 5, 5, 17 } }, { 5, 4, { 1, 1, 5, 5, 5 } },
    { 5, 7, { 1, 1, 7, 11, 19 } }, { 5, 11, { 1, 1, 5, 1, 1 } } };
}  // namespace

void sobol_directions(int dim, uint32_t v[32]) {
    if (dim == 0) { for (int i = 1; i <= 32; ++i) v[i - 1] = 1u << (32 - i); return; }
    const Dim& d = DIMS[dim - 1];
    uint32_t m[33];
    for (int i = 1; i <= 32; ++i) {
        if (i <= d.s) { m[i] = d.m[i - 1]; continue; }
        uint32_t x = m[i - d.s] ^ (m[i - d.s] << d.s);
        for (int k = 1; k < d.s; ++k)
            if ((d.a >> (d.s - 1 - k)) & 1u) x ^= m[i - k] << k;
        m[i] = x;
    }
    for (int i = 1; i <= 32; ++i) v[i - 1] = m[i] << (32 - i);
}

uint32_t sobol_point(uint32_t n, int dim) {
    uint32_t v[32];
    sobol_directions(dim, v);
    uint32_t g = n ^ (n >> 1), x = 0;
    for (int b = 0; b < 32; ++b) if ((g >> b) & 1u) x ^= v[b];
    return x;
}

}  // namespace orc
