// oracle/ga.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// The per-pixel genetic algorithm, Alg. 1 of the paper: create P0, evaluate; then
// per generation select (S), recombine (R), mutate (M),
// decode (eq. 4-5) and evaluate (F = eq. 16).  The paper leaves the operators' details
// open; BASELINE.json's north_star fixes them as tournament selection, arithmetic crossover, bounded
// mutation and elitism with a counter-based Philox stream, and DESIGN.md readings G0-G5 fix every
// remaining choice.  Discrete state (genes) is binary32 and every gene operation below is a single
// IEEE binary32 operation (or one fmaf), so that an independent implementation can match it bit for bit;
// the fitness is double here.
#include "oracle.hpp"
#include <cmath>
#include <algorithm>
#include <limits>
#include <vector>

namespace orc {

// G0: uniform in [0,1) from the top 24 bits: exact in binary32.
static inline float u01(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }
// G0: integer in [0, n) from the top 24 bits, in integer arithmetic: floor(u * n).
static inline int below(uint32_t x, int n) { return (int)(((uint64_t)(x >> 8) * (uint64_t)n) >> 24); }

static void draw(const GaCfg& c, uint64_t pixel, int t, int i, int k, uint32_t out[4]) {
    uint32_t ctr[4] = { (uint32_t)pixel, (uint32_t)t, (uint32_t)i, (uint32_t)k };
    uint32_t key[2] = { (uint32_t)(c.seed & 0xffffffffu), (uint32_t)(c.seed >> 32) };
    philox4x32_10(ctr, key, out);
}

// V0 / eq. 5: a 16-bit code k decodes to g = k / (2^N - 1); the real-coded variant holds g itself.  The result is
// rounded to binary32 so that both implementations feed the same gene value to the box mapping.
float gene_value(float stored, const GaCfg& c) { return c.variant == 1 ? stored / 65535.0f : stored; }   // one IEEE binary32 division

// G1: gene in [0,1] -> physical parameter, from the binary32 gene, in double.
double decode_gene(float g, double lo, double hi, int log_scale) {
    if (log_scale) return lo * std::pow(hi / lo, (double)g);
    return lo + (hi - lo) * (double)g;
}

// ---------------------------------------------------------------------------------------------------------
// Variant 1: the paper's own binary-coded GA (readings V0-V5 of DESIGN.md).
//   V0  genotype: one 16-bit unsigned code k per parameter, held here as an integer-valued float;
//       decode (eq. 5): g = k / (2^16 - 1), then the box mapping of reading G1.
//   V1  initial population: individual i = Sobol' point number i + 1 in M dimensions, top 16 bits per
//       dimension, xor a per-pixel digital shift (16 bits per dimension from Philox block (pixel, 0, 2^32-1, j/4)).
//   V2  restart: every N_samp = max(1, G/4) generations (t mod N_samp = 0, t < G) the worst floor(P/2)
//       members of generation t-1 (rank by chi2, ties by index) are dead: tournaments draw among the live ranks only
//       and the last floor(P/2) slots of generation t are the NEXT Sobol' points of the same shifted sequence.
//   V3  selection: the k-way tournament of reading G3.
//   V4  recombination: children come in pairs (2q-1, 2q) keyed by the odd index; parents A, B from
//       blocks 0, 1; block 2: u0 < p_cross ? one-point crossover at bit cut = 1 + floor(u1 (16 M - 1)) of the M x 16
//       bit string (gene 0 first, bit 0 = MSB) : copies; the odd child takes head(A) + tail(B), the even
//       child head(B) + tail(A).
//   V5  mutation ("less-significant bits more frequently"): gene j of child i, words (x_m, x_d) of
//       block 3 + j/2: if u(x_m) < p_mut flip the bits of ((x_d & 0xffff) & (x_d >> 16)) >> (x_m & 15), so that bit b
//       (0 = LSB) flips with probability (16 - b) / 64.
// ---------------------------------------------------------------------------------------------------------
static uint32_t digital_shift(const GaCfg& c, uint64_t pixel, int j) {
    uint32_t r[4];
    draw(c, pixel, 0, (int)0xFFFFFFFFu, j / 4, r);
    return r[j % 4] >> 16;
}

static float sobol_gene(const GaCfg& c, uint64_t pixel, uint32_t n, int j) {
    return (float)(((sobol_point(n, j) >> 16) ^ digital_shift(c, pixel, j)) & 0xFFFFu);
}

static void ga_init_binary(uint64_t pixel, const GaCfg& c, float* genes) {
    for (int i = 0; i < c.pop; ++i)
        for (int j = 0; j < c.npar; ++j) genes[i * c.npar + j] = sobol_gene(c, pixel, (uint32_t)i + 1u, j);
}

static void ga_step_binary(const float* genes, const double* chi2v, int t, uint64_t pixel, const GaCfg& c, float* out) {
    const int M = c.npar, P = c.pop;
    const int n_samp = c.generations / 4 > 1 ? c.generations / 4 : 1;
    const bool restart = (t % n_samp == 0) && t < c.generations;
    const int n_dead = restart ? P / 2 : 0, n_live = P - n_dead;
    std::vector<int> order(P);                                           // order[r] = index of the r-th best
    for (int i = 0; i < P; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return chi2v[a] < chi2v[b]; });
    for (int j = 0; j < M; ++j) out[j] = genes[order[0] * M + j];        // elite (ties -> lowest index)
    // V3: candidates are member indices exactly as in G3; only at a restart generation (V2) are they drawn among the
    // live RANKS and mapped through order[].
    auto member = [&](uint32_t x) { return restart ? order[below(x, n_live)] : below(x, P); };
    auto pick = [&](const uint32_t r[4]) {
        int best = member(r[0]);
        for (int m = 1; m < c.tournament_k; ++m) {
            int cand = member(r[m]);
            if (chi2v[cand] < chi2v[best] || (chi2v[cand] == chi2v[best] && cand < best)) best = cand;
        }
        return best;
    };
    for (int i = 1; i < P; ++i) {
        if (i >= n_live) {                                               // V2: fresh points
            const uint32_t n = (uint32_t)(P + (t / n_samp - 1) * n_dead + (i - n_live) + 1);
            for (int j = 0; j < M; ++j) out[i * M + j] = sobol_gene(c, pixel, n, j);
            continue;
        }
        const int key = 2 * ((i + 1) / 2) - 1;                           // V4: pair (2q-1, 2q) keyed by 2q-1
        uint32_t r[4];
        draw(c, pixel, t, key, 0, r);  const int A = pick(r);
        draw(c, pixel, t, key, 1, r);  const int B = pick(r);
        draw(c, pixel, t, key, 2, r);
        const bool cross = u01(r[0]) < c.p_cross;
        const int cut = 1 + below(r[1], 16 * M - 1);
        const int first = (i & 1) ? A : B, second = (i & 1) ? B : A;
        for (int j = 0; j < M; ++j) {
            uint32_t k1 = (uint32_t)genes[first * M + j], k2 = (uint32_t)genes[second * M + j], k = k1;
            if (cross) {
                int nhead = cut - 16 * j; nhead = nhead < 0 ? 0 : (nhead > 16 ? 16 : nhead);
                const uint32_t mask = (0xFFFFu << (16 - nhead)) & 0xFFFFu;
                k = (k1 & mask) | (k2 & ~mask & 0xFFFFu);
            }
            if (j % 2 == 0) draw(c, pixel, t, i, 3 + j / 2, r);          // V5: own draws of child i
            const uint32_t xm = r[2 * (j % 2)], xd = r[2 * (j % 2) + 1];
            if (u01(xm) < c.p_mut) k ^= ((xd & 0xFFFFu) & (xd >> 16)) >> (xm & 15u);
            out[i * M + j] = (float)k;
        }
    }
}

// G2: generation 0, gene j of individual i = lane (j mod 4) of block floor(j / 4).
void ga_init(uint64_t pixel, const GaCfg& c, float* genes) {
    if (c.variant == 1) { ga_init_binary(pixel, c, genes); return; }
    for (int i = 0; i < c.pop; ++i)
        for (int j = 0; j < c.npar; ++j) {
            uint32_t r[4];
            draw(c, pixel, 0, i, j / 4, r);
            genes[i * c.npar + j] = u01(r[j % 4]);
        }
}

static int argmin(const double* v, int n) {
    int b = 0;
    for (int i = 1; i < n; ++i) if (v[i] < v[b]) b = i;     // ties -> lowest index
    return b;
}

// G3 selection: k-way tournament with replacement; winner = smallest chi2, ties -> smallest index.
static int tournament(const uint32_t r[4], const double* chi2v, const GaCfg& c) {
    int best = below(r[0], c.pop);
    for (int m = 1; m < c.tournament_k; ++m) {
        int cand = below(r[m], c.pop);
        if (chi2v[cand] < chi2v[best] || (chi2v[cand] == chi2v[best] && cand < best)) best = cand;
    }
    return best;
}

void ga_step(const float* genes, const double* chi2v, int t, uint64_t pixel, const GaCfg& c, float* out) {
    if (c.variant == 1) { ga_step_binary(genes, chi2v, t, pixel, c, out); return; }
    const int M = c.npar;
    const int elite = argmin(chi2v, c.pop);
    for (int j = 0; j < M; ++j) out[j] = genes[elite * M + j];               // slot 0 <- elite of t-1
    const float s_t = c.mut_scale[t];
    for (int i = 1; i < c.pop; ++i) {
        uint32_t r[4];
        draw(c, pixel, t, i, 0, r);  const int A = tournament(r, chi2v, c);
        draw(c, pixel, t, i, 1, r);  const int B = tournament(r, chi2v, c);
        draw(c, pixel, t, i, 2, r);
        const bool cross = u01(r[0]) < c.p_cross;
        const float alpha = u01(r[1]);
        for (int j = 0; j < M; ++j) {
            const float gA = genes[A * M + j], gB = genes[B * M + j];
            float g = gA;
            if (cross) { const float d = gA - gB; g = std::fmaf(alpha, d, gB); }    // arithmetic crossover
            if (j % 2 == 0) draw(c, pixel, t, i, 3 + j / 2, r);                     // pair (u_2j, u_2j+1)
            const float um = u01(r[2 * (j % 2)]), ud = u01(r[2 * (j % 2) + 1]);
            if (um < c.p_mut) { const float step = 2.0f * ud - 1.0f; g = std::fmaf(s_t, step, g); }
            if (c.periodic[j]) g = g - std::floor(g);                               // wrap (azimuth)
            else g = std::fmin(std::fmax(g, 0.0f), 1.0f);                           // clamp to the box (eq. 4)
            out[i * M + j] = g;
        }
    }
}

static double fitness(const float* g, const double* obs, double mu, const double* lambda, int L,
                      const Lines& ln, const GaCfg& c, std::vector<double>& model) {
    double p[MAXPAR];
    for (int j = 0; j < c.npar; ++j) p[j] = decode_gene(gene_value(g[j], c), c.lo[j], c.hi[j], c.log_scale[j]);
    synth_n(p, c.npar, mu, lambda, L, ln, c.nm_profile, model.data(), false);
    double x = chi2(obs, model.data(), L, c.w, c.sigma, c.npar);                     // nu = 4L - M
    if (!std::isfinite(x)) x = std::numeric_limits<double>::infinity();              // G4
    return x;
}

// W1 (eq. 20-23): w_I = 1 / (I_c - I_0), w_Q,U,V = 1 / max |Q,U,V|, with I_c the largest and I_0 the
//    smallest observed intensity of the window (continuum and line core); each denominator is floored at the noise
//    level sigma_s so that an empty Stokes parameter cannot blow the weight up; as for the fixed weights (reading F11)
//    the weight enters eq. 16 as (w_s / sigma_s)^2.
// P1: the inclination box is cut to one polarity, "in agreement with the order of the blue- and
//    red-lobes of the observed Stokes V": if the maximum of V lies at a shorter wavelength than its minimum (first
//    occurrences) the blue lobe is positive, which is gamma < 90 deg (reading F4): box [lo, min(hi, 90)]; else
//    [max(lo, 90), hi].
void pixel_prologue(const double* obs, int L, const GaCfg& c, double out[6]) {
    for (int s = 0; s < 4; ++s) out[s] = c.w[s];
    out[4] = c.lo[P_GAMMA]; out[5] = c.hi[P_GAMMA];
    if (c.prologue & 1) {
        double imax = obs[0], imin = obs[0];
        for (int j = 1; j < L; ++j) { imax = std::fmax(imax, obs[j]); imin = std::fmin(imin, obs[j]); }
        out[0] = 1.0 / std::fmax(imax - imin, c.sigma[0]);
        for (int s = 1; s < 4; ++s) {
            double m = 0.0;
            for (int j = 0; j < L; ++j) m = std::fmax(m, std::fabs(obs[s * L + j]));
            out[s] = 1.0 / std::fmax(m, c.sigma[s]);
        }
    }
    if (c.prologue & 2) {
        int jmax = 0, jmin = 0;
        for (int j = 1; j < L; ++j) {
            if (obs[3 * L + j] > obs[3 * L + jmax]) jmax = j;
            if (obs[3 * L + j] < obs[3 * L + jmin]) jmin = j;
        }
        if (jmax < jmin) out[5] = std::fmin(c.hi[P_GAMMA], 90.0);
        else out[4] = std::fmax(c.lo[P_GAMMA], 90.0);
    }
}

// S1: "the initial population includes ... the longitudinal field strength estimated from the
// center-of-gravity approach by Rees & Semel (1979) ... [and] the trivial non-magnetic solution".  The paper prints no
// formula; the textbook centre-of-gravity method is taken:
//   lambda_+- = sum_j lambda_j (I_c - (I_j +- V_j)) / sum_j (I_c - (I_j +- V_j)),   B_los = (lambda_+ - lambda_-) / (2 C g lambda_0^2),
// C = 4.66857e-13 /A/G, on the line with the largest g lambda_0^2 (g = centre of gravity of its sigma_red shifts), over
// the samples closer to that line than half the distance to the nearest other line (all samples for a single line), with
// I_c the largest observed intensity.  With reading F4 a positive blue V lobe deepens I - V on the blue side, so
// lambda_+ > lambda_- and B_los > 0 means gamma < 90 deg.  Seeded members (generation 0 only, pop >= 3):
//   slot P-1: B gene = 0 (the non-magnetic solution); slot P-2: B = |B_los| clamped to its box, gamma at the end of its
//   (polarity-cut) box that matches the sign of B_los; both box coordinates quantised to 10 bits (a heuristic needs no
//   more, and the two implementations then agree on the gene except at a rounding boundary); other genes as drawn.
void pixel_seeds(const double* obs, const double* lambda, int L, const Lines& ln, const GaCfg& c, double out[3]) {
    const double CZ = 4.66857e-13;
    int best = 0; double gbest = -1.0, sens = -1.0;
    for (size_t l = 0; l < ln.lines.size(); ++l) {
        double g = 0.0;
        for (const Component& k : ln.lines[l].comps) if (k.kind == 1) g += k.weight * k.shift;
        const double s = g * ln.lines[l].lambda0 * ln.lines[l].lambda0;
        if (s > sens) { sens = s; best = (int)l; gbest = g; }
    }
    const double l0 = ln.lines[best].lambda0;
    double hw = std::numeric_limits<double>::infinity();
    for (size_t l = 0; l < ln.lines.size(); ++l)
        if ((int)l != best) hw = std::fmin(hw, 0.5 * std::fabs(ln.lines[l].lambda0 - l0));
    double ic = obs[0];
    for (int j = 1; j < L; ++j) ic = std::fmax(ic, obs[j]);
    double sp = 0, sm = 0, lp = 0, lm = 0;
    for (int j = 0; j < L; ++j) {
        const double d = lambda[j] - l0;
        if (std::fabs(d) > hw) continue;
        const double ap = ic - (obs[j] + obs[3 * L + j]), am = ic - (obs[j] - obs[3 * L + j]);
        sp += ap; sm += am; lp += d * ap; lm += d * am;
    }
    double blos = 0.0;
    if (sp > 0.0 && sm > 0.0 && gbest > 0.0) blos = (lp / sp - lm / sm) / (2.0 * CZ * gbest * l0 * l0);
    const double b = std::fmin(std::fmax(std::fabs(blos), c.lo[P_B]), c.hi[P_B]);
    double u = 0.0;
    if (c.hi[P_B] > c.lo[P_B]) u = c.log_scale[P_B] ? std::log(b / c.lo[P_B]) / std::log(c.hi[P_B] / c.lo[P_B]) : (b - c.lo[P_B]) / (c.hi[P_B] - c.lo[P_B]);
    out[0] = blos;
    out[1] = std::rint(u * 1023.0);
    out[2] = blos >= 0.0 ? 0.0 : 1023.0;
}

// Reading S2: the weak-field member of P0 "as in Auer et al. (1977)".  The paper states its content in two places:
// "the longitudinal field strength is calculated from the separation between the I+-V line-cores, while the field orientation
// is calculated from Stokes Q, U, and V maxima" and "the seed fields are checked to ensure that they are
// consistent with this polarity".  Weak-field theory (Zeeman splitting dl_B = C g lambda0^2 B << Doppler width):
//   V = -dl_B cos(gamma) I',    (Q, U) = -(1/4) dl_B^2 sin^2(gamma) I'' (cos 2chi, sin 2chi).
// On the seed line's window of reading S1 (samples with |lambda - lambda0| <= hw; "interior" = both neighbours inside too):
//   1. core of y = I+V and of y = I-V: first minimum sample, refined by the vertex of the parabola through it and its two
//      neighbours when it is interior;  B_los = (lambda_+ - lambda_-) / (2 C g lambda0^2)   (I+V sees sigma_red, pin P2)
//   2. I', I'' by three-point differences on the interior samples; D1 = max |I'|, D2 = max |I''|, Vm = max |V|,
//      jL = first maximum of Q^2 + U^2, Lm = sqrt of it
//   3. chi = (1/2) atan2(s U_jL, s Q_jL) mod 180 deg with s = -1 where I'' >= 0 at jL (line core), +1 otherwise
//   4. tan(gamma') = 2 sqrt(Lm) D1 / (Vm sqrt(D2)), gamma' in [0, 90] (90 when Vm = 0 or D2 = 0);
//      gamma = gamma' for B_los >= 0, else 180 - gamma'; if that lies outside the pixel's inclination box [glo, ghi]
//      (polarity restriction, reading P1) it is reflected, gamma -> 180 - gamma, then clamped to the box
//   5. B = |B_los| / max(|cos gamma|, 1/8), clamped to its box
// out: [0] B_los (G), [1] gamma (deg), [2] chi (deg), [3] B (G), [4..6] the 10-bit box coordinates q of (B, gamma, chi).
void pixel_seed_auer(const double* obs, const double* lambda, int L, const Lines& ln, const GaCfg& c, double glo, double ghi,
                     double out[7]) {
    const double CZ = 4.66857e-13;
    int best = 0; double gbest = -1.0, sens = -1.0;
    for (size_t l = 0; l < ln.lines.size(); ++l) {
        double g = 0.0;
        for (const Component& k : ln.lines[l].comps) if (k.kind == 1) g += k.weight * k.shift;
        const double s = g * ln.lines[l].lambda0 * ln.lines[l].lambda0;
        if (s > sens) { sens = s; best = (int)l; gbest = g; }
    }
    const double l0 = ln.lines[best].lambda0;
    double hw = std::numeric_limits<double>::infinity();
    for (size_t l = 0; l < ln.lines.size(); ++l)
        if ((int)l != best) hw = std::fmin(hw, 0.5 * std::fabs(ln.lines[l].lambda0 - l0));
    const double *I = obs, *Q = obs + L, *U = obs + 2 * L, *V = obs + 3 * L;
    auto in = [&](int j) { return j >= 0 && j < L && std::fabs(lambda[j] - l0) <= hw; };
    auto interior = [&](int j) { return in(j - 1) && in(j) && in(j + 1); };
    // 1. line cores of I + V and I - V
    double core[2] = { 0.0, 0.0 };
    for (int k = 0; k < 2; ++k) {
        const double sg = k == 0 ? 1.0 : -1.0;
        int jm = -1; double ym = 0.0;
        for (int j = 0; j < L; ++j) {
            if (!in(j)) continue;
            const double y = I[j] + sg * V[j];
            if (jm < 0 || y < ym) { jm = j; ym = y; }
        }
        if (jm < 0) { for (int q = 0; q < 7; ++q) out[q] = 0.0; return; }
        double x = lambda[jm] - l0;
        if (interior(jm)) {
            const double x0 = lambda[jm - 1] - l0, x2 = lambda[jm + 1] - l0;
            const double y0 = I[jm - 1] + sg * V[jm - 1], y2 = I[jm + 1] + sg * V[jm + 1];
            const double a0 = x - x0, a2 = x - x2, num = a0 * a0 * (ym - y2) - a2 * a2 * (ym - y0), den = a0 * (ym - y2) - a2 * (ym - y0);
            if (den != 0.0) x -= 0.5 * num / den;
        }
        core[k] = x;
    }
    const double blos = gbest > 0.0 ? (core[0] - core[1]) / (2.0 * CZ * gbest * l0 * l0) : 0.0;
    // 2. derivative measures of I and the polarisation maxima, interior samples
    double D1 = 0.0, D2 = 0.0, Vm = 0.0, L2m = -1.0, d2L = 0.0, QL = 0.0, UL = 0.0;
    for (int j = 0; j < L; ++j) {
        if (!interior(j)) continue;
        const double hm = lambda[j] - lambda[j - 1], hp = lambda[j + 1] - lambda[j];
        const double d1 = (I[j + 1] - I[j - 1]) / (hm + hp);
        const double d2 = 2.0 * ((I[j + 1] - I[j]) / hp - (I[j] - I[j - 1]) / hm) / (hm + hp);
        D1 = std::fmax(D1, std::fabs(d1)); D2 = std::fmax(D2, std::fabs(d2)); Vm = std::fmax(Vm, std::fabs(V[j]));
        const double l2 = Q[j] * Q[j] + U[j] * U[j];
        if (l2 > L2m) { L2m = l2; d2L = d2; QL = Q[j]; UL = U[j]; }
    }
    if (L2m < 0.0) L2m = 0.0;
    // 3. azimuth
    const double s = d2L >= 0.0 ? -1.0 : 1.0;
    double chi = 0.5 * std::atan2(s * UL, s * QL) * 180.0 / M_PI;
    if (chi < 0.0) chi += 180.0;
    if (chi >= 180.0) chi -= 180.0;
    // 4. inclination
    double gp = 90.0;
    if (Vm > 0.0 && D2 > 0.0) gp = std::atan(2.0 * std::sqrt(std::sqrt(L2m)) * D1 / (Vm * std::sqrt(D2))) * 180.0 / M_PI;
    double gam = blos >= 0.0 ? gp : 180.0 - gp;
    if (gam < glo || gam > ghi) gam = 180.0 - gam;
    gam = std::fmin(std::fmax(gam, glo), ghi);
    // 5. field strength
    const double cg = std::fmax(std::fabs(std::cos(gam * M_PI / 180.0)), 0.125);
    const double b = std::fmin(std::fmax(std::fabs(blos) / cg, c.lo[P_B]), c.hi[P_B]);
    auto coord = [&](double v, double lo, double hi, int logs) {
        if (!(hi > lo)) return 0.0;
        const double u = logs ? std::log(v / lo) / std::log(hi / lo) : (v - lo) / (hi - lo);
        return std::rint(std::fmin(std::fmax(u, 0.0), 1.0) * 1023.0);
    };
    out[0] = blos; out[1] = gam; out[2] = chi; out[3] = b;
    out[4] = coord(b, c.lo[P_B], c.hi[P_B], c.log_scale[P_B]);
    out[5] = coord(gam, glo, ghi, 0);
    out[6] = coord(std::fmin(std::fmax(chi, c.lo[P_CHI]), c.hi[P_CHI]), c.lo[P_CHI], c.hi[P_CHI], 0);
}

// stored gene for a 10-bit box coordinate q: the real-coded variant holds q / 1023 (one binary32 division), the
// binary-coded variant the 16-bit code q << 6
static float seed_gene(double q, const GaCfg& c) { return c.variant == 1 ? (float)(64.0 * q) : (float)q / 1023.0f; }

void ga_invert_pixel(const double* obs, double mu, const double* lambda, int L, const Lines& ln, const GaCfg& c0,
                     uint64_t pixel, double* best_params, double* best_chi2, float* best_genes, double* trace) {
    GaCfg c = c0;                                                  // per-pixel weights and inclination box
    if (c0.prologue) {
        double pr[6];
        pixel_prologue(obs, L, c0, pr);
        for (int s = 0; s < 4; ++s) c.w[s] = pr[s];
        c.lo[P_GAMMA] = pr[4]; c.hi[P_GAMMA] = pr[5];
    }
    const int M = c.npar;
    std::vector<float> genes(c.pop * M), next(c.pop * M);
    std::vector<double> f(c.pop), fnext(c.pop), model(4 * L);
    ga_init(pixel, c, genes.data());
    if ((c0.prologue & 4) && c.pop >= 3) {                          // reading S1
        double sd[3];
        pixel_seeds(obs, lambda, L, ln, c, sd);
        genes[(c.pop - 1) * M + P_B] = seed_gene(0.0, c);
        genes[(c.pop - 2) * M + P_B] = seed_gene(sd[1], c);
        genes[(c.pop - 2) * M + P_GAMMA] = seed_gene(sd[2], c);
    }
    if ((c0.prologue & 8) && c.pop >= 4) {                          // reading S2: the Auer weak-field member, slot P-3
        double au[7];
        pixel_seed_auer(obs, lambda, L, ln, c, c.lo[P_GAMMA], c.hi[P_GAMMA], au);
        genes[(c.pop - 3) * M + P_B] = seed_gene(au[4], c);
        genes[(c.pop - 3) * M + P_GAMMA] = seed_gene(au[5], c);
        genes[(c.pop - 3) * M + P_CHI] = seed_gene(au[6], c);
    }
    for (int i = 0; i < c.pop; ++i) f[i] = fitness(&genes[i * M], obs, mu, lambda, L, ln, c, model);
    if (trace) trace[0] = f[argmin(f.data(), c.pop)];
    for (int t = 1; t <= c.generations; ++t) {
        const int elite = argmin(f.data(), c.pop);
        ga_step(genes.data(), f.data(), t, pixel, c, next.data());
        fnext[0] = f[elite];                                                          // carried, not re-evaluated
        for (int i = 1; i < c.pop; ++i) fnext[i] = fitness(&next[i * M], obs, mu, lambda, L, ln, c, model);
        genes.swap(next); f.swap(fnext);
        if (trace) trace[t] = f[argmin(f.data(), c.pop)];
    }
    const int b = argmin(f.data(), c.pop);                                             // G5
    for (int j = 0; j < M; ++j) {
        best_params[j] = decode_gene(gene_value(genes[b * M + j], c), c.lo[j], c.hi[j], c.log_scale[j]);
        if (best_genes) best_genes[j] = genes[b * M + j];
    }
    *best_chi2 = f[b];
}

}  // namespace orc
