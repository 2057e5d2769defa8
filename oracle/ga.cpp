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
#include <limits>

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

// G1: gene in [0,1] -> physical parameter, from the binary32 gene, in double.
double decode_gene(float g, double lo, double hi, int log_scale) {
    if (log_scale) return lo * std::pow(hi / lo, (double)g);
    return lo + (hi - lo) * (double)g;
}

// G2: generation 0, gene j of individual i = lane (j mod 4) of block floor(j / 4).
void ga_init(uint64_t pixel, const GaCfg& c, float* genes) {
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
    for (int j = 0; j < c.npar; ++j) p[j] = decode_gene(g[j], c.lo[j], c.hi[j], c.log_scale[j]);
    synth_n(p, c.npar, mu, lambda, L, ln, c.nm_profile, model.data(), false);
    double x = chi2(obs, model.data(), L, c.w, c.sigma, c.npar);                     // nu = 4L - M
    if (!std::isfinite(x)) x = std::numeric_limits<double>::infinity();              // G4
    return x;
}

void ga_invert_pixel(const double* obs, double mu, const double* lambda, int L, const Lines& ln, const GaCfg& c,
                     uint64_t pixel, double* best_params, double* best_chi2, float* best_genes, double* trace) {
    const int M = c.npar;
    std::vector<float> genes(c.pop * M), next(c.pop * M);
    std::vector<double> f(c.pop), fnext(c.pop), model(4 * L);
    ga_init(pixel, c, genes.data());
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
        best_params[j] = decode_gene(genes[b * M + j], c.lo[j], c.hi[j], c.log_scale[j]);
        if (best_genes) best_genes[j] = genes[b * M + j];
    }
    *best_chi2 = f[b];
}

}  // namespace orc
