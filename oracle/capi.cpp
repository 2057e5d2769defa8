// oracle/capi.cpp — TEST INFRASTRUCTURE (see oracle.hpp): flat C entry points for ctypes, plus the
// std::thread fan-out over independent pixels / parameter vectors used when the oracle is timed.
#include "oracle.hpp"
#include <atomic>
#include <cmath>
#include <cstring>
#include <limits>
#include <thread>

using namespace orc;

namespace {

// Flat line description: per line (lambda0, strength, n_comp), components concatenated.
Lines make_lines(int n_lines, const double* lambda0, const double* strength, const int* n_comp,
                 const double* shift, const double* weight, const int* kind, double lambda_ref) {
    Lines ln; ln.lambda_ref = lambda_ref;
    int o = 0;
    for (int l = 0; l < n_lines; ++l) {
        Line li; li.lambda0 = lambda0[l]; li.strength = strength[l];
        for (int c = 0; c < n_comp[l]; ++c, ++o) li.comps.push_back(Component{ shift[o], weight[o], kind[o] });
        ln.lines.push_back(li);
    }
    return ln;
}

template <class F> void parallel_for(int64_t n, int threads, F f) {
    if (threads < 1) threads = 1;
    std::atomic<int64_t> next(0);
    std::vector<std::thread> th;
    for (int k = 0; k < threads; ++k)
        th.emplace_back([&]() { for (;;) { int64_t i = next.fetch_add(1); if (i >= n) break; f(i); } });
    for (auto& t : th) t.join();
}

GaCfg make_cfg(int pop, int generations, int tournament_k, float p_cross, float p_mut, const float* mut_scale,
               const double* lo, const double* hi, const int* log_scale, const int* periodic,
               const double* w, const double* sigma, uint64_t seed, int npar = NPAR, const double* nm_profile = nullptr, int variant = 0, int prologue = 0) {
    GaCfg c; c.prologue = prologue; c.variant = variant; c.npar = npar; c.nm_profile = nm_profile; c.pop = pop; c.generations = generations; c.tournament_k = tournament_k;
    c.p_cross = p_cross; c.p_mut = p_mut; c.mut_scale.assign(mut_scale, mut_scale + generations + 1);
    for (int j = 0; j < npar; ++j) { c.lo[j] = lo[j]; c.hi[j] = hi[j]; c.log_scale[j] = log_scale[j]; c.periodic[j] = periodic[j]; }
    for (int s = 0; s < 4; ++s) { c.w[s] = w[s]; c.sigma[s] = sigma[s]; }
    c.seed = seed;
    return c;
}

}  // namespace

extern "C" {

int orc_hardware_threads() { return (int)std::thread::hardware_concurrency(); }

void orc_faddeeva(const double* re, const double* im, int64_t n, double* wre, double* wim) {
    for (int64_t i = 0; i < n; ++i) { cplx w = faddeeva(cplx(re[i], im[i])); wre[i] = w.real(); wim[i] = w.imag(); }
}

double orc_lande_g(double S, double L, double J) { return lande_g(S, L, J); }
double orc_g_eff(double gl, double Jl, double gu, double Ju) { return g_eff(gl, Jl, gu, Ju); }

// Returns the number of components; fills up to cap entries.
int orc_zeeman_pattern(double Sl, double Ll, double Jl, double Su, double Lu, double Ju, int cap,
                       double* shift, double* weight, int* kind) {
    std::vector<Component> c = zeeman_pattern(Sl, Ll, Jl, Su, Lu, Ju);
    for (int i = 0; i < (int)c.size() && i < cap; ++i) { shift[i] = c[i].shift; weight[i] = c[i].weight; kind[i] = c[i].kind; }
    return (int)c.size();
}

// params[P][npar], mu[P] (or null => 1), out[P][4][L]; use_solve: 0 closed form, 1 Gaussian elimination of eq. 12.
// npar = 11 adds (alpha, s) and needs nm_profile[L] (reading F13).
void orc_synth(const double* params, int npar, const double* nm_profile, const double* mu, int64_t P, const double* lambda, int L,
               int n_lines, const double* lambda0, const double* strength, const int* n_comp,
               const double* shift, const double* weight, const int* kind, double lambda_ref,
               int use_solve, int threads, double* out) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    parallel_for(P, threads, [&](int64_t i) {
        synth_n(params + i * npar, npar, mu ? mu[i] : 1.0, lambda, L, ln, nm_profile, out + i * 4 * L, use_solve != 0);
    });
}

// Absorption-matrix elements at one wavelength: out[7] = eI,eQ,eU,eV,rQ,rU,rV.
void orc_absorption_matrix(const double* p, double lambda, int n_lines, const double* lambda0, const double* strength,
                           const int* n_comp, const double* shift, const double* weight, const int* kind,
                           double lambda_ref, double* out) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    Eta e = absorption_matrix(p, lambda, ln);
    out[0] = e.eI; out[1] = e.eQ; out[2] = e.eU; out[3] = e.eV; out[4] = e.rQ; out[5] = e.rU; out[6] = e.rV;
}

double orc_chi2(const double* obs, const double* model, int L, const double* w, const double* sigma, int M) {
    return chi2(obs, model, L, w, sigma, M);
}

void orc_philox(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t* out) {
    uint32_t ctr[4] = { c0, c1, c2, c3 }, key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    philox4x32_10(ctr, key, out);
}
// Per-pixel prologue: obs[N][4][L] -> out[N][6] (w_I, w_Q, w_U, w_V, gamma_lo, gamma_hi).
void orc_prologue(const double* obs, int64_t N, int L, const double* w, const double* sigma, double gamma_lo, double gamma_hi,
                  int prologue, double* out) {
    GaCfg c; c.prologue = prologue;
    for (int s = 0; s < 4; ++s) { c.w[s] = w[s]; c.sigma[s] = sigma[s]; }
    c.lo[P_GAMMA] = gamma_lo; c.hi[P_GAMMA] = gamma_hi;
    for (int64_t n = 0; n < N; ++n) pixel_prologue(obs + n * 4 * L, L, c, out + n * 6);
}

// Uncertainties (reading U1). params[N][npar] -> sigma_out[N][npar], chi2_out[N], hess_out[N][npar][npar] (each may be null).
double orc_uncertainty_step() { return UNC_H; }
void orc_uncertainty(const double* obs, const double* mu, int64_t N, const double* lambda, int L,
                     int n_lines, const double* lambda0, const double* strength, const int* n_comp,
                     const double* shift, const double* weight, const int* kind, double lambda_ref,
                     const double* lo, const double* hi, const int* log_scale, const double* w, const double* sigma,
                     int npar, int prologue, const double* nm_profile, const double* params, int threads,
                     double* sigma_out, double* chi2_out, double* hess_out /* [N][npar][npar] or null */) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    GaCfg c; c.npar = npar; c.nm_profile = nm_profile; c.prologue = prologue;
    for (int j = 0; j < npar; ++j) { c.lo[j] = lo[j]; c.hi[j] = hi[j]; c.log_scale[j] = log_scale[j]; c.periodic[j] = 0; }
    for (int s = 0; s < 4; ++s) { c.w[s] = w[s]; c.sigma[s] = sigma[s]; }
    parallel_for(N, threads, [&](int64_t n) {
        uncertainty_pixel(obs + n * 4 * L, mu ? mu[n] : 1.0, lambda, L, ln, c, params + n * npar, sigma_out + n * npar,
                          chi2_out ? chi2_out + n : nullptr, hess_out ? hess_out + n * npar * npar : nullptr);
    });
}

// The finite-difference machinery alone on a caller-supplied table of function values (pins): chi2v[n_eval(M)].
int orc_uncertainty_n_eval(int M) { return uncertainty_n_eval(M); }
void orc_uncertainty_offsets(int M, int e, double h, double* du) {
    std::vector<double> v; uncertainty_offsets(M, e, h, v);
    for (int j = 0; j < M; ++j) du[j] = v[j];
}
void orc_uncertainty_from_chi2(const double* chi2v, int M, double h, const int* active, double* sigma_u) {
    uncertainty_from_chi2(chi2v, M, h, active, sigma_u);
}

// Heuristic seeds of one batch: obs[N][4][L] -> out[N][3] = B_los [G], q_B, q_gamma (reading S1).
void orc_seeds(const double* obs, int64_t N, const double* lambda, int L,
               int n_lines, const double* lambda0, const double* strength, const int* n_comp,
               const double* shift, const double* weight, const int* kind, double lambda_ref,
               double b_lo, double b_hi, int b_log, double* out) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    GaCfg c; c.lo[P_B] = b_lo; c.hi[P_B] = b_hi; c.log_scale[P_B] = b_log;
    for (int64_t n = 0; n < N; ++n) pixel_seeds(obs + n * 4 * L, lambda, L, ln, c, out + n * 3);
}

// Auer weak-field member of one batch (reading S2): obs[N][4][L] -> out[N][7] = B_los, gamma, chi, B, q_B, q_gamma, q_chi.
// glo/ghi[N]: the per-pixel inclination box (the configured one, or the polarity-cut one of reading P1).
void orc_seed_auer(const double* obs, int64_t N, const double* lambda, int L,
                   int n_lines, const double* lambda0, const double* strength, const int* n_comp,
                   const double* shift, const double* weight, const int* kind, double lambda_ref,
                   double b_lo, double b_hi, int b_log, double chi_lo, double chi_hi, const double* glo, const double* ghi,
                   double* out) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    GaCfg c; c.lo[P_B] = b_lo; c.hi[P_B] = b_hi; c.log_scale[P_B] = b_log; c.lo[P_CHI] = chi_lo; c.hi[P_CHI] = chi_hi;
    for (int64_t n = 0; n < N; ++n) pixel_seed_auer(obs + n * 4 * L, lambda, L, ln, c, glo[n], ghi[n], out + n * 7);
}

// count Sobol' points starting at index n0, dims dimensions: out[count][dims] (32-bit fixed point).
void orc_sobol(uint32_t n0, int count, int dims, uint32_t* out) {
    for (int i = 0; i < count; ++i)
        for (int j = 0; j < dims; ++j) out[i * dims + j] = sobol_point(n0 + (uint32_t)i, j);
}
void orc_philox_raw(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

void orc_decode(const float* genes, int npar, int variant, int64_t n, const double* lo, const double* hi, const int* log_scale, double* out) {
    GaCfg c; c.variant = variant;
    for (int64_t i = 0; i < n; ++i)
        for (int j = 0; j < npar; ++j) out[i * npar + j] = decode_gene(gene_value(genes[i * npar + j], c), lo[j], hi[j], log_scale[j]);
}

void orc_ga_init(int64_t N, uint64_t pixel_base, int pop, int npar, int variant, uint64_t seed, float* genes) {
    GaCfg c; c.pop = pop; c.seed = seed; c.npar = npar; c.variant = variant;
    for (int64_t n = 0; n < N; ++n) ga_init(pixel_base + n, c, genes + n * pop * npar);
}

// One generation for N pixels: genes_in[N][pop][9], chi2_in[N][pop] (double) -> genes_out.
void orc_ga_step(const float* genes_in, const double* chi2_in, int64_t N, uint64_t pixel_base, int t,
                 int pop, int generations, int tournament_k, float p_cross, float p_mut, const float* mut_scale,
                 const int* periodic, int npar, int variant, uint64_t seed, float* genes_out) {
    double z[MAXPAR] = {0}; int zi[MAXPAR] = {0}; double w4[4] = {1, 1, 1, 1};
    GaCfg c = make_cfg(pop, generations, tournament_k, p_cross, p_mut, mut_scale, z, z, zi, periodic, w4, w4, seed, npar, nullptr, variant);
    for (int64_t n = 0; n < N; ++n)
        ga_step(genes_in + n * pop * npar, chi2_in + n * pop, t, pixel_base + n, c, genes_out + n * pop * npar);
}

// Fitness (decode -> synth -> chi2) of genes[N][pop][9] against obs[N][4][L]: chi2_out[N][pop].
void orc_ga_fitness(const float* genes, const double* obs, const double* mu, int64_t N, int pop, const double* lambda, int L,
                    int n_lines, const double* lambda0, const double* strength, const int* n_comp,
                    const double* shift, const double* weight, const int* kind, double lambda_ref,
                    const double* lo, const double* hi, const int* log_scale, const double* w, const double* sigma,
                    int npar, int variant, const double* nm_profile, int threads, double* chi2_out) {
    GaCfg gv; gv.variant = variant;
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    parallel_for(N * pop, threads, [&](int64_t k) {
        int64_t n = k / pop;
        double p[MAXPAR];
        for (int j = 0; j < npar; ++j) p[j] = decode_gene(gene_value(genes[k * npar + j], gv), lo[j], hi[j], log_scale[j]);
        std::vector<double> model(4 * L);
        synth_n(p, npar, mu ? mu[n] : 1.0, lambda, L, ln, nm_profile, model.data(), false);
        double x = chi2(obs + n * 4 * L, model.data(), L, w, sigma, npar);
        chi2_out[k] = std::isfinite(x) ? x : std::numeric_limits<double>::infinity();
    });
}

// Whole inversion of N pixels (mask[n] == 0 => skipped, outputs NaN).  trace may be null, else [N][generations+1].
void orc_ga_invert(const double* obs, const unsigned char* mask, const double* mu, int64_t N, uint64_t pixel_base,
                   const double* lambda, int L,
                   int n_lines, const double* lambda0, const double* strength, const int* n_comp,
                   const double* shift, const double* weight, const int* kind, double lambda_ref,
                   int pop, int generations, int tournament_k, float p_cross, float p_mut, const float* mut_scale,
                   const double* lo, const double* hi, const int* log_scale, const int* periodic,
                   const double* w, const double* sigma, int npar, int variant, int prologue, const double* nm_profile, uint64_t seed, int threads,
                   double* out_params, double* out_chi2, float* out_genes, double* trace) {
    Lines ln = make_lines(n_lines, lambda0, strength, n_comp, shift, weight, kind, lambda_ref);
    GaCfg c = make_cfg(pop, generations, tournament_k, p_cross, p_mut, mut_scale, lo, hi, log_scale, periodic, w, sigma, seed, npar, nm_profile, variant, prologue);
    parallel_for(N, threads, [&](int64_t n) {
        if (mask && !mask[n]) {
            for (int j = 0; j < npar; ++j) out_params[n * npar + j] = std::nan("");
            out_chi2[n] = std::nan("");
            return;
        }
        ga_invert_pixel(obs + n * 4 * L, mu ? mu[n] : 1.0, lambda, L, ln, c, pixel_base + n,
                        out_params + n * npar, out_chi2 + n, out_genes ? out_genes + n * npar : nullptr,
                        trace ? trace + n * (generations + 1) : nullptr);
    });
}

}  // extern "C"
