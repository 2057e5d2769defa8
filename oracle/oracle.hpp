// oracle/oracle.hpp — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, double-precision CPU statement of what the GENESIS hot path computes
// (Harker & Mighell, arxiv 1208.0302): Milne-Eddington forward synthesis of I,Q,U,V, the
// chi-square merit (eq. 16) and the per-pixel genetic algorithm (Alg. 1).  It exists so that the
// CUDA path under paper_1208_0302_b200/csrc has something independent to be compared with.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call it.  It shares no source, header, table or helper with the CUDA path.
//
// Citations are PAPER.md line numbers plus the equation they fall in;
// "reading Fn/Gn" refers to the list of readings in DESIGN.md (taken from SURVEY.md §8(c)).
//
// Parity pins (tests/test_oracle_*.py, -m "not gpu"):
//   faddeeva       pinned  (erfc / Dawson closed forms, scipy.special.wofz, ODE w' = -2zw + 2i/sqrt(pi))
//   zeeman_pattern pinned  (Table 1 g_eff, 12 components for 6301.5, centre-of-gravity identity)
//   synth          pinned  (B=0 and gamma=0 closed forms, 4x4 solve of eq. 12, symmetries, weak field;
//                           P12 gamma=90/chi=0 closed form I+-Q through scipy's wofz fixes the linear-polarisation
//                           amplitude kL; P13 eta0 -> 0 expansion e - eta0 A e + eta0^2 A^2 e, A built in numpy from the
//                           LL04 matrix, fixes the signs of rho_Q, rho_U, rho_V and of K: both fail when kL is halved
//                           or the .imag() terms are negated)
//   chi2           pinned  (expected value at truth, brute-force grid minimum)
//   philox4x32_10  pinned  (published known-answer vectors of Salmon et al. 2011)
//   synth_n (11 parameters, reading F13) pinned (alpha=1,s=0 -> synth; alpha=0 -> B=0 closed form; s=1 -> I_fixed;
//                  Q,U,V scale with (1-s) alpha; bilinearity in alpha and s)
//   uncertainty    pinned  (exact Hessian of quadratic / quartic test functions, closed-form inverse; noise scaling)
//   ga             operators pinned by brute-force re-derivation in Python on tiny inputs (both variants, incl. the
//                  member-index rule of variant-1 tournaments inside and outside restart generations) and by
//                  invariants; absolute recovery accuracy: PARITY UNPINNED (the paper prints no
//                  reproducible recovery numbers, Table 4 PAPER.md:340-345 is for SOLIS data).
#pragma once
#include <complex>
#include <cstdint>
#include <vector>

namespace orc {

typedef std::complex<double> cplx;

// ---- Faddeeva function w(z) = exp(-z^2) erfc(-iz), Im z > 0  (H = Re w, F = Im w; reading F3) ----
cplx faddeeva(cplx z);

// ---- Zeeman pattern in LS coupling ("full Zeeman pattern ... calculated at the start") ----
struct Component { double shift; double weight; int kind; };   // kind: 0 = pi, -1 = sigma_blue, +1 = sigma_red
double lande_g(double S, double L, double J);
double g_eff(double gl, double Jl, double gu, double Ju);
std::vector<Component> zeeman_pattern(double Sl, double Ll, double Jl, double Su, double Lu, double Ju);
std::vector<Component> zeeman_triplet(double geff);

// ---- Line table + model ----
struct Line { double lambda0; double strength; std::vector<Component> comps; };
struct Lines { std::vector<Line> lines; double lambda_ref; };

// Parameter order (BASELINE config 0; differs from eq. 14):
// [B (G), gamma (deg), chi (deg), eta0, dlambdaD (mA at lambda_ref), a, v_los (km/s), S0, S1]
enum { P_B = 0, P_GAMMA, P_CHI, P_ETA0, P_DLD, P_A, P_VLOS, P_S0, P_S1, NPAR = 9,
       P_ALPHA = 9, P_STRAY = 10, MAXPAR = 11 };
// 11-parameter model (eq. 19 PAPER.md:245-247 + stray light PAPER.md:251; reading F13 of DESIGN.md):
//   I = (1 - s) [ alpha I^M(p) + (1 - alpha) I(p; B = 0) e ] + s I_fixed(lambda) e
// alpha = magnetic fill fraction, s = stray-light fraction, I_fixed = a fixed unpolarised profile (nm_profile[L]).

// Absorption-matrix elements at one wavelength (eq. 8; reading F1/F2).
struct Eta { double eI, eQ, eU, eV, rQ, rU, rV; };
Eta absorption_matrix(const double* p, double lambda, const Lines& ln);

// Unno-Rachkovsky solution, closed form (eq. 12-13, 15 PAPER.md:204-216; reading F6): out[4].
void stokes_closed_form(const Eta& e, double S0, double muS1, double out[4]);
// The same by building K and solving K x = e by Gaussian elimination (eq. 12 as printed).
void stokes_by_solve(const Eta& e, double S0, double muS1, double out[4]);

// Full profile: out[4][L].  use_solve selects the second path.
void synth(const double* p, double mu, const double* lambda, int L, const Lines& ln, double* out, bool use_solve);
// The same for npar = 9 (identical to synth) or npar = 11 (reading F13; nm_profile[L] is I_fixed).
void synth_n(const double* p, int npar, double mu, const double* lambda, int L, const Lines& ln,
             const double* nm_profile, double* out, bool use_solve);

// eq. 16, reading F11: chi2 = 1/nu * sum_s sum_j (w_s/sigma_s)^2 (O - M)^2, nu = 4L - M.
double chi2(const double* obs, const double* model, int L, const double w[4], const double sigma[4], int M);

// ---- Philox4x32-10 (Salmon et al. 2011), reading G0 ----
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

// ---- Sobol' sequence (Bratley & Fox 1988), dims 0..10 ----
void sobol_directions(int dim, uint32_t v[32]);
uint32_t sobol_point(uint32_t n, int dim);      // 32-bit fixed point, Gray-code order, n = 0 is the origin

// ---- GA (Alg. 1; readings G0-G5) ----
struct GaCfg {
    int pop, generations, tournament_k;
    float p_cross, p_mut;
    std::vector<float> mut_scale;              // s_t for t = 0..generations (built by the caller, binary32)
    int npar = NPAR;                           // 9 or 11 genes
    int variant = 0;                           // 0: real-coded operators (north_star, readings G1-G3)
                                               // 1: the paper's binary-coded GA (16-bit genotype, one-point crossover,
                                               //    LSB-biased bit mutation, Sobol init + restarts; readings V0-V5)
    const double* nm_profile = nullptr;        // I_fixed[L] for npar = 11
    double lo[MAXPAR], hi[MAXPAR];
    int log_scale[MAXPAR], periodic[MAXPAR];
    double w[4], sigma[4];
    uint64_t seed;
    int prologue = 0;                          // bit 0: inverse-max weights (eq. 20-23), bit 1: polarity restriction of gamma,
                                               // bit 2: heuristic seeds in P0 (reading S1)
};
// Per-pixel prologue of the paper (SURVEY.md par. 8(f)-3; readings W1, P1 of DESIGN.md), computed from the observed
// profile alone.  out[6] = w_I, w_Q, w_U, w_V (eq. 20-23; unchanged c.w if bit 0 is clear) and the
// inclination box [gamma_lo, gamma_hi] (the configured box if bit 1 is clear).
void pixel_prologue(const double* obs, int L, const GaCfg& c, double out[6]);
// Heuristic seeds (reading S1 of DESIGN.md): the centre-of-gravity longitudinal field B_los (Rees &
// Semel 1979) of the most Zeeman-sensitive line, in Gauss (signed), and the box coordinates (u_B, u_gamma) of the seeded
// member, quantised to 10 bits: out[3] = B_los, q_B, q_gamma (q in 0..1023).
void pixel_seeds(const double* obs, const double* lambda, int L, const Lines& ln, const GaCfg& c, double out[3]);
// Reading S2: the weak-field member "as in Auer et al. (1977)"; [glo, ghi] = the pixel's inclination box.
// out: B_los, gamma, chi, B, then the 10-bit box coordinates of (B, gamma, chi).  prologue bit 8, slot P-3 of P0 (pop >= 4).
void pixel_seed_auer(const double* obs, const double* lambda, int L, const Lines& ln, const GaCfg& c, double glo, double ghi,
                     double out[7]);
double decode_gene(float g, double lo, double hi, int log_scale);
float gene_value(float stored, const GaCfg& c);   // variant 1: 16-bit code -> g = k / 65535 (eq. 5), rounded to binary32
// Next generation from (genes[pop][NPAR], chi2[pop]) at generation t >= 1 for global pixel id `pixel`.
void ga_step(const float* genes, const double* chi2v, int t, uint64_t pixel, const GaCfg& c, float* out);
void ga_init(uint64_t pixel, const GaCfg& c, float* genes);
// Whole inversion of one pixel: obs[4][L] (double). Returns best decoded params and chi2;
// if trace != nullptr it receives best chi2 per generation (generations+1 values).
void ga_invert_pixel(const double* obs, double mu, const double* lambda, int L, const Lines& ln, const GaCfg& c,
                     uint64_t pixel, double* best_params, double* best_chi2, float* best_genes, double* trace);

// ---- Uncertainties (eq. 25-26; reading U1 of DESIGN.md) ----
// Step of the central second differences in box coordinates (the paper names none).  2^-6: the FP64 sigmas
// move by <= 1.6 % (median 0.00 %) against 2^-7 and by up to 58 % on an ill-conditioned pixel at 2^-5 (measured on config-0
// optima when the reading was amended), while a binary32 evaluation of chi2 puts a noise ~ eps chi2 / h^2 on every curvature.
const double UNC_H = 1.0 / 64.0;
int uncertainty_n_eval(int M);
void uncertainty_offsets(int M, int e, double h, std::vector<double>& du);
void uncertainty_from_chi2(const double* chi2v, int M, double h, const int* active, double* sigma_u, double* hess_out = nullptr);
void uncertainty_pixel(const double* obs, double mu, const double* lambda, int L, const Lines& ln, const GaCfg& c,
                       const double* params, double* sigma_p, double* chi2_opt, double* hess_out = nullptr);

}  // namespace orc
