// oracle/synth.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// Milne-Eddington forward synthesis, written in the order of DESIGN.md "Forward synthesis" (readings
// F1-F12), which restates eq. 7-16 of the paper.
#include "oracle.hpp"
#include <cmath>
#include <vector>

namespace orc {

static const double C_KMS = 299792.458;          // speed of light, km/s
static const double ZEEMAN = 4.66857e-13;        // e / (4 pi m_e c^2) in A^-1 G^-1 (reading: step 1)

// eq. 8: K = 1 + eta0 * Phi.  Elements of Phi after Landi Degl'Innocenti & Landolfi
// (2004), which the paper cites without printing them (reading F1), with the 1/sqrt(pi)
// normalisation of the profiles (reading F2) and F = Im w (reading F3).
Eta absorption_matrix(const double* p, double lambda, const Lines& ln) {
    const double B = p[P_B], gam = p[P_GAMMA] * M_PI / 180.0, chi = p[P_CHI] * M_PI / 180.0;
    const double eta0 = p[P_ETA0], dld_ref = p[P_DLD] * 1e-3, a = p[P_A], vlos = p[P_VLOS];
    cplx prof[3] = { cplx(0, 0), cplx(0, 0), cplx(0, 0) };   // index kind+1: [blue, pi, red]
    for (const Line& l : ln.lines) {
        double dld = dld_ref * l.lambda0 / ln.lambda_ref;                       // Doppler width of this line, A
        double v = ((lambda - l.lambda0) - l.lambda0 * vlos / C_KMS) / dld;     // distance from shifted centre
        double vB = ZEEMAN * l.lambda0 * l.lambda0 * B / dld;                   // Zeeman splitting, Doppler units
        for (const Component& c : l.comps) {
            cplx w = faddeeva(cplx(v - c.shift * vB, a));
            prof[c.kind + 1] += l.strength / std::sqrt(M_PI) * c.weight * w;
        }
    }
    const double h = 0.5 * eta0;
    const double sg = std::sin(gam), cg = std::cos(gam), s2 = sg * sg;
    const double c2x = std::cos(2.0 * chi), s2x = std::sin(2.0 * chi);
    const cplx pb = prof[0], pp = prof[1], pr = prof[2];
    cplx kI = h * (pp * s2 + 0.5 * (pb + pr) * (1.0 + cg * cg));
    cplx kL = h * (pp - 0.5 * (pb + pr)) * s2;          // linear-polarisation amplitude
    cplx kV = h * (pr - pb) * cg;
    Eta e;
    e.eI = 1.0 + kI.real();
    e.eQ = kL.real() * c2x;  e.eU = kL.real() * s2x;  e.eV = kV.real();
    e.rQ = kL.imag() * c2x;  e.rU = kL.imag() * s2x;  e.rV = kV.imag();
    return e;
}

// eq. 12 multiplied by I_c = S0 + mu S1 (eq. 15):  I = S0 e + mu S1 K^-1 e, K^-1 e in closed form
// (the Unno-Rachkovsky solution).
void stokes_closed_form(const Eta& e, double S0, double muS1, double out[4]) {
    const double eI = e.eI, eQ = e.eQ, eU = e.eU, eV = e.eV, rQ = e.rQ, rU = e.rU, rV = e.rV;
    const double Pi = eQ * rQ + eU * rU + eV * rV;
    const double Delta = eI * eI * (eI * eI - eQ * eQ - eU * eU - eV * eV + rQ * rQ + rU * rU + rV * rV) - Pi * Pi;
    out[0] = S0 + muS1 * eI * (eI * eI + rQ * rQ + rU * rU + rV * rV) / Delta;
    out[1] = -muS1 * (eI * eI * eQ + eI * (eV * rU - eU * rV) + rQ * Pi) / Delta;
    out[2] = -muS1 * (eI * eI * eU + eI * (eQ * rV - eV * rQ) + rU * Pi) / Delta;
    out[3] = -muS1 * (eI * eI * eV + eI * (eU * rQ - eQ * rU) + rV * Pi) / Delta;
}

// eq. 12 as printed: build K = 1 + eta0 Phi and solve K x = e-hat by Gaussian elimination with partial pivoting.
void stokes_by_solve(const Eta& e, double S0, double muS1, double out[4]) {
    double K[4][5] = {
        { e.eI,  e.eQ,  e.eU,  e.eV, 1.0 },
        { e.eQ,  e.eI,  e.rV, -e.rU, 0.0 },
        { e.eU, -e.rV,  e.eI,  e.rQ, 0.0 },
        { e.eV,  e.rU, -e.rQ,  e.eI, 0.0 } };
    for (int c = 0; c < 4; ++c) {
        int piv = c;
        for (int r = c + 1; r < 4; ++r) if (std::fabs(K[r][c]) > std::fabs(K[piv][c])) piv = r;
        for (int k = 0; k < 5; ++k) std::swap(K[c][k], K[piv][k]);
        for (int r = c + 1; r < 4; ++r) {
            double f = K[r][c] / K[c][c];
            for (int k = c; k < 5; ++k) K[r][k] -= f * K[c][k];
        }
    }
    double x[4];
    for (int r = 3; r >= 0; --r) {
        double s = K[r][4];
        for (int k = r + 1; k < 4; ++k) s -= K[r][k] * x[k];
        x[r] = s / K[r][r];
    }
    out[0] = S0 + muS1 * x[0];
    out[1] = muS1 * x[1];
    out[2] = muS1 * x[2];
    out[3] = muS1 * x[3];
}

void synth(const double* p, double mu, const double* lambda, int L, const Lines& ln, double* out, bool use_solve) {
    for (int j = 0; j < L; ++j) {
        Eta e = absorption_matrix(p, lambda[j], ln);
        double s[4];
        if (use_solve) stokes_by_solve(e, p[P_S0], mu * p[P_S1], s);
        else stokes_closed_form(e, p[P_S0], mu * p[P_S1], s);
        for (int k = 0; k < 4; ++k) out[k * L + j] = s[k];
    }
}

// 11-parameter model, reading F13: eq. 19 mixes the magnetic profile with a non-magnetic
// one by the fill fraction alpha; the non-magnetic component is the SAME atmosphere with B = 0; a fraction s of stray
// light with a fixed unpolarised profile is added on top (PAPER.md:251 treats it as a fixed 5 % correction; BASELINE
// config 4 makes it a free parameter):
//   I = (1 - s) [ alpha I^M(p) + (1 - alpha) I(p; B = 0) e ] + s I_fixed e.
void synth_n(const double* p, int npar, double mu, const double* lambda, int L, const Lines& ln,
             const double* nm_profile, double* out, bool use_solve) {
    synth(p, mu, lambda, L, ln, out, use_solve);                 // I^M(p): the first nine parameters
    if (npar == NPAR) return;
    const double alpha = p[P_ALPHA], s = p[P_STRAY];
    double q[NPAR];
    for (int j = 0; j < NPAR; ++j) q[j] = p[j];
    q[P_B] = 0.0;                                                // the same atmosphere without field
    std::vector<double> nm(4 * L);
    synth(q, mu, lambda, L, ln, nm.data(), use_solve);
    for (int j = 0; j < L; ++j) {
        out[j] = (1.0 - s) * (alpha * out[j] + (1.0 - alpha) * nm[j]) + s * nm_profile[j];
        for (int k = 1; k < 4; ++k) out[k * L + j] = (1.0 - s) * alpha * out[k * L + j];   // e = (1,0,0,0)
    }
}

// eq. 16 with weights constant over wavelength and nu = 4 N_lambda - M.
double chi2(const double* obs, const double* model, int L, const double w[4], const double sigma[4], int M) {
    double acc = 0.0;
    for (int s = 0; s < 4; ++s) {
        double ws = w[s] / sigma[s];
        for (int j = 0; j < L; ++j) {
            double d = obs[s * L + j] - model[s * L + j];
            acc += ws * ws * d * d;
        }
    }
    return acc / (4.0 * L - M);
}

}  // namespace orc
