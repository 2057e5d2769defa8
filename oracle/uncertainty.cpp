// oracle/uncertainty.cpp — TEST INFRASTRUCTURE (see oracle.hpp).
//
// Parameter uncertainties from the curvature of the chi-square manifold at the optimum:
// "The Hessian matrix H is ... calculated as the Jacobian of the resulting gradient vector and the variance of the
// i-th model parameter is given by  sigma_i^2 = [H^-1]_ii chi2(p_opt) / M"  (eq. 26), with the derivatives
// "bootstrap[ped] to higher accuracy by Richardson extrapolation to zero stepsize within Neville's algorithm".
// The paper starts from a population-based gradient (eq. 25) whose choice of members it does not specify; reading U1
// of DESIGN.md takes the deterministic equivalent: central second differences of chi2 on the box coordinates
// u in [0,1]^M (p = decode(u), reading G1) at steps h = UNC_H = 2^-6 and h/2, one Neville/Richardson level
//     D = (4 D(h/2) - D(h)) / 3,
//     D_jj(h) = [chi2(u + h e_j) - 2 chi2(u) + chi2(u - h e_j)] / h^2,
//     D_jk(h) = [chi2(++) - chi2(+-) - chi2(-+) + chi2(--)] / (4 h^2),
// H = D, sigma_u,i^2 = [H^-1]_ii chi2(u_opt) / M, and sigma_p,i = |dp_i/du_i| sigma_u,i (span for linear genes,
// p ln(hi/lo) for log-scaled ones).  A gene with lo == hi is fixed: it is left out of H and gets sigma = 0.
// A Hessian that is singular or gives [H^-1]_ii <= 0 yields NaN for that pixel's sigmas.
#include "oracle.hpp"
#include <cmath>
#include <limits>

namespace orc {

// Evaluation list shared by every implementation of reading U1: index 0 = centre, then for level l = 0, 1 (h_l = h / 2^l):
// 2 M diagonal points (j: +h, -h), then for each pair j < k the four points (++, +-, -+, --).
int uncertainty_n_eval(int M) { return 1 + 2 * (2 * M + 2 * M * (M - 1)); }

void uncertainty_offsets(int M, int e, double h, std::vector<double>& du) {
    du.assign(M, 0.0);
    if (e == 0) return;
    const int per_level = 2 * M + 2 * M * (M - 1);
    int r = e - 1;
    const int level = r / per_level;
    r -= level * per_level;
    const double hl = level == 0 ? h : 0.5 * h;
    if (r < 2 * M) { du[r / 2] = (r % 2 == 0) ? hl : -hl; return; }
    r -= 2 * M;
    int pair = r / 4, q = r % 4, j = 0;
    while (pair >= M - 1 - j) { pair -= M - 1 - j; ++j; }
    const int k = j + 1 + pair;
    du[j] = (q < 2) ? hl : -hl;
    du[k] = (q % 2 == 0) ? hl : -hl;
}

// Gauss-Jordan inversion with partial pivoting; returns false if singular.
static bool invert(std::vector<double>& a, int n) {
    std::vector<double> inv(n * n, 0.0);
    for (int i = 0; i < n; ++i) inv[i * n + i] = 1.0;
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (std::fabs(a[r * n + c]) > std::fabs(a[piv * n + c])) piv = r;
        if (!(std::fabs(a[piv * n + c]) > 0.0)) return false;
        for (int k = 0; k < n; ++k) { std::swap(a[c * n + k], a[piv * n + k]); std::swap(inv[c * n + k], inv[piv * n + k]); }
        const double d = 1.0 / a[c * n + c];
        for (int k = 0; k < n; ++k) { a[c * n + k] *= d; inv[c * n + k] *= d; }
        for (int r = 0; r < n; ++r) {
            if (r == c) continue;
            const double f = a[r * n + c];
            if (f == 0.0) continue;
            for (int k = 0; k < n; ++k) { a[r * n + k] -= f * a[c * n + k]; inv[r * n + k] -= f * inv[c * n + k]; }
        }
    }
    a = inv;
    return true;
}

// chi2v[n_eval] in the order of uncertainty_offsets -> sigma_u[M] (NaN on failure); active[j] = 0 leaves gene j out.
// hess_out (optional): the M x M Richardson-extrapolated Hessian in box coordinates, all genes (tests use its eigenvalues
// to say how well-posed eq. 26 is for a pixel).
void uncertainty_from_chi2(const double* chi2v, int M, double h, const int* active, double* sigma_u, double* hess_out) {
    const int per_level = 2 * M + 2 * M * (M - 1);
    std::vector<double> H(M * M, 0.0);
    for (int j = 0; j < M; ++j)
        for (int k = j; k < M; ++k) {
            double D[2];
            for (int level = 0; level < 2; ++level) {
                const double hl = level == 0 ? h : 0.5 * h;
                const double* c = chi2v + 1 + level * per_level;
                if (j == k) D[level] = (c[2 * j] - 2.0 * chi2v[0] + c[2 * j + 1]) / (hl * hl);
                else {
                    int pair = 0;
                    for (int a = 0; a < j; ++a) pair += M - 1 - a;
                    pair += k - j - 1;
                    const double* q = c + 2 * M + 4 * pair;
                    D[level] = (q[0] - q[1] - q[2] + q[3]) / (4.0 * hl * hl);
                }
            }
            H[j * M + k] = H[k * M + j] = (4.0 * D[1] - D[0]) / 3.0;          // Richardson / Neville, one level
        }
    if (hess_out) for (int q = 0; q < M * M; ++q) hess_out[q] = H[q];
    std::vector<int> idx;
    for (int j = 0; j < M; ++j) if (active[j]) idx.push_back(j);
    const int n = (int)idx.size();
    std::vector<double> A(n * n);
    for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) A[a * n + b] = H[idx[a] * M + idx[b]];
    const double nan = std::numeric_limits<double>::quiet_NaN();
    for (int j = 0; j < M; ++j) sigma_u[j] = active[j] ? nan : 0.0;
    if (n == 0 || !invert(A, n)) return;
    bool ok = true;
    for (int a = 0; a < n; ++a) if (!(A[a * n + a] > 0.0)) ok = false;
    if (!ok) return;
    for (int a = 0; a < n; ++a) sigma_u[idx[a]] = std::sqrt(A[a * n + a] * chi2v[0] / M);   // eq. 26
}

void uncertainty_pixel(const double* obs, double mu, const double* lambda, int L, const Lines& ln, const GaCfg& c0,
                       const double* params, double* sigma_p, double* chi2_opt, double* hess_out) {
    GaCfg c = c0;
    if (c0.prologue) {
        double pr[6];
        pixel_prologue(obs, L, c0, pr);
        for (int s = 0; s < 4; ++s) c.w[s] = pr[s];
        c.lo[P_GAMMA] = pr[4]; c.hi[P_GAMMA] = pr[5];
    }
    const int M = c.npar;
    const double h = UNC_H;
    std::vector<double> u0(M), p(M), du, model(4 * L);
    std::vector<int> active(M);
    for (int j = 0; j < M; ++j) {
        active[j] = c.hi[j] > c.lo[j];
        if (!active[j]) u0[j] = 0.0;
        else if (c.log_scale[j]) u0[j] = std::log(params[j] / c.lo[j]) / std::log(c.hi[j] / c.lo[j]);
        else u0[j] = (params[j] - c.lo[j]) / (c.hi[j] - c.lo[j]);
    }
    const int ne = uncertainty_n_eval(M);
    std::vector<double> chi2v(ne);
    for (int e = 0; e < ne; ++e) {
        uncertainty_offsets(M, e, h, du);
        for (int j = 0; j < M; ++j) {
            const double u = u0[j] + du[j];
            p[j] = c.log_scale[j] ? c.lo[j] * std::pow(c.hi[j] / c.lo[j], u) : c.lo[j] + (c.hi[j] - c.lo[j]) * u;
        }
        synth_n(p.data(), M, mu, lambda, L, ln, c.nm_profile, model.data(), false);
        chi2v[e] = chi2(obs, model.data(), L, c.w, c.sigma, M);
    }
    std::vector<double> su(M);
    uncertainty_from_chi2(chi2v.data(), M, h, active.data(), su.data(), hess_out);
    for (int j = 0; j < M; ++j) {
        const double dpdu = c.log_scale[j] ? params[j] * std::log(c.hi[j] / c.lo[j]) : (c.hi[j] - c.lo[j]);
        sigma_p[j] = su[j] * std::fabs(dpdu);
    }
    if (chi2_opt) *chi2_opt = chi2v[0];
}

}  // namespace orc
