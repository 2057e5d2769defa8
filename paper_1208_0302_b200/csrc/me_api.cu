// me_api.cu — the C ABI of include/me.h: argument validation, descriptor construction (host), launches.
#include <cmath>
#include <cstring>
#include <string>
#include <vector>

#include "me_device.cuh"
#include "me_launch.h"

namespace {

thread_local std::string g_cuda_err;

int cuda_fail(cudaError_t e) {
    g_cuda_err = cudaGetErrorString(e);
    return ME_ERR_CUDA;
}

const double C_KMS = 299792.458;       // speed of light, km/s
const double ZEEMAN = 4.66857e-13;     // e / (4 pi m_e c^2), A^-1 G^-1

// Build the kernel-side synthesis descriptor from the caller's line list and wavelength grid.
int build_synth_desc(const double* lambda, int L, const me_line_data* ld, me::SynthDesc& d) {
    if (lambda == nullptr || ld == nullptr || ld->lines == nullptr) return ME_ERR_NULL;
    if (L < 2 || L > ME_MAX_L) return ME_ERR_SHAPE;
    if (ld->n_lines < 1 || ld->n_lines > ME_MAX_LINES) return ME_ERR_SHAPE;
    if (ld->n_params != ME_NPAR && ld->n_params != ME_MAX_NPAR) return ME_ERR_SHAPE;
    if (4 * L <= ld->n_params) return ME_ERR_SHAPE;           // nu = 4 L - M of eq. 16 must be positive
    for (int j = 0; j < L; ++j) {                             // finite and strictly increasing (the prologue's lobe order and
        if (!std::isfinite(lambda[j])) return ME_ERR_RANGE;   // centre of gravity, readings P1 / S1, assume ascending wavelength)
        if (j > 0 && !(lambda[j] > lambda[j - 1])) return ME_ERR_RANGE;
    }
    if (ld->n_params == ME_MAX_NPAR && ld->nm_profile == nullptr) return ME_ERR_NULL;   // reading F13 needs I_fixed
    if (ld->n_params == ME_NPAR && ld->nm_profile != nullptr) return ME_ERR_SHAPE;
    if (!(ld->lambda_ref_A > 0.0)) return ME_ERR_RANGE;
    std::memset(&d, 0, sizeof(d));
    d.L = L; d.n_lines = ld->n_lines; d.all_triplets = 1;
    d.npar = ld->n_params; d.nm_profile = ld->nm_profile;
    int o = 0;
    for (int l = 0; l < ld->n_lines; ++l) {
        const me_line& ln = ld->lines[l];
        if (ln.n_comp < 1 || ln.shift == nullptr || ln.weight == nullptr || ln.kind == nullptr) return ME_ERR_NULL;
        if (o + ln.n_comp > ME_MAX_COMP) return ME_ERR_SHAPE;
        if (!(ln.lambda0_A > 0.0) || !(ln.strength >= 0.0f)) return ME_ERR_RANGE;
        me::LineDesc& q = d.line[l];
        q.lam0_over_c = (float)(ln.lambda0_A / C_KMS);
        q.dld_scale = (float)(1e-3 * ln.lambda0_A / ld->lambda_ref_A);
        q.zeeman = (float)(ZEEMAN * ln.lambda0_A * ln.lambda0_A);
        q.strength = ln.strength;
        int cnt[3] = {0, 0, 0};
        for (int kind = -1; kind <= 1; ++kind) {          // sorted [blue | pi | red]
            q.kind_begin[kind + 1] = o;
            for (int c = 0; c < ln.n_comp; ++c) {
                if (ln.kind[c] < -1 || ln.kind[c] > 1) return ME_ERR_RANGE;
                if (ln.kind[c] != kind) continue;
                d.shift[o] = ln.shift[c]; d.weight[o] = ln.weight[c]; ++o; ++cnt[kind + 1];
            }
        }
        q.kind_begin[3] = o;
        const int b = q.kind_begin[0], p = q.kind_begin[1], r = q.kind_begin[2];
        q.triplet = (cnt[0] == 1 && cnt[1] == 1 && cnt[2] == 1 && d.weight[b] == 1.0f && d.weight[p] == 1.0f &&
                     d.weight[r] == 1.0f && d.shift[p] == 0.0f && d.shift[b] == -d.shift[r]) ? 1 : 0;
        q.g = q.triplet ? d.shift[r] : 0.0f;
        q.smax = 0.0f;
        for (int c = q.kind_begin[0]; c < o; ++c) q.smax = std::fmax(q.smax, std::fabs(d.shift[c]));
        if (!q.triplet) d.all_triplets = 0;
        for (int j = 0; j < L; ++j) d.off[l][j] = (float)(lambda[j] - ln.lambda0_A);   // formed in double, rounded once
    }
    d.n_comp = o;
    return ME_OK;
}

// Sobol' direction numbers v_1..v_16 (as 32-bit fixed point) of dimension `dim` (0-based), Bratley & Fox (1988) /
// Antonov & Saleev recurrence on a primitive polynomial of degree s with coefficient bits a and initial values m_1..m_s
// (Joe & Kuo's table for the first 11 dimensions; reading V1).  m_i = xor_k 2^k a_k m_(i-k) xor 2^s m_(i-s) xor m_(i-s).
void sobol_directions16(int dim, uint32_t v[16]) {
    static const int S[11] = {0, 1, 2, 3, 3, 4, 4, 5, 5, 5, 5};
    static const unsigned A[11] = {0, 0, 1, 1, 2, 1, 4, 2, 4, 7, 11};
    static const unsigned M0[11][5] = {{0, 0, 0, 0, 0}, {1, 0, 0, 0, 0}, {1, 3, 0, 0, 0}, {1, 3, 1, 0, 0}, {1, 1, 1, 0, 0},
                                       {1, 1, 3, 3, 0}, {1, 3, 5, 13, 0}, {1, 1, 5, 5, 17}, {1, 1, 5, 5, 5},
                                       {1, 1, 7, 11, 19}, {1, 1, 5, 1, 1}};
    uint32_t m[17];
    const int s = S[dim];
    for (int i = 1; i <= 16; ++i) {
        if (dim == 0) { m[i] = 1; continue; }                 // van der Corput
        if (i <= s) { m[i] = M0[dim][i - 1]; continue; }
        uint32_t x = m[i - s] ^ (m[i - s] << s);
        for (int k = 1; k < s; ++k)
            if ((A[dim] >> (s - 1 - k)) & 1u) x ^= m[i - k] << k;
        m[i] = x;
    }
    for (int i = 1; i <= 16; ++i) v[i - 1] = m[i] << (32 - i);
}

// box_only: the caller is ga_uncertainty or ga_prologue, for which me.h says "the GA fields of cfg are ignored": population,
// generations, tournament, elitism, probabilities and the mutation schedule are neither checked nor used.
int build_ga_desc(const ga_cfg* c, int npar, const float* sigma, int L, uint64_t seed, int64_t N, bool need_sigma,
                  me::GaDesc& g, bool box_only = false) {
    if (c == nullptr) return ME_ERR_NULL;
    if (npar != ME_NPAR && npar != ME_MAX_NPAR) return ME_ERR_SHAPE;
    if (need_sigma && sigma == nullptr) return ME_ERR_NULL;
    if (!box_only) {
        if (c->pop < 2 || c->pop > ME_MAX_POP) return ME_ERR_SHAPE;
        if (c->generations < 0 || c->generations > ME_MAX_GEN) return ME_ERR_SHAPE;
        if (c->tournament_k < 1 || c->tournament_k > 4) return ME_ERR_RANGE;
        if (c->elite != 1) return ME_ERR_UNSUPPORTED;
        if (!(c->p_cross >= 0.f && c->p_cross <= 1.f) || !(c->p_mut >= 0.f && c->p_mut <= 1.f)) return ME_ERR_RANGE;
        if ((c->prologue & 4) && c->pop < 3) return ME_ERR_SHAPE;             // reading S1: the seeds take the last two slots of P0
        if ((c->prologue & 8) && c->pop < 4) return ME_ERR_SHAPE;             // reading S2: the Auer member takes slot P-3
    }
    if (c->variant != 0 && c->variant != 1) return ME_ERR_RANGE;
    if (c->prologue < 0 || c->prologue > 15) return ME_ERR_RANGE;
    if ((c->prologue & 2) && c->log_scale[1]) return ME_ERR_UNSUPPORTED;      // the polarity box is linear in gamma
    if (c->pixel_id_base < 0 || N < 0 || (uint64_t)c->pixel_id_base + (uint64_t)N > 0x100000000ULL) return ME_ERR_RANGE;
    std::memset(&g, 0, sizeof(g));
    g.pop = c->pop; g.generations = c->generations; g.tournament_k = c->tournament_k;
    g.p_cross = c->p_cross; g.p_mut = c->p_mut;
    if (box_only) { g.pop = 3; g.generations = 0; g.tournament_k = 1; g.p_cross = g.p_mut = 0.f; }
    g.key0 = (uint32_t)(seed & 0xffffffffu); g.key1 = (uint32_t)(seed >> 32);
    g.pixel_base = (uint32_t)c->pixel_id_base;
    g.inv_nu = (float)(1.0 / (4.0 * L - npar));          // nu = 4 N_lambda - M
    for (int s = 0; s < 4; ++s) {
        double sg = need_sigma ? (double)sigma[s] : 1.0;
        if (!(sg > 0.0) || !(c->stokes_weight[s] >= 0.f)) return ME_ERR_RANGE;
        double w = (double)c->stokes_weight[s] / sg;
        g.w2[s] = (float)(w * w);
        g.w_cfg[s] = c->stokes_weight[s];
        g.sigma[s] = (float)sg;
    }
    for (int j = 0; j < npar; ++j) {
        if (!(c->lo[j] <= c->hi[j])) return ME_ERR_RANGE;
        g.lo[j] = c->lo[j];
        g.span[j] = (float)((double)c->hi[j] - (double)c->lo[j]);
        g.log_scale[j] = c->log_scale[j] ? 1 : 0;
        g.periodic[j] = c->periodic[j] ? 1 : 0;
        if (g.log_scale[j]) {
            if (!(c->lo[j] > 0.f)) return ME_ERR_RANGE;
            g.log2ratio[j] = (float)std::log2((double)c->hi[j] / (double)c->lo[j]);
        }
    }
    g.prologue = c->prologue;
    g.variant = c->variant;
    g.n_samp = c->generations / 4 > 1 ? c->generations / 4 : 1;
    for (int j = 0; j < ME_MAX_NPAR; ++j) sobol_directions16(j, g.sobol_v[j]);
    if (c->variant == 1 || box_only) return ME_OK;            // the mutation-scale schedule is not used
    if (c->mut_scale_table != nullptr) {
        for (int t = 0; t <= c->generations; ++t) g.mut_scale[t] = c->mut_scale_table[t];
    } else {
        if (!(c->mut_scale0 > 0.f) || !(c->mut_scale_end > 0.f)) return ME_ERR_RANGE;
        const int G = c->generations > 0 ? c->generations : 1;
        for (int t = 0; t <= c->generations; ++t)
            g.mut_scale[t] = (float)((double)c->mut_scale0 * std::pow((double)c->mut_scale_end / (double)c->mut_scale0, (double)t / G));
    }
    return ME_OK;
}

// Reading S1: the line the centre-of-gravity seed is taken on (largest g lambda^2, g = centre of gravity of the sigma_red
// shifts), its window half-width and the wavelength-to-field scale 1 / (2 C g lambda^2).
void fill_seed_desc(const me_line_data* ld, me::GaDesc& g) {
    g.seed_line = 0; g.seed_hw = INFINITY; g.seed_scale = 0.0f;
    double best = -1.0, gbest = 0.0;
    for (int l = 0; l < ld->n_lines; ++l) {
        const me_line& ln = ld->lines[l];
        double geff = 0.0;
        for (int c = 0; c < ln.n_comp; ++c) if (ln.kind[c] == 1) geff += (double)ln.weight[c] * (double)ln.shift[c];
        const double s = geff * ln.lambda0_A * ln.lambda0_A;
        if (s > best) { best = s; g.seed_line = l; gbest = geff; }
    }
    const double l0 = ld->lines[g.seed_line].lambda0_A;
    double hw = INFINITY;
    for (int l = 0; l < ld->n_lines; ++l)
        if (l != g.seed_line) hw = std::fmin(hw, 0.5 * std::fabs(ld->lines[l].lambda0_A - l0));
    g.seed_hw = (float)hw;
    if (gbest > 0.0) g.seed_scale = (float)(1.0 / (2.0 * ZEEMAN * gbest * l0 * l0));
}

}  // namespace

extern "C" {

int me_version(void) { return 110; }

const char* me_last_cuda_error(void) { return g_cuda_err.c_str(); }

const char* me_strerror(int code) {
    switch (code) {
        case ME_OK: return "ok";
        case ME_ERR_NULL: return "a required pointer is NULL";
        case ME_ERR_SHAPE: return "a size is out of range";
        case ME_ERR_RANGE: return "a value is out of range";
        case ME_ERR_UNSUPPORTED: return "not implemented in this build";
        case ME_ERR_CUDA: return "CUDA runtime error (see me_last_cuda_error)";
        case ME_ERR_TOO_LARGE: return "P exceeds me_synth_static_max_vectors(): the library's fixed scratch array cannot hold this batch";
        default: return "unknown error code";
    }
}

size_t me_synth_workspace_bytes(int64_t P) { return me::synth_workspace_bytes(P); }

int me_synth(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
             const me_line_data* line_data, float* out_stokes,
             const float* obs_ref, const float* w_over_sigma, float* out_chi2, void* stream) {
    return me_synth_ws(params, P, mu, lambda_grid_A, L, line_data, out_stokes, obs_ref, w_over_sigma, out_chi2, nullptr, 0, stream);
}

int me_synth_ws(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
                const me_line_data* line_data, float* out_stokes,
                const float* obs_ref, const float* w_over_sigma, float* out_chi2,
                void* workspace, size_t workspace_bytes, void* stream) {
    if (P < 0) return ME_ERR_SHAPE;
    me::SynthDesc sd;
    int rc = build_synth_desc(lambda_grid_A, L, line_data, sd);
    if (rc != ME_OK) return rc;
    if (P == 0) return ME_OK;
    if (out_stokes == nullptr && out_chi2 == nullptr) return ME_ERR_NULL;
    if (out_chi2 != nullptr && (obs_ref == nullptr || w_over_sigma == nullptr)) return ME_ERR_NULL;
    if (params == nullptr) return ME_ERR_NULL;
    float w2[4] = {0, 0, 0, 0};
    if (out_chi2 != nullptr)
        for (int s = 0; s < 4; ++s) {
            if (!(w_over_sigma[s] >= 0.f)) return ME_ERR_RANGE;
            w2[s] = w_over_sigma[s] * w_over_sigma[s];
        }
    cudaError_t e = me::launch_synth(sd, params, mu, P, out_stokes, obs_ref, w2, (float)(1.0 / (4.0 * L - sd.npar)),
                                     out_chi2, workspace, workspace_bytes, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int64_t me_synth_static_max_vectors(void) { return me::synth_static_max_vectors(); }

int me_synth_static(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
                    const me_line_data* line_data, float* out_stokes,
                    const float* obs_ref, const float* w_over_sigma, float* out_chi2, void* stream) {
    if (P < 0) return ME_ERR_SHAPE;
    if (P > me::synth_static_max_vectors()) return ME_ERR_TOO_LARGE;        // before anything touches the device
    void* scratch = nullptr;
    size_t scratch_bytes = 0;
    cudaError_t e = me::synth_static_scratch(&scratch, &scratch_bytes);     // cudaGetSymbolAddress, once per device
    if (e != cudaSuccess) return cuda_fail(e);
    return me_synth_ws(params, P, mu, lambda_grid_A, L, line_data, out_stokes, obs_ref, w_over_sigma, out_chi2, scratch,
                       scratch_bytes, stream);
}

int ga_invert(const float* obs, int64_t N, const uint8_t* mask, const float* sigma,
              const double* lambda_grid_A, int L, const me_line_data* line_data, const ga_cfg* cfg, uint64_t seed,
              float* out_params, float* out_chi2, void* stream) {
    me::SynthDesc sd; me::GaDesc gd;
    int rc = build_synth_desc(lambda_grid_A, L, line_data, sd);
    if (rc != ME_OK) return rc;
    rc = build_ga_desc(cfg, sd.npar, sigma, L, seed, N, true, gd);
    if (rc != ME_OK) return rc;
    fill_seed_desc(line_data, gd);
    if (N == 0) return ME_OK;
    if (obs == nullptr || out_params == nullptr || out_chi2 == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_ga_invert(sd, gd, obs, mask, cfg->mu, N, out_params, out_chi2, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int ga_uncertainty(const float* obs, int64_t N, const uint8_t* mask, const float* sigma, const double* lambda_grid_A, int L,
                   const me_line_data* line_data, const ga_cfg* cfg, const float* params, float* out_sigma, float* out_chi2,
                   void* stream) {
    me::SynthDesc sd; me::GaDesc gd;
    int rc = build_synth_desc(lambda_grid_A, L, line_data, sd);
    if (rc != ME_OK) return rc;
    rc = build_ga_desc(cfg, sd.npar, sigma, L, 0, N, true, gd, true);
    if (rc != ME_OK) return rc;
    if (N == 0) return ME_OK;
    if (obs == nullptr || params == nullptr || out_sigma == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_uncertainty(sd, gd, obs, mask, cfg->mu, N, params, out_sigma, out_chi2, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int ga_fitness(const float* genes, const float* obs, int64_t N, const float* sigma, const double* lambda_grid_A, int L,
               const me_line_data* line_data, const ga_cfg* cfg, float* chi2_out, void* stream) {
    me::SynthDesc sd; me::GaDesc gd;
    int rc = build_synth_desc(lambda_grid_A, L, line_data, sd);
    if (rc != ME_OK) return rc;
    rc = build_ga_desc(cfg, sd.npar, sigma, L, 0, N, true, gd);
    if (rc != ME_OK) return rc;
    if (N == 0) return ME_OK;
    if (genes == nullptr || obs == nullptr || chi2_out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_ga_fitness(sd, gd, genes, obs, cfg->mu, N, chi2_out, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int ga_step(const float* genes_in, const float* chi2_in, int64_t N, int generation, const ga_cfg* cfg, int n_params,
            uint64_t seed, float* genes_out, void* stream) {
    me::GaDesc gd;
    int rc = build_ga_desc(cfg, n_params, nullptr, 4, seed, N, false, gd);
    if (rc != ME_OK) return rc;
    if (generation < 1 || generation > cfg->generations) return ME_ERR_RANGE;
    if (N == 0) return ME_OK;
    if (genes_in == nullptr || chi2_in == nullptr || genes_out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_ga_step(gd, n_params, genes_in, chi2_in, N, generation, genes_out, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int ga_prologue(const float* obs, int64_t N, const float* sigma, const double* lambda_grid_A, int L,
                const me_line_data* line_data, const ga_cfg* cfg, float* out, void* stream) {
    me::SynthDesc sd; me::GaDesc gd;
    int rc = build_synth_desc(lambda_grid_A, L, line_data, sd);
    if (rc != ME_OK) return rc;
    rc = build_ga_desc(cfg, sd.npar, sigma, L, 0, N, true, gd, true);
    if (rc != ME_OK) return rc;
    fill_seed_desc(line_data, gd);
    if (N == 0) return ME_OK;
    if (obs == nullptr || out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_ga_prologue(sd, gd, obs, N, out, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int ga_init(int64_t N, const ga_cfg* cfg, int n_params, uint64_t seed, float* genes_out, void* stream) {
    me::GaDesc gd;
    int rc = build_ga_desc(cfg, n_params, nullptr, 4, seed, N, false, gd);
    if (rc != ME_OK) return rc;
    if (N == 0) return ME_OK;
    if (genes_out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_ga_init(gd, n_params, N, genes_out, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int me_philox_many(uint64_t seed, uint32_t c0_base, uint32_t c1, uint32_t c2, uint32_t c3, int64_t n, uint32_t* out,
                   void* stream) {
    if (n < 0) return ME_ERR_SHAPE;
    if (n == 0) return ME_OK;
    if (out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_philox((uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32), c0_base, c1, c2, c3, n, out,
                                      (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int me_philox(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t out[4]) {
    if (out == nullptr) return ME_ERR_NULL;
    uint32_t* d = nullptr;
    cudaError_t e = cudaMalloc(&d, 16);
    if (e != cudaSuccess) return cuda_fail(e);
    e = me::launch_philox((uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32), c0, c1, c2, c3, 1, d, nullptr);
    if (e == cudaSuccess) e = cudaMemcpy(out, d, 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int me_faddeeva(const float* v, const float* a, int64_t n, float* H, float* F, void* stream) {
    if (n < 0) return ME_ERR_SHAPE;
    if (n == 0) return ME_OK;
    if (v == nullptr || a == nullptr || H == nullptr || F == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_faddeeva(v, a, n, H, F, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

int me_peak_probe(int kind, int iters, int blocks, float* out, void* stream) {
    if (kind < 0 || kind > 10) return ME_ERR_RANGE;
    if (iters < 1 || blocks < 1) return ME_ERR_SHAPE;
    if (out == nullptr) return ME_ERR_NULL;
    cudaError_t e = me::launch_probe(kind, iters, blocks, out, (cudaStream_t)stream);
    return e == cudaSuccess ? ME_OK : cuda_fail(e);
}

// Zeeman pattern in LS coupling: Lande factors, shifts g_l M_l - g_u M_u, dipole strengths per Delta M.
int me_zeeman_pattern(double S_lo, double L_lo, double J_lo, double S_up, double L_up, double J_up,
                      int cap, float* shift, float* weight, int8_t* kind) {
    if (cap > 0 && (shift == nullptr || weight == nullptr || kind == nullptr)) return ME_ERR_NULL;
    const double dJd = J_up - J_lo;
    const int dJ = (int)std::lround(dJd);
    if (J_lo < 0 || J_up < 0 || std::fabs(dJd - dJ) > 1e-9 || dJ < -1 || dJ > 1 || (J_lo == 0 && J_up == 0)) return ME_ERR_RANGE;
    auto lande = [](double S, double L, double J) {
        return J == 0.0 ? 0.0 : 1.5 + (S * (S + 1) - L * (L + 1)) / (2 * J * (J + 1));
    };
    const double gl = lande(S_lo, L_lo, J_lo), gu = lande(S_up, L_up, J_up);
    int n = 0;
    for (int q = 1; q >= -1; --q) {                       // q = M_up - M_lo: +1 -> sigma_blue, 0 -> pi, -1 -> sigma_red
        std::vector<double> sh, st;
        double tot = 0;
        const int nM = (int)std::lround(2 * J_lo) + 1;
        for (int k = 0; k < nM; ++k) {
            const double M = -J_lo + k, Mu = M + q;
            if (std::fabs(Mu) > J_up + 1e-9) continue;
            double s;
            if (dJ == 0)      s = q == 0 ? M * M : (q == 1 ? (J_lo - M) * (J_lo + M + 1) : (J_lo + M) * (J_lo - M + 1));
            else if (dJ == 1) s = q == 0 ? (J_lo + 1) * (J_lo + 1) - M * M : (q == 1 ? (J_lo + M + 1) * (J_lo + M + 2) : (J_lo - M + 1) * (J_lo - M + 2));
            else              s = q == 0 ? J_lo * J_lo - M * M : (q == 1 ? (J_lo - M) * (J_lo - M - 1) : (J_lo + M) * (J_lo + M - 1));
            if (s <= 0) continue;
            sh.push_back(gl * M - gu * Mu); st.push_back(s); tot += s;
        }
        for (size_t c = 0; c < sh.size(); ++c, ++n)
            if (n < cap) { shift[n] = (float)sh[c]; weight[n] = (float)(st[c] / tot); kind[n] = (int8_t)(-q); }
    }
    return n;
}

}  // extern "C"
