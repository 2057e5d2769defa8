/* include/me.h — C ABI of libme_b200.so: GA inversion of Milne-Eddington Stokes profiles on one B200 (sm_100a).
 *
 * The two product calls follow the paper's statement of the problem (Harker & Mighell, arxiv 1208.0302;
 * citations are PAPER.md line numbers + equation):
 *   me_synth   — ME forward synthesis of I,Q,U,V (eq. 7-15) for P parameter vectors, optionally
 *                fused with the chi-square merit (eq. 16) against one fixed profile;
 *   ga_invert  — the per-pixel genetic algorithm of Alg. 1 with the evaluation operator F
 *                (synthesis + eq. 16) fused on-chip; one kernel launch for the whole map.
 * ga_step / ga_fitness / me_philox* are test hooks that expose single stages of ga_invert; me_zeeman_pattern is the
 * once-per-run host precompute of PAPER.md:218.
 *
 * Conventions
 *  - Bulk arrays are DEVICE pointers owned by the caller unless marked "host". Descriptors (me_line_data, ga_cfg,
 *    lambda grid, sigma) are HOST pointers, read during the call and not retained.
 *  - Calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream) and return
 *    without synchronising, except me_philox which synchronises to return host data.
 *  - Return value: ME_OK (0) or a negative me_status. On error nothing is launched and no output is written.
 *    me_strerror(code) returns a static string.
 *  - No global mutable state, no allocation visible to the caller.
 *  - Parameter vector order (BASELINE config 0 order; eq. 14 PAPER.md:211 lists the same quantities as
 *    [B, psi, chi, lambda0, a, dlambdaD, eta0, S0, beta0]):
 *       [0] B (G)  [1] gamma (deg)  [2] chi (deg)  [3] eta0  [4] dlambdaD (mA, quoted at lambda_ref)
 *       [5] a (damping)  [6] v_los (km/s, + = redshift)  [7] S0  [8] S1
 *    Stokes output is in absolute units: continuum = S0 + mu*S1 (eq. 15).
 *  - Arithmetic is FP32 on the device; the wavelength grid is taken in double and converted once, on the host,
 *    to FP32 offsets from each line centre.
 */
#ifndef ME_B200_H
#define ME_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ME_NPAR        9      /* model parameters / genes per individual (base model, eq. 14) */
#define ME_MAX_NPAR    11     /* with fill fraction alpha [9] and stray-light fraction s [10] (n_params = 11) */
#define ME_MAX_LINES   4
#define ME_MAX_COMP    48     /* Zeeman components summed over all lines */
#define ME_MAX_L       512    /* wavelength samples */
#define ME_MAX_POP     1024
#define ME_MAX_GEN     1023   /* generations */

typedef enum {
    ME_OK = 0,
    ME_ERR_NULL = -1,         /* a required pointer is NULL */
    ME_ERR_SHAPE = -2,        /* a size is out of range (L, P, N, pop, n_lines, n_comp ...) */
    ME_ERR_RANGE = -3,        /* a value is out of range (lo > hi, sigma <= 0, log-scaled gene with lo <= 0 ...) */
    ME_ERR_UNSUPPORTED = -4,  /* valid request that this build does not implement (elite != 1) */
    ME_ERR_CUDA = -5,         /* a CUDA runtime call failed; see me_last_cuda_error() */
    ME_ERR_TOO_LARGE = -6     /* me_synth_static: P exceeds me_synth_static_max_vectors() */
} me_status;

/* One spectral line (Table 1). Components are (shift, weight, kind) triples in any order. */
typedef struct {
    double lambda0_A;         /* laboratory centre, Angstrom */
    float strength;           /* eta0 multiplier relative to the reference line (1.0 for it) */
    int n_comp;               /* number of Zeeman components */
    const float* shift;       /* host [n_comp], in Lorentz units (multiples of the Zeeman splitting); > 0 = red */
    const float* weight;      /* host [n_comp], relative strengths; sum to 1 within each kind */
    const int8_t* kind;       /* host [n_comp]: 0 = pi, -1 = sigma_blue, +1 = sigma_red */
} me_line;

typedef struct {
    int n_lines;              /* 1..ME_MAX_LINES */
    const me_line* lines;     /* host [n_lines] */
    double lambda_ref_A;      /* wavelength at which dlambdaD is quoted; dlambdaD_l = dlambdaD * lambda_l / lambda_ref */
    int n_params;             /* 9, or 11: adds [9] alpha = magnetic fill fraction (eq. 19) and
                                 [10] s = stray-light fraction:
                                   I = (1-s) [ alpha I^M(p) + (1-alpha) I(p; B=0) e ] + s I_fixed e   (reading F13) */
    const float* nm_profile;  /* DEVICE [L] f32: I_fixed, the fixed unpolarised profile; required for n_params = 11,
                                 must be NULL for n_params = 9 */
} me_line_data;

/* ME forward synthesis (eq. 12-13, 15) of P parameter vectors on an L-point grid.
 *   params        device [P, n_params] f32   mu          device [P] f32 or NULL (=> 1)
 *   lambda_grid_A host [L] f64 (Angstrom)    out_stokes  device [P, 4, L] f32 or NULL
 *   obs_ref       device [4, L] f32 or NULL  w_over_sigma host [4] f32 (w_s / sigma_s of eq. 16) or NULL
 *   out_chi2      device [P] f32 or NULL: chi2 of each vector against obs_ref, nu = 4L - n_params.
 * At least one of out_stokes / out_chi2 must be given; out_chi2 requires obs_ref and w_over_sigma. P = 0 is a no-op.
 * me_synth allocates nothing: the vectors are visited in index order. */
int me_synth(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
             const me_line_data* line_data, float* out_stokes,
             const float* obs_ref, const float* w_over_sigma, float* out_chi2, void* stream);

/* The same with an optional caller-provided DEVICE workspace ("no allocation visible to the caller
 * except an optional caller-provided workspace").  With workspace_bytes >= me_synth_workspace_bytes(P) (and that size
 * non-zero) the vectors are visited in the order of a counting sort on a coarse key of (dlambdaD, v_los, B), which keeps the
 * lanes of a warp on the same Voigt tiers, and the warps draw their 32-vector tasks from a counter in the workspace instead
 * of a fixed stride; every output stays at its own index and is bit-identical to me_synth's.
 * workspace = NULL or too small: exactly me_synth.  The workspace is scratch: owned by the caller, 16-byte aligned, not
 * read after the work enqueued by this call has run; it may be reused by later calls on the same stream.
 * me_synth_workspace_bytes returns 0 where sorting does not pay (small P) or is not possible (P >= 2^31). */
size_t me_synth_workspace_bytes(int64_t P);
int me_synth_ws(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
                const me_line_data* line_data, float* out_stokes,
                const float* obs_ref, const float* w_over_sigma, float* out_chi2,
                void* workspace, size_t workspace_bytes, void* stream);

/* me_synth_ws for callers that can allocate NOTHING (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): the ordering scratch is a fixed device array inside the library (`static __device__`, 16.1 MiB, held
 * by every GPU that loads the library until the process exits) instead of a caller workspace.  Inputs and outputs are the
 * caller's, with me_synth's meaning, layout and ownership; outputs are bit-identical to me_synth's and me_synth_ws's.
 *   - P <= me_synth_static_max_vectors() (2 097 152); larger batches are refused with ME_ERR_TOO_LARGE before anything is
 *     launched: split them, or use me_synth_ws.  Below 400 000 vectors no scratch is needed and none is touched.
 *   - The call runs no cudaMalloc / cudaFree and no allocating library routine: once per device it asks for the array's
 *     address (cudaGetSymbolAddress, with that device current), then enqueues one cudaMemsetAsync of the 128 KB of histogram
 *     and counters that must start at zero, the two ordering passes and the synthesis on `stream`.
 *   - Every call on a device shares the ONE array, which keeps the previous call's keys and permutation: calls whose work
 *     overlaps on the GPU (different streams, or graphs replayed concurrently) race on it and give wrong results.  Calls on
 *     one stream, or otherwise ordered, are safe. */
int64_t me_synth_static_max_vectors(void);
int me_synth_static(const float* params, int64_t P, const float* mu, const double* lambda_grid_A, int L,
                    const me_line_data* line_data, float* out_stokes,
                    const float* obs_ref, const float* w_over_sigma, float* out_chi2, void* stream);

/* GA configuration (readings G0-G5 in DESIGN.md; the paper leaves the operators' details open). */
typedef struct {
    int pop;                  /* population size, 2..ME_MAX_POP */
    int generations;          /* G >= 0 */
    int tournament_k;         /* 1..4 candidates per tournament */
    int elite;                /* must be 1: slot 0 of every generation is the previous best, not re-evaluated */
    float p_cross;            /* probability of arithmetic crossover, else the child copies parent A */
    float p_mut;              /* per-gene mutation probability */
    float mut_scale0;         /* mutation half-width at t = 0 and t = G, geometric in between:            */
    float mut_scale_end;      /*   s_t = s0 (s_end/s0)^(t/G), built on the host in double, rounded to f32 */
    const float* mut_scale_table; /* host [generations+1] or NULL; if given it replaces the schedule above */
    float lo[ME_MAX_NPAR], hi[ME_MAX_NPAR];  /* per-gene box (eq. 4); lo == hi fixes a gene; the first
                                                n_params entries are used */
    uint8_t log_scale[ME_MAX_NPAR];  /* decode p = lo (hi/lo)^g instead of lo + (hi-lo) g */
    uint8_t periodic[ME_MAX_NPAR];   /* gene wraps (g - floor g) instead of clamping to [0,1] */
    float stokes_weight[4];   /* w_s of eq. 16 (1,4,4,2 in the configs); enters squared */
    const float* mu;          /* device [N] f32 or NULL (=> 1): cosine of the heliocentric angle per pixel */
    int64_t pixel_id_base;    /* added to the pixel index in the RNG key so that shards reproduce the full run */
    int variant;              /* 0: real-coded operators above (tournament, arithmetic crossover, bounded mutation);
                                 1: the paper's own binary-coded GA (readings V0-V5): 16-bit genotype per
                                    parameter decoded by eq. 5, one-point crossover of the
                                    M x 16 bit string, bit mutation favouring less-significant bits
                                    (PAPER.md:103-105), Sobol' initial population and re-seeding of the worst half
                                    every max(1, G/4) generations. mut_scale* are ignored.
                                    In the test hooks a gene then holds its code k in [0, 65535] as a float. */
    int prologue;             /* per-pixel prologue of the paper, bit flags (readings W1, P1):
                                 1: inverse-max weights, eq. 20-23: w_I = 1/(I_c - I_0), w_Q,U,V =
                                    1/max|Q,U,V| from the observed profile (denominators floored at sigma_s) replace
                                    stokes_weight;
                                 2: the inclination box [lo[1], hi[1]] is cut to the polarity given by the order of the
                                    Stokes-V lobes: positive lobe on the blue side => gamma <= 90 deg.
                                 4: two heuristic members replace the last two slots of the initial population
                                    (reading S1): B = |B_los| from the centre of gravity of I +- V
                                    (Rees & Semel 1979) with gamma at the matching end of its box, and the non-magnetic
                                    solution B = lo[0]; other genes as drawn. Needs pop >= 3.
                                 8: the weak-field member "as in Auer et al. (1977)" (reading S2)
                                    takes slot pop-3: B_los from the separation of the I+V and I-V line cores, azimuth
                                    and inclination from the maxima of Q^2+U^2, |V| and the derivatives of I, reflected
                                    into the (polarity-cut) inclination box, B = |B_los| / |cos gamma|. Needs pop >= 4.
                                 ga_fitness ignores these flags (fixed weights, configured box). */
} ga_cfg;

/* GA inversion of N pixels.
 *   obs    device [N, 4, L] f32            mask   device [N] u8 or NULL; 0 => pixel skipped, outputs NaN
 *   sigma  host [4] f32 per-Stokes noise   seed   Philox key
 *   out_params device [N, n_params] f32 (decoded best individual)   out_chi2 device [N] f32 (its chi2, eq. 16)
 * RNG: Philox4x32-10, key = (seed lo, seed hi), counter = (pixel_id_base + n, generation, individual, block).
 * Requires pixel_id_base + N <= 2^32. N = 0 is a no-op. */
int ga_invert(const float* obs, int64_t N, const uint8_t* mask, const float* sigma,
              const double* lambda_grid_A, int L, const me_line_data* line_data, const ga_cfg* cfg, uint64_t seed,
              float* out_params, float* out_chi2, void* stream);

/* Parameter uncertainties at the optimum (eq. 26; reading U1): the Hessian H of chi2 on the
 * box coordinates (central second differences at h = 2^-6 and h/2, one Richardson/Neville level; 1 + 2(2M + 2M(M-1))
 * syntheses per pixel through the same fused fitness as ga_invert), sigma_i^2 = [H^-1]_ii chi2(p_opt)/M, scaled to
 * parameter units. Genes with lo == hi are left out (sigma = 0). A singular or indefinite Hessian gives NaN.
 *   params     device [N, n_params] f32: the optimum (ga_invert's out_params)
 *   out_sigma  device [N, n_params] f32        out_chi2  device [N] f32 or NULL: chi2 at params
 * mask, sigma, cfg (boxes, weights, prologue flags, mu) as for ga_invert; the GA fields of cfg are ignored. */
int ga_uncertainty(const float* obs, int64_t N, const uint8_t* mask, const float* sigma, const double* lambda_grid_A, int L,
                   const me_line_data* line_data, const ga_cfg* cfg, const float* params, float* out_sigma, float* out_chi2,
                   void* stream);

/* Test hooks (not timed). */
/* One generation t >= 1 of selection/crossover/mutation/elitism from given genes and given fitness. */
int ga_step(const float* genes_in /*[N,pop,n_params]*/, const float* chi2_in /*[N,pop]*/, int64_t N, int generation,
            const ga_cfg* cfg, int n_params, uint64_t seed, float* genes_out /*[N,pop,n_params]*/, void* stream);
/* The fused fitness alone: decode -> synthesis -> chi2 for every individual of every pixel. */
int ga_fitness(const float* genes /*[N,pop,n_params]*/, const float* obs /*[N,4,L]*/, int64_t N, const float* sigma /*host[4]*/,
               const double* lambda_grid_A, int L, const me_line_data* line_data, const ga_cfg* cfg,
               float* chi2_out /*[N,pop]*/, void* stream);
/* The per-pixel prologue alone: out device [N,12] f32 = w_I, w_Q, w_U, w_V, gamma_lo, gamma_hi as ga_invert uses them,
 * then B_los [G] and the stored genes (B, gamma) of the centre-of-gravity member (0 unless prologue bit 4), then the stored
 * genes (B, gamma, chi) of the Auer weak-field member (0 unless prologue bit 8).  Allocates nothing, does not synchronise. */
int ga_prologue(const float* obs /*[N,4,L]*/, int64_t N, const float* sigma /*host[4]*/, const double* lambda_grid_A, int L,
                const me_line_data* line_data, const ga_cfg* cfg, float* out, void* stream);
/* Generation-0 population (reading G2): genes_out device [N,pop,n_params]. */
int ga_init(int64_t N, const ga_cfg* cfg, int n_params, uint64_t seed, float* genes_out, void* stream);
/* One Philox4x32-10 block computed ON THE DEVICE; out is a HOST pointer; synchronises. */
int me_philox(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t out[4]);
/* n blocks with counters (c0_base + i, c1, c2, c3): out device [n,4] u32. */
int me_philox_many(uint64_t seed, uint32_t c0_base, uint32_t c1, uint32_t c2, uint32_t c3, int64_t n,
                   uint32_t* out, void* stream);
/* Device Faddeeva evaluator alone: w(v + i a) -> (H, F), all device [n] f32. */
int me_faddeeva(const float* v, const float* a, int64_t n, float* H, float* F, void* stream);

/* Instruction-throughput probe for the roofline denominators (SURVEY.md par. 8(d)): launches `blocks` CTAs of 256
 * threads, each thread running `iters` x 32 slots of one instruction class in 8 independent register chains.
 * kind: 0 FFMA (scalar), 1 FFMA2 (packed fp32x2, the form the fitness loop is written in), 3 MUFU.RCP/EX2; any other
 *       value is ME_ERR_CUDA (invalid value).
 * out: device [blocks*256] f32 scratch (never written in practice). The caller times the call with CUDA events. */
int me_peak_probe(int kind, int iters, int blocks, float* out, void* stream);

/* Host-only: Zeeman pattern of an LS-coupling transition, lower/upper = (S, L, J).
 * Fills up to cap entries and returns the number of components (> cap means truncated), or a negative me_status. */
int me_zeeman_pattern(double S_lo, double L_lo, double J_lo, double S_up, double L_up, double J_up,
                      int cap, float* shift, float* weight, int8_t* kind);

const char* me_strerror(int code);
const char* me_last_cuda_error(void);   /* text of the last CUDA failure seen by this thread ("" if none) */
int me_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ME_B200_H */
