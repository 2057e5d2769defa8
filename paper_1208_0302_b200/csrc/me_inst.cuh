// me_inst.cuh — the heavy template kernels (fused GA inversion, fused fitness hook, forward synthesis) and their
// per-(NL, TRIPLET) launchers.  Included by me_inst_<nl>_<t>.cu with ME_INST_NL / ME_INST_TRIPLET defined, so that the
// specialisations compile in parallel translation units.
#pragma once
#include "me_device.cuh"
#include "me_launch.h"

namespace me {

// ------------------------------------------------------------------------------------------------------------
// Fitness of one individual held in registers: decode -> per-individual constants -> wavelength loop.
// obs_s: shared memory, per wavelength pair two float4 = (I0,I1,Q0,Q1), (U0,U1,V0,V1) (broadcast reads, conflict-free).
// nm_s:  shared memory, per wavelength pair one float2 of I_fixed (M = 11 only).
// ------------------------------------------------------------------------------------------------------------
// far_s != nullptr (FARS): [ME_FAR_ROWS NL][far_stride] float4 of shared memory, this thread's column.
// off_s != nullptr: the offsets lambda_j - lambda_l staged pair-wise in shared memory, off_s[jp * NL + l] = (off[l][2jp],
// off[l][2jp+1]), with one padding pair at the end (stage_offsets); else they are read from the constant bank.
template <int NL, bool TRIPLET, int M, bool FARS = false>
__device__ __forceinline__ float fitness_params(const float* p, float mu, const SynthDesc& sd, const GaDesc& gd,
                                                const float4* obs_s, const float2* nm_s, const float* pix,
                                                float4* far_s = nullptr, int far_stride = 0, const f2* off_s = nullptr) {
    Individual<NL> ind;
    setup_individual<NL, M>(ind, p, mu, sd, TRIPLET);
    ind.far_addr = 0; ind.far_stride = 16 * far_stride;
    if (FARS) {
#pragma unroll
        for (int l = 0; l < NL; ++l) far_store(far_s + ME_FAR_ROWS * l * far_stride, far_stride, ind.far[l]);
        ind.far_addr = (unsigned)__cvta_generic_to_shared(far_s);
        keep_in_register(ind.far_addr);          // else S2R + LEA + moves are re-issued in every far-tier branch (r2c)
    }
    f2 aI = bc(0.f), aQ = bc(0.f), aU = bc(0.f), aV = bc(0.f);
    const int L = sd.L, npair = L >> 1;
    // the offsets lambda_j - lambda_l of the NEXT pair are loaded one iteration ahead: the load otherwise stalls the first
    // FFMA2 of every line (profiles/r1_history.md, step r1e).  From shared memory this is one LDS.128 per pair for two lines, and the padding
    // pair makes the look-ahead of the last iteration a valid read (r2c: the constant-bank form cost 2 LDC + 2 index
    // instructions per wavelength point).
    f2 offn[NL];
#pragma unroll
    for (int l = 0; l < NL; ++l) offn[l] = off_s != nullptr ? off_s[l] : *reinterpret_cast<const f2*>(&sd.off[l][0]);
    for (int jp = 0; jp < npair; ++jp) {
        f2 I, Q, U, V, vc[NL];
        // The reduced wavelengths of BOTH lines are formed at the top, which is the last use of this pair's offsets, so the
        // look-ahead load below lands in the same registers: carried as (current, next) copies the rotation cost 6 MOV per pair
        // (r2l SASS; in pairs where both lines are in the far tier the issue slots, not the FMA pipe, are what is short).
#pragma unroll
        for (int l = 0; l < NL; ++l) vc[l] = fma2(ind.invD[l], offn[l], ind.v0[l]);
        if (off_s != nullptr) {
            if (NL == 2) {
                const float4 o = *reinterpret_cast<const float4*>(off_s + 2 * (jp + 1));
                offn[0] = make_float2(o.x, o.y); offn[NL - 1] = make_float2(o.z, o.w);
            } else {
#pragma unroll
                for (int l = 0; l < NL; ++l) offn[l] = off_s[(jp + 1) * NL + l];
            }
        } else {
            const int jn = 2 * min(jp + 1, npair - 1);
#pragma unroll
            for (int l = 0; l < NL; ++l) offn[l] = *reinterpret_cast<const f2*>(&sd.off[l][jn]);
        }
        const float4 o0 = obs_s[2 * jp], o1 = obs_s[2 * jp + 1];           // (I0,I1,Q0,Q1), (U0,U1,V0,V1)
        I = make_float2(o0.x, o0.y); Q = make_float2(o0.z, o0.w); U = make_float2(o1.x, o1.y); V = make_float2(o1.z, o1.w);
        // observed in, residuals observed - model out (stokes_pair RES mode)
        stokes_pair<NL, TRIPLET, M, FARS, true>(ind, sd, 2 * jp, false, M == ME_MAX_NPAR ? nm_s[jp] : bc(0.f), I, Q, U, V, nullptr, vc);
        aI = fma2(I, I, aI); aQ = fma2(Q, Q, aQ); aU = fma2(U, U, aU); aV = fma2(V, V, aV);
    }
    if (L & 1) {                                                            // odd tail: second half is a duplicate, dropped
        f2 I, Q, U, V;
        stokes_pair<NL, TRIPLET, M, FARS>(ind, sd, L - 1, true, M == ME_MAX_NPAR ? nm_s[npair] : bc(0.f), I, Q, U, V);
        const float4 o0 = obs_s[2 * npair], o1 = obs_s[2 * npair + 1];
        const float dI = o0.x - I.x, dQ = o0.z - Q.x, dU = o1.x - U.x, dV = o1.z - V.x;
        aI.x = fmaf(dI, dI, aI.x); aQ.x = fmaf(dQ, dQ, aQ.x); aU.x = fmaf(dU, dU, aU.x); aV.x = fmaf(dV, dV, aV.x);
    }
    const float sI = aI.x + aI.y, sQ = aQ.x + aQ.y, sU = aU.x + aU.y, sV = aV.x + aV.y;
    const volatile float* pw = pix;      // per-pixel (w_s/sigma_s)^2, read HERE (volatile: not hoisted above the loop, where it would cost 4 registers)
    float chi2 = gd.inv_nu * fmaf(pw[0], sI, fmaf(pw[1], sQ, fmaf(pw[2], sU, pw[3] * sV)));
    if (!(chi2 < __int_as_float(0x7f800000))) chi2 = __int_as_float(0x7f800000);   // NaN / Inf -> +Inf (reading G4)
    return chi2;
}

// Fitness of one individual held in registers as genes: decode (readings G1 / V0; inclination on the per-pixel box,
// reading P1) -> fitness_params.
template <int NL, bool TRIPLET, int M, bool FARS = false>
__device__ __forceinline__ float fitness(const float* g, float mu, const SynthDesc& sd, const GaDesc& gd,
                                         const float4* obs_s, const float2* nm_s, const float* pix,
                                         float4* far_s = nullptr, int far_stride = 0, const f2* off_s = nullptr) {
    float p[M];
#pragma unroll
    for (int j = 0; j < M; ++j) p[j] = decode_gene(gene_value(g[j], gd), gd, j);
    if (!gd.log_scale[1]) p[1] = fmaf(pix[5], gene_value(g[1], gd), pix[4]);   // inclination: per-pixel box (reading P1)
    return fitness_params<NL, TRIPLET, M, FARS>(p, mu, sd, gd, obs_s, nm_s, pix, far_s, far_stride, off_s);
}

// Stage I_fixed[L] pair-wise: nm_s[jp] = (F[2jp], F[2jp+1]); the odd tail duplicates its single value.
__device__ __forceinline__ void stage_nm(float2* nm_s, const float* nm, int L, int tid, int nthreads) {
    for (int jp = tid; jp < (L + 1) / 2; jp += nthreads) {
        const float a = __ldg(nm + 2 * jp), b = 2 * jp + 1 < L ? __ldg(nm + 2 * jp + 1) : a;
        nm_s[jp] = make_float2(a, b);
    }
}

// Stage the wavelength offsets pair-wise: off_s[jp * NL + l] = (off[l][2 jp], off[l][2 jp + 1]) for jp < L / 2, plus one padding
// pair (a copy of the last) that the loop's look-ahead reads.  Same for every pixel: once per CTA.  16-byte aligned for NL = 2.
template <int NL>
__device__ __forceinline__ void stage_offsets(f2* off_s, const SynthDesc& sd, int tid, int nthreads) {
    const int npair = sd.L >> 1;
    for (int k = tid; k < (npair + 1) * NL; k += nthreads) {
        const int jp = min(k / NL, max(npair - 1, 0)), l = k % NL;
        off_s[k] = (NL == ME_MAX_LINES && l >= sd.n_lines) ? make_float2(0.f, 0.f)
                                                            : make_float2(sd.off[l][2 * jp], sd.off[l][2 * jp + 1]);
    }
}

// ------------------------------------------------------------------------------------------------------------
// The fused GA inversion kernel.
// Dynamic shared memory: scratch [64] | pix [ME_PIX_WORDS] (per-pixel weights and inclination box) | far [ME_FAR_ROWS NL][THREADS] float4
//                        (far-tier coefficients of every thread) | obs_s [ceil(L/2)] 2 x float4 | off_s [(L/2 + 1) NL] float2
//                        (wavelength offsets, pair-wise) | nm_s [ceil(L/2)] float2 | genes [2][pop][M] | chi2 [2][pop] |
//                        order [pop] u16 (variant 1: ranks at restarts)
// ------------------------------------------------------------------------------------------------------------
template <int NL, bool TRIPLET, int M, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
ga_invert_kernel(const __grid_constant__ SynthDesc sd, const __grid_constant__ GaDesc gd,
                 const float* __restrict__ obs, const uint8_t* __restrict__ mask, const float* __restrict__ mu_arr,
                 int64_t N, float* __restrict__ out_params, float* __restrict__ out_chi2) {
    extern __shared__ float4 smem4[];
    const int L = sd.L, pop = gd.pop;
    // fixed offsets first (compile-time shared addresses, no pointer registers): scratch [64] | pix [8] | obs_s ...
    uint32_t* scratch = reinterpret_cast<uint32_t*>(smem4);
    float* pix_s = reinterpret_cast<float*>(scratch + 64);
    constexpr bool FARS = TRIPLET && NL <= 2;                  // far-tier coefficients parked in shared memory
    float4* far_s = reinterpret_cast<float4*>(pix_s + ME_PIX_WORDS) + threadIdx.x;   // [ME_FAR_ROWS NL][THREADS] float4, own column
    float* obs_s = reinterpret_cast<float*>(far_s - threadIdx.x + (FARS ? ME_FAR_ROWS * NL * THREADS : 0));
    f2* off_s = reinterpret_cast<f2*>(obs_s + 8 * ((L + 1) >> 1));                     // [(L/2 + 1) NL] float2, 16-byte aligned
    float2* nm_s = reinterpret_cast<float2*>(off_s + ((L >> 1) + 1) * NL);
    float* genes_s = reinterpret_cast<float*>(nm_s + ((L + 1) >> 1));
    float* chi2_s = genes_s + 2 * pop * M;
    uint16_t* order_s = reinterpret_cast<uint16_t*>(chi2_s + 2 * pop);
    if (M == ME_MAX_NPAR) stage_nm(nm_s, sd.nm_profile, L, threadIdx.x, THREADS);     // once per CTA; synced below
    stage_offsets<NL>(off_s, sd, threadIdx.x, THREADS);                                // once per CTA; synced below
    const int tid = threadIdx.x;
    const float INF = __int_as_float(0x7f800000);

    for (int64_t n = blockIdx.x; n < N; n += gridDim.x) {
        if (mask != nullptr && mask[n] == 0) {
            const float qnan = __int_as_float(0x7fc00000);
            if (tid < M) out_params[n * M + tid] = qnan;
            if (tid == 0) out_chi2[n] = qnan;
            continue;
        }
        const uint32_t pixel = gd.pixel_base + (uint32_t)n;
        const float mu = mu_arr != nullptr ? __ldg(mu_arr + n) : 1.0f;
        __syncthreads();                                   // previous pixel's shared memory is no longer read
        stage_obs(obs_s, obs + n * 4 * (int64_t)L, L, tid, THREADS);
        __syncthreads();
        pixel_prologue(obs_s, L, gd, pix_s, tid == 0, sd.off[gd.seed_line]);   // every warp reduces, thread 0 writes; visible after the next barrier
        if (gd.prologue & 8) pixel_seed_auer(obs_s, L, gd, pix_s, tid == 0, sd.off[gd.seed_line]);   // reading S2

        // generations 0..G with ONE fitness call site (keeps the loop body inside the instruction cache)
        float g[M];
        float f = INF;
        int cur = 1;                                       // generation t reads buffer cur, writes cur ^ 1
        const bool alive = tid < pop;
        for (int t = 0; t <= gd.generations; ++t) {
            float fe = INF; int ie = 0;
            if (t > 0) block_argmin(f, tid, scratch, fe, ie);   // elite of generation t-1
            else __syncthreads();                          // obs staged
            const float* gprev = genes_s + cur * pop * M;
            const float* fprev = chi2_s + cur * pop;
            float* gnext = genes_s + (cur ^ 1) * pop * M;
            // variant 1, restart generation (reading V2): rank the previous generation; the worst half is dead
            const bool restart = gd.variant != 0 && t > 0 && t < gd.generations && (t % gd.n_samp) == 0;
            if (restart) {
                if (alive) order_s[rank_of(fprev, pop, tid)] = (uint16_t)tid;
                __syncthreads();
            }
            if (alive) {
                bool evaluate = true;
                if (t == 0) {
                    if (gd.variant) sobol_genes<M>(g, pixel, (uint32_t)tid + 1u, gd);  // reading V1
                    else init_genes<M>(g, pixel, (uint32_t)tid, gd);                  // reading G2
                    if ((gd.prologue & 4) && pop >= 3) {                              // reading S1: heuristic members of P0
                        if (tid == pop - 1) g[0] = 0.0f;                              // the non-magnetic solution
                        if (tid == pop - 2) { g[0] = pix_s[7]; g[1] = pix_s[8]; }     // centre-of-gravity longitudinal field
                    }
                    if ((gd.prologue & 8) && pop >= 4 && tid == pop - 3) {            // reading S2: the Auer weak-field member
                        g[0] = pix_s[10]; g[1] = pix_s[11]; g[2] = pix_s[12];
                    }
                } else if (tid == 0) {
#pragma unroll
                    for (int j = 0; j < M; ++j) g[j] = gprev[ie * M + j];
                    f = fe;                                // carried, not re-evaluated (reading G3)
                    evaluate = false;
                } else if (gd.variant) {
                    make_child_binary<M>(g, gprev, fprev, restart ? order_s : nullptr, restart ? pop - pop / 2 : pop, pixel,
                                         (uint32_t)t, (uint32_t)tid, gd);
                } else {
                    make_child<M>(g, gprev, fprev, pixel, (uint32_t)t, (uint32_t)tid, gd.mut_scale[t], gd);
                }
                // the genes go to the next buffer BEFORE the fitness call: nothing reads that buffer until the barrier below, and
                // the M registers are then free inside the wavelength loop (the far-tier loads are asm with a memory clobber,
                // across which the compiler does not move this store by itself)
#pragma unroll
                for (int j = 0; j < M; ++j) gnext[tid * M + j] = g[j];
                if (evaluate) f = fitness<NL, TRIPLET, M, FARS>(g, mu, sd, gd, reinterpret_cast<const float4*>(obs_s), nm_s, pix_s, far_s, THREADS, off_s);
                chi2_s[(cur ^ 1) * pop + tid] = f;
            }
            cur ^= 1;
            __syncthreads();
        }

        float fe; int ie;
        block_argmin(f, tid, scratch, fe, ie);             // reading G5
        if (tid == ie) {
            const float* gfin = genes_s + cur * pop * M + tid * M;     // the last generation's buffer (cur was flipped after it)
#pragma unroll
            for (int j = 0; j < M; ++j) out_params[n * M + j] = decode_gene(gene_value(gfin[j], gd), gd, j);
            if (!gd.log_scale[1]) out_params[n * M + 1] = fmaf(pix_s[5], gene_value(gfin[1], gd), pix_s[4]);
            out_chi2[n] = f;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// me_synth: thread = parameter vector (as in the GA kernel: the lanes of a warp sit at the SAME wavelength, so the
// Voigt tier branches stay mostly warp-uniform), serial loop over wavelength pairs.  out_stokes[P,4,L] is written
// through a warp-private shared-memory tile: every SYNTH_CW wavelengths the warp transposes its 32 vectors x 4 Stokes
// rows and streams them out as 64-byte row segments (two per store instruction, full 32-byte sectors).
// chi2 (optional) accumulates in registers as in the fused fitness.
// Tile: [32 vectors][4 * SYNTH_CW + 4] floats per warp; rows are read back as float4 (8 rows = 512 B per store
// instruction) when L % 4 == 0, else element-wise.
// ------------------------------------------------------------------------------------------------------------
#define SYNTH_CW 16
#define SYNTH_VS (4 * SYNTH_CW + 4)      /* row stride: 16-byte aligned rows for LDS.128 / STG.128 */
#define SYNTH_THREADS 128

// OUT: out_stokes is written (plain tail, transpose tile); !OUT: chi2 only (residual tail, no tile).  One tail per instantiation:
// with both inlined behind a run-time flag the 11-parameter and 4-line variants spilled.
template <int NL, bool TRIPLET, int M, bool OUT>
__global__ void __launch_bounds__(SYNTH_THREADS, (!OUT && NL <= 2) ? 5 : 4)    // chi2 only: no transpose tile, 15 KB of shared memory, 5 CTAs per SM (the run-time-sized NL = 4 form would spill 1 KB)
me_synth_kernel(const __grid_constant__ SynthDesc sd, const float* __restrict__ params, const float* __restrict__ mu_arr,
                const int* __restrict__ perm, int* __restrict__ task_counter, int64_t P, float* __restrict__ out_stokes,
                const float* __restrict__ obs_ref, float w2I, float w2Q, float w2U, float w2V, float inv_nu,
                float* __restrict__ out_chi2) {
    extern __shared__ float4 smem4[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* tile = reinterpret_cast<float*>(smem4) + warp * (32 * SYNTH_VS);
    const int L = sd.L, npair = L >> 1;
    // as in the GA kernel (r2c: this kernel still rematerialised the far-tier coefficients with scalar FMULs, 4.4 per
    // wavelength point against 1.8, and read the offsets with two constant loads per point): coefficients parked in shared
    // memory, one column per thread, and the wavelength offsets staged pair-wise once per CTA
    constexpr bool FARS = TRIPLET && NL <= 2;
    float4* far_s = smem4 + (OUT ? (SYNTH_THREADS / 32) * 32 * SYNTH_VS / 4 : 0) + threadIdx.x;        // [ME_FAR_ROWS NL][SYNTH_THREADS] float4, own column
    // ref_s: obs_ref staged like the GA kernel's observation (per pair two float4: (I0,I1,Q0,Q1), (U0,U1,V0,V1)); the chi2 leg
    // read it with eight scalar global loads per pair before (r2c)
    float* ref_s = reinterpret_cast<float*>(far_s - threadIdx.x + (FARS ? ME_FAR_ROWS * NL * SYNTH_THREADS : 0));   // [ceil(L/2)] 2 x float4
    f2* off_s = reinterpret_cast<f2*>(ref_s + 8 * ((L + 1) >> 1));                                         // [(L/2 + 1) NL] float2
    constexpr bool want_out = OUT;
    const bool want_chi2 = out_chi2 != nullptr;
    stage_offsets<NL>(off_s, sd, threadIdx.x, SYNTH_THREADS);
    if (want_chi2) stage_obs(ref_s, obs_ref, L, threadIdx.x, SYNTH_THREADS);
    __syncthreads();
    const float4* ref4 = reinterpret_cast<const float4*>(ref_s);
    // A task = 32 consecutive slots of the processing order, one warp.  Warps share nothing after the staging above, so with
    // a task counter (the ordered visit of large batches) every warp pulls its next task when it is done with the last one:
    // r2l's static grid-stride left 18 % of the resident warp slots empty (sm__warps_active 13.2 of 16: 13.2 passes per CTA
    // at P = 1e6, so a fifth of the CTAs ran a 14th while the others idled, and the cost per task follows the sort key).
    // Tasks are handed out from the END of the order: the key's leading field is the Doppler width, and wide lines (more
    // wavelengths in the core tier) are the expensive ones, so the longest tasks start first.
    const int64_t ntask = (P + 31) >> 5;
    int64_t task = (int64_t)blockIdx.x * (SYNTH_THREADS / 32) + warp;
    for (;; task += (int64_t)gridDim.x * (SYNTH_THREADS / 32)) {
        if (task_counter != nullptr) {
            int t = 0;
            if (lane == 0) t = atomicAdd(task_counter, 1);
            task = __shfl_sync(0xffffffffu, t, 0);
        }
        if (task >= ntask) break;
        const int64_t wbase = (task_counter != nullptr ? ntask - 1 - task : task) << 5;   // first slot of this warp
        const int64_t slot = wbase + lane < P ? wbase + lane : P - 1;   // idle lanes recompute the last vector, never store
        const int64_t v = perm != nullptr ? (int64_t)__ldg(perm + slot) : slot;   // processing order -> vector (synth_order_kernel)
        float p[M];
#pragma unroll
        for (int j = 0; j < M; ++j) p[j] = __ldg(params + v * M + j);
        const float mu = mu_arr != nullptr ? __ldg(mu_arr + v) : 1.0f;
        Individual<NL> ind;
        setup_individual<NL, M>(ind, p, mu, sd, TRIPLET);
        ind.far_addr = 0; ind.far_stride = 16 * SYNTH_THREADS;
        if (FARS) {
#pragma unroll
            for (int l = 0; l < NL; ++l) far_store(far_s + ME_FAR_ROWS * l * SYNTH_THREADS, SYNTH_THREADS, ind.far[l]);
            ind.far_addr = (unsigned)__cvta_generic_to_shared(far_s);
            keep_in_register(ind.far_addr);
        }
        const float* nm = sd.nm_profile;
        f2 aI = bc(0.f), aQ = bc(0.f), aU = bc(0.f), aV = bc(0.f);
        for (int jp0 = 0; jp0 < npair; jp0 += SYNTH_CW / 2) {
            const int nloc = min(SYNTH_CW / 2, npair - jp0);
            for (int i = 0; i < nloc; ++i) {
                const int j = 2 * (jp0 + i);
                f2 I, Q, U, V;
                const f2 nmF = M == ME_MAX_NPAR ? make_float2(__ldg(nm + j), __ldg(nm + j + 1)) : bc(0.f);
                // more than two lines (the run-time-sized fallback) sits at the register limit: it keeps the round-1 form of the
                // offsets, read from the constant bank (the staged form spilled there)
                constexpr bool LEAN = NL > 2;
                f2 offc[LEAN ? 1 : NL];
                if constexpr (!LEAN) {
#pragma unroll
                    for (int l = 0; l < NL; ++l) offc[l] = off_s[(jp0 + i) * NL + l];
                }
                const f2* offp = LEAN ? nullptr : offc;
                if constexpr (!OUT) {                                    // chi2 only: residuals straight out of the tail's FMAs
                    const float4 o0 = ref4[2 * (jp0 + i)], o1 = ref4[2 * (jp0 + i) + 1];
                    I = make_float2(o0.x, o0.y); Q = make_float2(o0.z, o0.w); U = make_float2(o1.x, o1.y); V = make_float2(o1.z, o1.w);
                    stokes_pair<NL, TRIPLET, M, FARS, true>(ind, sd, j, false, nmF, I, Q, U, V, offp);
                    aI = fma2(I, I, aI); aQ = fma2(Q, Q, aQ); aU = fma2(U, U, aU); aV = fma2(V, V, aV);
                    continue;
                } else {
                stokes_pair<NL, TRIPLET, M, FARS>(ind, sd, j, false, nmF, I, Q, U, V, offp);
                {
                    float2* t = reinterpret_cast<float2*>(tile + lane * SYNTH_VS + 2 * i);
                    t[0] = I; t[SYNTH_CW / 2] = Q; t[SYNTH_CW] = U; t[3 * SYNTH_CW / 2] = V;
                }
                if (want_chi2) {
                    const float4 o0 = ref4[2 * (jp0 + i)], o1 = ref4[2 * (jp0 + i) + 1];
                    const f2 dI = sub2(make_float2(o0.x, o0.y), I), dQ = sub2(make_float2(o0.z, o0.w), Q);
                    const f2 dU = sub2(make_float2(o1.x, o1.y), U), dV = sub2(make_float2(o1.z, o1.w), V);
                    aI = fma2(dI, dI, aI); aQ = fma2(dQ, dQ, aQ); aU = fma2(dU, dU, aU); aV = fma2(dV, dV, aV);
                }
                }
            }
            if (want_out) {
                __syncwarp();
                const int ncol = 2 * nloc;
                const int64_t nvec = P - wbase < 32 ? P - wbase : 32;
                if ((L & 3) == 0 && nloc == SYNTH_CW / 2 && nvec == 32 && P <= 0xffffffffLL) {
                    // Full tile (all but the last task and a ragged last chunk): lane -> (Stokes row st, column group q) is
                    // fixed, only the vector 2 it + (lane >> 4) moves with the iteration, so a store is SHFL (32-bit vector
                    // index), one IMAD.WIDE for the address, LDS.128 at an immediate offset, STG.128.  The general loop
                    // below spent 28 instructions per store on 64-bit index arithmetic and predicates (r2r: a quarter
                    // of the warp instructions of this instantiation).
                    const int st = (lane >> 2) & 3, q = 4 * (lane & 3), hi = lane >> 4;
                    const float* trow = tile + hi * SYNTH_VS + st * SYNTH_CW + q;
                    char* obase = reinterpret_cast<char*>(out_stokes + (int64_t)st * L + 2 * jp0 + q);
                    const unsigned vbytes = 16u * (unsigned)L;                    // bytes per vector: 4 L floats
                    const unsigned v32 = (unsigned)v;
#pragma unroll
                    for (int it = 0; it < 16; ++it) {
                        const unsigned vv = __shfl_sync(0xffffffffu, v32, 2 * it + hi);
                        __stcs(reinterpret_cast<float4*>(obase + (uint64_t)vv * vbytes),
                               *reinterpret_cast<const float4*>(trow + 2 * it * SYNTH_VS));
                    }
                } else if ((L & 3) == 0) {                           // 16-byte aligned rows: 8 rows per store instruction
                    const int q = 4 * (lane & 3);
#pragma unroll 4
                    for (int it = 0; it < 16; ++it) {
                        const int row = 8 * it + (lane >> 2), lv = row >> 2, st = row & 3;
                        const int64_t vv = __shfl_sync(0xffffffffu, v, lv);
                        if (lv < nvec && q < ncol)
                            __stcs(reinterpret_cast<float4*>(out_stokes + (vv * 4 + st) * (int64_t)L + 2 * jp0 + q),
                                   *reinterpret_cast<const float4*>(tile + lv * SYNTH_VS + st * SYNTH_CW + q));
                    }
                } else {
                    const int k = lane & 15;
#pragma unroll 4
                    for (int it = 0; it < 64; ++it) {
                        const int row = 2 * it + (lane >> 4), lv = row >> 2, st = row & 3;
                        const int64_t vv = __shfl_sync(0xffffffffu, v, lv);
                        if (lv < nvec && k < ncol)
                            __stcs(out_stokes + (vv * 4 + st) * (int64_t)L + 2 * jp0 + k, tile[lv * SYNTH_VS + st * SYNTH_CW + k]);
                    }
                }
                __syncwarp();
            }
        }
        if (L & 1) {                                             // odd tail: one wavelength, written directly
            f2 I, Q, U, V;
            stokes_pair<NL, TRIPLET, M, FARS>(ind, sd, L - 1, true, M == ME_MAX_NPAR ? bc(__ldg(nm + L - 1)) : bc(0.f), I, Q, U, V);
            if (want_out && wbase + lane < P) {
                float* o = out_stokes + v * 4 * (int64_t)L + (L - 1);
                __stcs(o, I.x); __stcs(o + L, Q.x); __stcs(o + 2 * L, U.x); __stcs(o + 3 * L, V.x);
            }
            if (want_chi2) {
                const float dI = __ldg(obs_ref + L - 1) - I.x, dQ = __ldg(obs_ref + 2 * L - 1) - Q.x;
                const float dU = __ldg(obs_ref + 3 * L - 1) - U.x, dV = __ldg(obs_ref + 4 * L - 1) - V.x;
                aI.x = fmaf(dI, dI, aI.x); aQ.x = fmaf(dQ, dQ, aQ.x); aU.x = fmaf(dU, dU, aU.x); aV.x = fmaf(dV, dV, aV.x);
            }
        }
        if (want_chi2 && wbase + lane < P) {
            const float sI = aI.x + aI.y, sQ = aQ.x + aQ.y, sU = aU.x + aU.y, sV = aV.x + aV.y;
            out_chi2[v] = inv_nu * fmaf(w2I, sI, fmaf(w2Q, sQ, fmaf(w2U, sU, w2V * sV)));
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// ga_uncertainty: sigma of every parameter from the curvature of chi2 at the optimum (eq. 26; reading
// U1 of DESIGN.md).  CTA = pixel.  The 1 + 2 (2M + 2M(M-1)) chi2 evaluations (325 for M = 9) of the central second
// differences at h = 2^-6 and h/2 are spread over the block and run through the same fused fitness as the GA; thread 0
// then builds the Richardson-extrapolated Hessian and inverts it in FP64 (Gauss-Jordan, partial pivoting; M <= 11).
// Dynamic shared memory: scratch [64] | pix [8] | obs_s | nm_s | chi2v [n_eval]
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ int unc_n_eval(int M) { return 1 + 2 * (2 * M + 2 * M * (M - 1)); }

// offsets of evaluation e (same list as the specification): returns the step and the (at most two) displaced coordinates
__device__ __forceinline__ void unc_offsets(int M, int e, float h, int& j, float& dj, int& k, float& dk) {
    j = k = -1; dj = dk = 0.f;
    if (e == 0) return;
    const int per_level = 2 * M + 2 * M * (M - 1);
    int r = e - 1;
    const int level = r / per_level;
    r -= level * per_level;
    const float hl = level == 0 ? h : 0.5f * h;
    if (r < 2 * M) { j = r >> 1; dj = (r & 1) ? -hl : hl; return; }
    r -= 2 * M;
    int pair = r >> 2;
    const int q = r & 3;
    j = 0;
    while (pair >= M - 1 - j) { pair -= M - 1 - j; ++j; }
    k = j + 1 + pair;
    dj = (q < 2) ? hl : -hl;
    dk = (q & 1) ? -hl : hl;
}

template <int NL, bool TRIPLET, int M>
__global__ void __launch_bounds__(128, 4)
ga_uncertainty_kernel(const __grid_constant__ SynthDesc sd, const __grid_constant__ GaDesc gd,
                      const float* __restrict__ obs, const uint8_t* __restrict__ mask, const float* __restrict__ mu_arr,
                      int64_t N, const float* __restrict__ params, float* __restrict__ out_sigma, float* __restrict__ out_chi2) {
    extern __shared__ float4 smem4[];
    const int L = sd.L, tid = threadIdx.x;
    uint32_t* scratch = reinterpret_cast<uint32_t*>(smem4);
    float* pix_s = reinterpret_cast<float*>(scratch + 64);
    float* obs_s = pix_s + ME_PIX_WORDS;
    float2* nm_s = reinterpret_cast<float2*>(obs_s + 8 * ((L + 1) >> 1));
    float* chi2v = reinterpret_cast<float*>(nm_s + ((L + 1) >> 1));
    if (M == ME_MAX_NPAR) stage_nm(nm_s, sd.nm_profile, L, tid, 128);
    const int ne = unc_n_eval(M);
    const float h = 1.0f / 64.0f;     // reading U1 (amended in round 2): the FP32 noise on a curvature goes as eps chi2 / h^2
    const float qnan = __int_as_float(0x7fc00000);
    for (int64_t n = blockIdx.x; n < N; n += gridDim.x) {
        if (mask != nullptr && mask[n] == 0) {
            if (tid < M) out_sigma[n * M + tid] = qnan;
            if (tid == 0 && out_chi2 != nullptr) out_chi2[n] = qnan;
            continue;
        }
        const float mu = mu_arr != nullptr ? __ldg(mu_arr + n) : 1.0f;
        __syncthreads();
        stage_obs(obs_s, obs + n * 4 * (int64_t)L, L, tid, 128);
        __syncthreads();
        pixel_prologue(obs_s, L, gd, pix_s, tid == 0);
        __syncthreads();
        // box coordinates of the optimum (inverse of the decode of reading G1; inclination on the per-pixel box)
        float u0[M], lo[M], span[M];
#pragma unroll
        for (int j = 0; j < M; ++j) {
            const float pj = __ldg(params + n * M + j);
            lo[j] = gd.lo[j]; span[j] = gd.log_scale[j] ? gd.log2ratio[j] : gd.span[j];
            if (j == 1 && !gd.log_scale[1]) { lo[j] = pix_s[4]; span[j] = pix_s[5]; }
            if (gd.log_scale[j]) u0[j] = span[j] != 0.f ? log2f(pj / lo[j]) / span[j] : 0.f;
            else u0[j] = span[j] != 0.f ? (pj - lo[j]) / span[j] : 0.f;
        }
        for (int e = tid; e < ne; e += 128) {
            int j1, j2; float d1, d2;
            unc_offsets(M, e, h, j1, d1, j2, d2);
            float p[M];
#pragma unroll
            for (int j = 0; j < M; ++j) {
                const float u = u0[j] + (j == j1 ? d1 : 0.f) + (j == j2 ? d2 : 0.f);
                p[j] = gd.log_scale[j] ? lo[j] * exp2f(u * span[j]) : fmaf(span[j], u, lo[j]);
            }
            chi2v[e] = fitness_params<NL, TRIPLET, M>(p, mu, sd, gd, reinterpret_cast<const float4*>(obs_s), nm_s, pix_s);
        }
        __syncthreads();
        if (tid == 0) {
            const int per_level = 2 * M + 2 * M * (M - 1);
            double H[M * M], Vn[M * M];
            int idx[M], na = 0;
            for (int j = 0; j < M; ++j) if (span[j] != 0.f) idx[na++] = j;
            const double c0 = (double)chi2v[0];
            for (int a = 0; a < na; ++a)
                for (int b = a; b < na; ++b) {
                    const int j = idx[a], k = idx[b];
                    double D[2];
                    for (int level = 0; level < 2; ++level) {
                        const double hl = level == 0 ? (double)h : 0.5 * (double)h;
                        const float* c = chi2v + 1 + level * per_level;
                        if (j == k) D[level] = ((double)c[2 * j] - 2.0 * c0 + (double)c[2 * j + 1]) / (hl * hl);
                        else {
                            int pair = 0;
                            for (int q = 0; q < j; ++q) pair += M - 1 - q;
                            pair += k - j - 1;
                            const float* q4 = c + 2 * M + 4 * pair;
                            D[level] = ((double)q4[0] - (double)q4[1] - (double)q4[2] + (double)q4[3]) / (4.0 * hl * hl);
                        }
                    }
                    H[a * na + b] = H[b * na + a] = (4.0 * D[1] - D[0]) / 3.0;      // Richardson / Neville, one level
                }
            for (int a = 0; a < na; ++a) for (int b = 0; b < na; ++b) Vn[a * na + b] = a == b ? 1.0 : 0.0;
            bool ok = na > 0;
            for (int c = 0; c < na && ok; ++c) {                                     // Gauss-Jordan, partial pivoting
                int piv = c;
                for (int r = c + 1; r < na; ++r) if (fabs(H[r * na + c]) > fabs(H[piv * na + c])) piv = r;
                if (!(fabs(H[piv * na + c]) > 0.0)) { ok = false; break; }
                for (int q = 0; q < na; ++q) {
                    double t = H[c * na + q]; H[c * na + q] = H[piv * na + q]; H[piv * na + q] = t;
                    t = Vn[c * na + q]; Vn[c * na + q] = Vn[piv * na + q]; Vn[piv * na + q] = t;
                }
                const double d = 1.0 / H[c * na + c];
                for (int q = 0; q < na; ++q) { H[c * na + q] *= d; Vn[c * na + q] *= d; }
                for (int r = 0; r < na; ++r) {
                    if (r == c) continue;
                    const double f = H[r * na + c];
                    if (f == 0.0) continue;
                    for (int q = 0; q < na; ++q) { H[r * na + q] -= f * H[c * na + q]; Vn[r * na + q] -= f * Vn[c * na + q]; }
                }
            }
            for (int a = 0; a < na && ok; ++a) if (!(Vn[a * na + a] > 0.0)) ok = false;
            for (int j = 0; j < M; ++j) out_sigma[n * M + j] = span[j] != 0.f ? qnan : 0.f;
            if (ok)
                for (int a = 0; a < na; ++a) {
                    const int j = idx[a];
                    const double su = sqrt(Vn[a * na + a] * c0 / M);                 // eq. 26
                    const double dpdu = gd.log_scale[j] ? (double)__ldg(params + n * M + j) * 0.6931471805599453 * (double)span[j]
                                                        : (double)span[j];
                    out_sigma[n * M + j] = (float)(su * fabs(dpdu));
                }
            if (out_chi2 != nullptr) out_chi2[n] = chi2v[0];
        }
    }
}

// Test hook: the fused fitness alone (128 threads per pixel, individuals strided over the block).
template <int NL, bool TRIPLET, int M>
__global__ void __launch_bounds__(128, 4)
ga_fitness_kernel(const __grid_constant__ SynthDesc sd, const __grid_constant__ GaDesc gd,
                  const float* __restrict__ genes, const float* __restrict__ obs, const float* __restrict__ mu_arr,
                  int64_t N, float* __restrict__ chi2_out) {
    extern __shared__ float4 smem4[];
    float* obs_s = reinterpret_cast<float*>(smem4);
    const int L = sd.L, pop = gd.pop, tid = threadIdx.x;
    float2* nm_s = reinterpret_cast<float2*>(obs_s + 8 * ((L + 1) >> 1));
    if (M == ME_MAX_NPAR) stage_nm(nm_s, sd.nm_profile, L, tid, 128);
    float* pix_s = reinterpret_cast<float*>(nm_s + ((L + 1) >> 1));               // fixed weights, configured box
    if (tid < 4) pix_s[tid] = gd.w2[tid];
    if (tid == 4) { pix_s[4] = gd.lo[1]; pix_s[5] = gd.span[1]; }
    for (int64_t n = blockIdx.x; n < N; n += gridDim.x) {
        __syncthreads();
        stage_obs(obs_s, obs + n * 4 * (int64_t)L, L, tid, 128);
        __syncthreads();
        const float mu = mu_arr != nullptr ? __ldg(mu_arr + n) : 1.0f;
        for (int i = tid; i < pop; i += 128) {
            float g[M];
#pragma unroll
            for (int j = 0; j < M; ++j) g[j] = genes[(n * pop + i) * M + j];
            chi2_out[n * pop + i] = fitness<NL, TRIPLET, M>(g, mu, sd, gd, reinterpret_cast<const float4*>(obs_s), nm_s, pix_s);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Launchers of this translation unit's specialisation
// ------------------------------------------------------------------------------------------------------------
static inline unsigned grid_for_(int64_t n) { return (unsigned)(n < 0x7fffffffLL ? n : 0x7fffffffLL); }

template <int NL, bool TRIPLET, int M, int THREADS, int MINB>
static cudaError_t launch_ga_invert_t(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask,
                                      const float* mu, int64_t N, float* out_params, float* out_chi2, cudaStream_t st) {
    auto k = ga_invert_kernel<NL, TRIPLET, M, THREADS, MINB>;
    const size_t smem = (size_t)40 * ((sd.L + 1) / 2) + (size_t)2 * gd.pop * M * 4 + (size_t)2 * gd.pop * 4 + 64 * 4 +
                        (size_t)2 * gd.pop + 16 + ME_PIX_WORDS * 4 + (size_t)8 * NL * (sd.L / 2 + 1) +
                        ((TRIPLET && NL <= 2) ? (size_t)ME_FAR_ROWS * NL * THREADS * 16 : 0);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k<<<grid_for_(N), THREADS, smem, st>>>(sd, gd, obs, mask, mu, N, out_params, out_chi2);
    return cudaGetLastError();
}

// (pop -> block size, min blocks/SM).  64- and 128-thread blocks run at 5 warps per scheduler (96 registers, 60 B of spill
// stores outside the wavelength loop): since the genes are stored before the fitness call the loop body needs 119 registers
// unconstrained, and at that baseline the fifth warp wins (+3.5 %; at the 125 of rounds 1-2 it lost to 232 B of spills, and a
// sixth warp at 80 registers loses again: profiles/r2_experiments.md).  Larger blocks keep <= 128 registers/thread.
#define ME_DISPATCH_THREADS(FN, ...)                                                                          \
    do {                                                                                                        \
        const int pop_ = gd.pop;                                                                                \
        if (pop_ <= 64) return FN<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, 64, 10>(__VA_ARGS__);                  \
        if (pop_ <= 128) return FN<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, 128, 5>(__VA_ARGS__);                \
        if (pop_ <= 256) return FN<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, 256, 2>(__VA_ARGS__);                \
        if (pop_ <= 512) return FN<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, 512, 1>(__VA_ARGS__);                \
        return FN<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, 1024, 1>(__VA_ARGS__);                                \
    } while (0)

#define ME_CAT4_(a, b, c, d) a##_##b##_##c##_##d
#define ME_CAT4(a, b, c, d) ME_CAT4_(a, b, c, d)
#define ME_INST_NAME(base) ME_CAT4(base, ME_INST_NL, ME_INST_TAG, ME_INST_M)

cudaError_t ME_INST_NAME(launch_ga_invert)(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask,
                                           const float* mu, int64_t N, float* out_params, float* out_chi2, cudaStream_t st) {
    ME_DISPATCH_THREADS(launch_ga_invert_t, sd, gd, obs, mask, mu, N, out_params, out_chi2, st);
}

cudaError_t ME_INST_NAME(launch_ga_fitness)(const SynthDesc& sd, const GaDesc& gd, const float* genes, const float* obs,
                                            const float* mu, int64_t N, float* chi2_out, cudaStream_t st) {
    const size_t smem = (size_t)40 * ((sd.L + 1) / 2) + ME_PIX_WORDS * 4;
    ga_fitness_kernel<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M><<<grid_for_(N), 128, smem, st>>>(sd, gd, genes, obs, mu, N, chi2_out);
    return cudaGetLastError();
}

cudaError_t ME_INST_NAME(launch_uncertainty)(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask,
                                             const float* mu, int64_t N, const float* params, float* out_sigma,
                                             float* out_chi2, cudaStream_t st) {
    const size_t smem = 64 * 4 + ME_PIX_WORDS * 4 + (size_t)40 * ((sd.L + 1) / 2) + (size_t)4 * (1 + 2 * (2 * ME_INST_M + 2 * ME_INST_M * (ME_INST_M - 1)));
    ga_uncertainty_kernel<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M><<<grid_for_(N), 128, smem, st>>>(sd, gd, obs, mask, mu, N, params,
                                                                                                  out_sigma, out_chi2);
    return cudaGetLastError();
}

cudaError_t ME_INST_NAME(launch_synth)(const SynthDesc& sd, const float* params, const float* mu, const int* perm,
                                       int* task_counter, int64_t P, float* out_stokes, const float* obs_ref, const float* w2,
                                       float inv_nu, float* out_chi2, cudaStream_t st) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t blocks_needed = (P + SYNTH_THREADS - 1) / SYNTH_THREADS;
    const int64_t cap = (int64_t)sms * ((out_stokes == nullptr && ME_INST_NL <= 2) ? 5 : 4);   // persistent grid: the resident blocks per SM
    const unsigned grid = (unsigned)(blocks_needed < cap ? blocks_needed : cap);
    const size_t smem = (out_stokes != nullptr ? (size_t)(SYNTH_THREADS / 32) * 32 * SYNTH_VS * sizeof(float) : 0) +
                        ((ME_INST_TRIPLET && ME_INST_NL <= 2) ? (size_t)ME_FAR_ROWS * ME_INST_NL * SYNTH_THREADS * 16 : 0) +
                        (size_t)32 * ((sd.L + 1) / 2) + (size_t)8 * ME_INST_NL * (sd.L / 2 + 1);
    auto k = out_stokes != nullptr ? me_synth_kernel<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, true>
                                   : me_synth_kernel<ME_INST_NL, ME_INST_TRIPLET, ME_INST_M, false>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    k<<<grid, SYNTH_THREADS, smem, st>>>(sd, params, mu, perm, task_counter, P, out_stokes, obs_ref, w2[0], w2[1], w2[2], w2[3], inv_nu, out_chi2);
    return cudaGetLastError();
}

}  // namespace me
