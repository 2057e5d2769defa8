// me_kernels.cu — small kernels (GA hooks, Philox, Faddeeva hook) and the launch dispatch of libme_b200.so (sm_100a).
// The heavy template kernels are in me_inst.cuh:
//
//   ga_invert_kernel   CTA = one pixel, thread = one individual; the whole GA of Alg. 1 runs
//                      on-chip: observation staged once in shared memory, population double-buffered in shared
//                      memory, fitness (synthesis + eq. 16) accumulated in registers over a serial wavelength loop.
//   me_synth_kernel    thread = one parameter vector (the lanes of a warp sit at the same wavelength, as in the GA kernel),
//                      [P,4,L] stores through a warp-private transpose tile, optional chi2; persistent grid.
//   ga_fitness_kernel / ga_step_kernel / ga_init_kernel / philox_kernel / faddeeva_kernel: test hooks.
//
// The paper's own mapping (block = individual, thread = wavelength, GA on the host with per-generation PCIe
// transfers) is prior art for a Tesla C1060 and is deliberately not followed:
// see DESIGN.md "What differs from the paper".
#include <mutex>

#include "me_device.cuh"
#include "me_launch.h"

namespace me {

// ------------------------------------------------------------------------------------------------------------
// Test hooks
// ------------------------------------------------------------------------------------------------------------
// One generation from given genes and given fitness (shared: genes [pop][M] | chi2 [pop] | scratch [64]).
template <int M>
__global__ void __launch_bounds__(ME_MAX_POP)    // pop threads per block, up to 1024: at most 64 registers (the 11-gene body took 66)
ga_step_kernel(const __grid_constant__ GaDesc gd, const float* __restrict__ genes_in,
                               const float* __restrict__ chi2_in, int64_t N, int t, float* __restrict__ genes_out) {
    extern __shared__ float4 smem4[];
    const int pop = gd.pop, tid = threadIdx.x;
    float* genes_s = reinterpret_cast<float*>(smem4);
    float* chi2_s = genes_s + pop * M;
    uint32_t* scratch = reinterpret_cast<uint32_t*>(chi2_s + pop);
    uint16_t* order_s = reinterpret_cast<uint16_t*>(scratch + 64);
    const float INF = __int_as_float(0x7f800000);
    const bool restart = gd.variant != 0 && t < gd.generations && (t % gd.n_samp) == 0;
    for (int64_t n = blockIdx.x; n < N; n += gridDim.x) {
        __syncthreads();
        for (int k = tid; k < pop * M; k += blockDim.x) genes_s[k] = genes_in[n * pop * M + k];
        float f = INF;
        if (tid < pop) {
            f = chi2_in[n * pop + tid];
            if (!(f < INF)) f = INF;
            chi2_s[tid] = f;
        }
        __syncthreads();
        float fe; int ie;
        block_argmin(f, tid, scratch, fe, ie);
        if (restart) {
            if (tid < pop) order_s[rank_of(chi2_s, pop, tid)] = (uint16_t)tid;
            __syncthreads();
        }
        if (tid < pop) {
            float g[M];
            if (tid == 0) {
#pragma unroll
                for (int j = 0; j < M; ++j) g[j] = genes_s[ie * M + j];
            } else if (gd.variant) {
                make_child_binary<M>(g, genes_s, chi2_s, restart ? order_s : nullptr, restart ? pop - pop / 2 : pop,
                                     gd.pixel_base + (uint32_t)n, (uint32_t)t, (uint32_t)tid, gd);
            } else {
                make_child<M>(g, genes_s, chi2_s, gd.pixel_base + (uint32_t)n, (uint32_t)t, (uint32_t)tid, gd.mut_scale[t], gd);
            }
#pragma unroll
            for (int j = 0; j < M; ++j) genes_out[(n * pop + tid) * M + j] = g[j];
        }
    }
}

template <int M>
__global__ void ga_init_kernel(const __grid_constant__ GaDesc gd, int64_t N, float* __restrict__ genes_out) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N * gd.pop) return;
    const int64_t n = k / gd.pop;
    const int i = (int)(k - n * gd.pop);
    float g[M];
    if (gd.variant) sobol_genes<M>(g, gd.pixel_base + (uint32_t)n, (uint32_t)i + 1u, gd);
    else init_genes<M>(g, gd.pixel_base + (uint32_t)n, (uint32_t)i, gd);
#pragma unroll
    for (int j = 0; j < M; ++j) genes_out[k * M + j] = g[j];
}

// The per-pixel prologue alone (one warp per pixel): out[n][12] = w_I, w_Q, w_U, w_V, gamma_lo, gamma_hi, B_los (centre of
// gravity), the stored genes (B, gamma) of the centre-of-gravity member, and the stored genes (B, gamma, chi) of the Auer
// weak-field member.  The offsets lambda_j - lambda_(seed line) are read from the descriptor in the constant bank.
__global__ void ga_prologue_kernel(const __grid_constant__ SynthDesc sd, const __grid_constant__ GaDesc gd,
                                   const float* __restrict__ obs, int64_t N, float* __restrict__ out) {
    extern __shared__ float4 smem4[];
    const int L = sd.L;
    float* obs_s = reinterpret_cast<float*>(smem4);
    float* pix_s = obs_s + 8 * ((L + 1) >> 1);
    const float* off = sd.off[gd.seed_line];
    for (int64_t n = blockIdx.x; n < N; n += gridDim.x) {
        __syncwarp();
        stage_obs(obs_s, obs + n * 4 * (int64_t)L, L, threadIdx.x, 32);
        __syncwarp();
        if (threadIdx.x == 0) for (int k = 7; k < 14; ++k) pix_s[k] = 0.f;
        __syncwarp();
        pixel_prologue(obs_s, L, gd, pix_s, threadIdx.x == 0, off);
        if (gd.prologue & 8) pixel_seed_auer(obs_s, L, gd, pix_s, threadIdx.x == 0, off);
        __syncwarp();
        if (threadIdx.x < 4) out[n * 12 + threadIdx.x] = sqrtf(pix_s[threadIdx.x]) * gd.sigma[threadIdx.x];   // back to w_s
        if (threadIdx.x == 4) {
            out[n * 12 + 4] = pix_s[4]; out[n * 12 + 5] = pix_s[6];
            out[n * 12 + 6] = pix_s[9]; out[n * 12 + 7] = pix_s[7]; out[n * 12 + 8] = pix_s[8];
            out[n * 12 + 9] = pix_s[10]; out[n * 12 + 10] = pix_s[11]; out[n * 12 + 11] = pix_s[12];
        }
    }
}

__global__ void philox_kernel(uint32_t k0, uint32_t k1, uint32_t c0_base, uint32_t c1, uint32_t c2, uint32_t c3,
                              int64_t n, uint4* __restrict__ out) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = philox4x32_10(c0_base + (uint32_t)i, c1, c2, c3, k0, k1);
}

__global__ void faddeeva_kernel(const float* __restrict__ v, const float* __restrict__ a, int64_t n,
                                float* __restrict__ H, float* __restrict__ F) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    f2 wr, wi;
    faddeeva_pair(make_float2(v[i], i + 1 < n ? v[i + 1] : v[i]), fad_const(a[i]), wr, wi);   // pair (i, i+1) at a[i]
    H[i] = wr.x; F[i] = wi.x;
}

// ------------------------------------------------------------------------------------------------------------
// Launchers
// ------------------------------------------------------------------------------------------------------------
static inline unsigned grid_for(int64_t n) { return (unsigned)(n < 0x7fffffffLL ? n : 0x7fffffffLL); }

// The heavy kernels live in me_inst_<nl>_<t|g>.cu (one translation unit per specialisation).
#define ME_DECL_INST(NL, TAG, M)                                                                                                \
    cudaError_t launch_ga_invert_##NL##_##TAG##_##M(const SynthDesc&, const GaDesc&, const float*, const uint8_t*, const float*, \
                                                    int64_t, float*, float*, cudaStream_t);                                     \
    cudaError_t launch_ga_fitness_##NL##_##TAG##_##M(const SynthDesc&, const GaDesc&, const float*, const float*, const float*,  \
                                                     int64_t, float*, cudaStream_t);                                            \
    cudaError_t launch_uncertainty_##NL##_##TAG##_##M(const SynthDesc&, const GaDesc&, const float*, const uint8_t*,           \
                                                      const float*, int64_t, const float*, float*, float*, cudaStream_t);        \
    cudaError_t launch_synth_##NL##_##TAG##_##M(const SynthDesc&, const float*, const float*, const int*, int*, int64_t, float*,  \
                                                const float*, const float*, float, float*, cudaStream_t);
ME_DECL_INST(1, t, 9) ME_DECL_INST(2, t, 9) ME_DECL_INST(4, t, 9) ME_DECL_INST(1, g, 9) ME_DECL_INST(2, g, 9) ME_DECL_INST(4, g, 9)
ME_DECL_INST(1, t, 11) ME_DECL_INST(2, t, 11) ME_DECL_INST(4, t, 11) ME_DECL_INST(1, g, 11) ME_DECL_INST(2, g, 11) ME_DECL_INST(4, g, 11)

#define ME_DISPATCH_M(BASE, M, ...)                                                  \
    do {                                                                             \
        if (sd.all_triplets) {                                                       \
            if (sd.n_lines == 1) return BASE##_1_t_##M(__VA_ARGS__);                 \
            if (sd.n_lines == 2) return BASE##_2_t_##M(__VA_ARGS__);                 \
            return BASE##_4_t_##M(__VA_ARGS__);                                      \
        }                                                                            \
        if (sd.n_lines == 1) return BASE##_1_g_##M(__VA_ARGS__);                     \
        if (sd.n_lines == 2) return BASE##_2_g_##M(__VA_ARGS__);                     \
        return BASE##_4_g_##M(__VA_ARGS__);                                          \
    } while (0)
#define ME_DISPATCH(BASE, ...)                                                       \
    do {                                                                             \
        if (sd.npar == ME_MAX_NPAR) ME_DISPATCH_M(BASE, 11, __VA_ARGS__);            \
        ME_DISPATCH_M(BASE, 9, __VA_ARGS__);                                         \
    } while (0)

static cudaError_t launch_synth_ordered(const SynthDesc& sd, const float* params, const float* mu, const int* perm,
                                        int* task_counter, int64_t P, float* out_stokes, const float* obs_ref, const float* w2,
                                        float inv_nu, float* out_chi2, cudaStream_t st) {
    ME_DISPATCH(launch_synth, sd, params, mu, perm, task_counter, P, out_stokes, obs_ref, w2, inv_nu, out_chi2, st);
}

cudaError_t launch_ga_invert(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask, const float* mu,
                             int64_t N, float* out_params, float* out_chi2, cudaStream_t st) {
    ME_DISPATCH(launch_ga_invert, sd, gd, obs, mask, mu, N, out_params, out_chi2, st);
}

cudaError_t launch_uncertainty(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask, const float* mu,
                               int64_t N, const float* params, float* out_sigma, float* out_chi2, cudaStream_t st) {
    ME_DISPATCH(launch_uncertainty, sd, gd, obs, mask, mu, N, params, out_sigma, out_chi2, st);
}

cudaError_t launch_ga_fitness(const SynthDesc& sd, const GaDesc& gd, const float* genes, const float* obs, const float* mu,
                              int64_t N, float* chi2_out, cudaStream_t st) {
    ME_DISPATCH(launch_ga_fitness, sd, gd, genes, obs, mu, N, chi2_out, st);
}

// ------------------------------------------------------------------------------------------------------------
// Processing order of me_synth.  The Voigt tier a thread takes at wavelength j depends on its vector's Doppler width
// (scale), line-of-sight velocity (shift) and field strength (splitting); with thread = vector the 32 lanes of a warp
// branch together only if their vectors are alike.  A GA population is; a batch of unrelated vectors (BASELINE config 2)
// is not.  So large batches are visited in the order of a counting sort on a coarse key of those three parameters
// (log dlambdaD in 5 % bins, v_los in 1 km/s bins, log2 B in half-octave bins); outputs stay at their own index.
// ------------------------------------------------------------------------------------------------------------
#define SYNTH_NKEY 32768
#define SYNTH_SORT_MIN 400000     /* below this the four extra launches cost more than the coherence wins (measured) */

__device__ __forceinline__ int synth_key(const float* p) {
    const float B = fabsf(p[0]), dld = fmaxf(p[4], 1e-3f), vlos = p[6];
    const int kd = min(max((int)(log2f(dld) * 14.2f), 0), 127);          // 2^(1/14.2) = 1.05
    const int kv = min(max((int)floorf(vlos) + 8, 0), 15);
    const int kb = min(max((int)(log2f(B + 1.0f) * 2.0f), 0), 15);
    return (kd * 16 + kv) * 16 + kb;
}

// Pass 1: keys and their histogram.  One CTA per SM, each with a PRIVATE histogram of all SYNTH_NKEY bins in shared memory
// (128 KB) over a contiguous slice of the batch; only its non-empty bins go to the global histogram.  A batch populates few
// bins (config 2: ~900 of 32 768, on ~50 cache lines), and run r2q measured what one global atomic per vector costs on so
// few lines: 31 us for this pass and 34 us for the scatter at P = 1e6, against 700 us for the synthesis itself.
// The last CTA to finish (ticket in ctr[1]) turns the global histogram into its exclusive prefix sums in place, which
// was a launch of its own (37 us on one SM with strided loads).
#define SYNTH_SORT_THREADS 1024
__global__ void __launch_bounds__(SYNTH_SORT_THREADS)
synth_hist_kernel(const float* __restrict__ params, int npar, int64_t P, int* __restrict__ keys, int* hist, int* ctr) {
    extern __shared__ int sh[];                                      // [SYNTH_NKEY]
    __shared__ int warp_tot[32];
    __shared__ int ticket_s;
    const int tid = threadIdx.x;
    for (int i = tid; i < SYNTH_NKEY / 4; i += SYNTH_SORT_THREADS) reinterpret_cast<int4*>(sh)[i] = make_int4(0, 0, 0, 0);
    __syncthreads();
    const int64_t chunk = (P + gridDim.x - 1) / gridDim.x, begin = blockIdx.x * chunk, end = begin + chunk < P ? begin + chunk : P;
    for (int64_t v = begin + tid; v < end; v += SYNTH_SORT_THREADS) {
        const int k = synth_key(params + v * npar);
        keys[v] = k;
        atomicAdd(sh + k, 1);
    }
    __syncthreads();
    for (int i = tid; i < SYNTH_NKEY; i += SYNTH_SORT_THREADS) {
        const int c = sh[i];
        if (c != 0) atomicAdd(hist + i, c);
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) ticket_s = atomicAdd(ctr + 1, 1);
    __syncthreads();
    if (ticket_s != (int)gridDim.x - 1) return;
    __threadfence();
    // exclusive scan of the SYNTH_NKEY counts by this one CTA: thread t owns the 32 consecutive bins [32 t, 32 t + 32)
    constexpr int PER = SYNTH_NKEY / SYNTH_SORT_THREADS;             // 32
    int4* h4 = reinterpret_cast<int4*>(hist) + tid * (PER / 4);
    int4 c[PER / 4];
    int sum = 0;
#pragma unroll
    for (int i = 0; i < PER / 4; ++i) { c[i] = __ldcg(h4 + i); sum += c[i].x + c[i].y + c[i].z + c[i].w; }
    int incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int x = __shfl_up_sync(0xffffffffu, incl, d); if ((tid & 31) >= d) incl += x; }
    if ((tid & 31) == 31) warp_tot[tid >> 5] = incl;
    __syncthreads();
    if (tid < 32) {
        int w = warp_tot[tid];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int x = __shfl_up_sync(0xffffffffu, w, d); if (tid >= d) w += x; }
        warp_tot[tid] = w;
    }
    __syncthreads();
    int run = incl - sum + (tid >= 32 ? warp_tot[(tid >> 5) - 1] : 0);
#pragma unroll
    for (int i = 0; i < PER / 4; ++i) {
        int4 o;
        o.x = run; run += c[i].x; o.y = run; run += c[i].y; o.z = run; run += c[i].z; o.w = run; run += c[i].w;
        h4[i] = o;
    }
}

// Pass 2: the same slices again.  Each CTA re-counts its slice in shared memory, reserves one range per non-empty bin with a
// single global atomic on the bin's cursor (the prefix sums of pass 1), and hands out the slots of its ranges with
// shared-memory atomics.  The order inside a bin is arbitrary, as it was; every vector is computed on its own.
__global__ void __launch_bounds__(SYNTH_SORT_THREADS)
synth_scatter_kernel(const int* __restrict__ keys, int64_t P, int* __restrict__ cursor, int* __restrict__ perm) {
    extern __shared__ int sh[];                                      // [SYNTH_NKEY]: counts, then next free slot per bin
    const int tid = threadIdx.x;
    for (int i = tid; i < SYNTH_NKEY / 4; i += SYNTH_SORT_THREADS) reinterpret_cast<int4*>(sh)[i] = make_int4(0, 0, 0, 0);
    __syncthreads();
    const int64_t chunk = (P + gridDim.x - 1) / gridDim.x, begin = blockIdx.x * chunk, end = begin + chunk < P ? begin + chunk : P;
    for (int64_t v = begin + tid; v < end; v += SYNTH_SORT_THREADS) atomicAdd(sh + keys[v], 1);
    __syncthreads();
    for (int i = tid; i < SYNTH_NKEY; i += SYNTH_SORT_THREADS) {
        const int c = sh[i];
        if (c != 0) sh[i] = atomicAdd(cursor + i, c);
    }
    __syncthreads();
    for (int64_t v = begin + tid; v < end; v += SYNTH_SORT_THREADS) perm[atomicAdd(sh + keys[v], 1)] = (int)v;
}

// Bytes of caller-provided scratch the ordered visit needs (histogram [SYNTH_NKEY] | task counter and ticket, padded
// to 32 ints | keys [P] | perm [P]); 0 = not used.
#define SYNTH_NCTR 32
size_t synth_workspace_bytes(int64_t P) {
    if (P < SYNTH_SORT_MIN || P >= 0x7fffffffLL) return 0;
    return (size_t)(2 * P + SYNTH_NKEY + SYNTH_NCTR) * sizeof(int);
}

// work: caller-provided device scratch or nullptr.  Nothing is allocated here; every launch is checked, and a failure of
// the two ordering passes is returned before the synthesis is enqueued.
cudaError_t launch_synth(const SynthDesc& sd, const float* params, const float* mu, int64_t P, float* out_stokes,
                         const float* obs_ref, const float* w2, float inv_nu, float* out_chi2, void* work_v, size_t work_bytes,
                         cudaStream_t st) {
    const int* perm = nullptr;
    int* task_counter = nullptr;
    const size_t need = synth_workspace_bytes(P);
    if (work_v != nullptr && need != 0 && work_bytes >= need) {     // worth two light passes over the parameters
        int* work = static_cast<int*>(work_v);
        int *hist = work, *keys = work + SYNTH_NKEY + SYNTH_NCTR, *pm = keys + P;     // histogram first: it is read and written as int4
        cudaError_t e = cudaMemsetAsync(hist, 0, (SYNTH_NKEY + SYNTH_NCTR) * sizeof(int), st);   // histogram and task counter
        if (e != cudaSuccess) return e;
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const size_t sort_smem = SYNTH_NKEY * sizeof(int);            // 128 KB: one CTA per SM
        if ((e = cudaFuncSetAttribute(synth_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(synth_scatter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sort_smem)) != cudaSuccess) return e;
        synth_hist_kernel<<<sms, SYNTH_SORT_THREADS, sort_smem, st>>>(params, sd.npar, P, keys, hist, hist + SYNTH_NKEY);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        synth_scatter_kernel<<<sms, SYNTH_SORT_THREADS, sort_smem, st>>>(keys, P, hist, pm);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        perm = pm;
        task_counter = hist + SYNTH_NKEY;
    }
    return launch_synth_ordered(sd, params, mu, perm, task_counter, P, out_stokes, obs_ref, w2, inv_nu, out_chi2, st);
}

// ------------------------------------------------------------------------------------------------------------
// me_synth_static: the ordered visit of launch_synth with its scratch in a FIXED device array of this library instead of a
// caller workspace, for callers that may not allocate at all (CUDA graph capture, serving loops, harnesses that forbid
// cudaMalloc).  The array holds the workspace of a batch of SYNTH_STATIC_MAX_P vectors (histogram | counters | keys | perm:
// 16.1 MiB); every device that loads the library carries it until the process exits.
// In host code the array's NAME is only the host-side stand-in of the symbol, not a device address: a kernel handed
// `g_synth_static_scratch` from the host would fault (or, where the GPU can reach host memory, silently use the wrong bytes).
// The device address is asked for once per device, with that device current, by cudaGetSymbolAddress.
// ------------------------------------------------------------------------------------------------------------
#define SYNTH_STATIC_MAX_P (1 << 21)
#define SYNTH_STATIC_INTS (2 * SYNTH_STATIC_MAX_P + SYNTH_NKEY + SYNTH_NCTR)
#define SYNTH_STATIC_MAX_DEVICES 64
static __device__ __align__(256) int g_synth_static_scratch[SYNTH_STATIC_INTS];

int64_t synth_static_max_vectors() { return SYNTH_STATIC_MAX_P; }

// The scratch array's address on the CURRENT device and its size.  Allocates nothing.
cudaError_t synth_static_scratch(void** ptr, size_t* bytes) {
    static std::mutex mtx;
    static void* addr[SYNTH_STATIC_MAX_DEVICES] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= SYNTH_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mtx);
    if (addr[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_synth_static_scratch);
        if (e != cudaSuccess) return e;
        addr[dev] = p;
    }
    *ptr = addr[dev];
    *bytes = (size_t)SYNTH_STATIC_INTS * sizeof(int);
    return cudaSuccess;
}

cudaError_t launch_ga_step(const GaDesc& gd, int npar, const float* genes_in, const float* chi2_in, int64_t N, int t,
                           float* genes_out, cudaStream_t st) {
    const int threads = ((gd.pop + 31) / 32) * 32;
    const size_t smem = (size_t)gd.pop * npar * 4 + (size_t)gd.pop * 4 + 64 * 4 + (size_t)2 * gd.pop + 16;
    // pop = 1024 with 11 genes needs 51 472 B: above the 48 KB a kernel gets without opting in (me.h allows pop up to ME_MAX_POP)
    cudaError_t e = npar == ME_MAX_NPAR
        ? cudaFuncSetAttribute(ga_step_kernel<ME_MAX_NPAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
        : cudaFuncSetAttribute(ga_step_kernel<ME_NPAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (npar == ME_MAX_NPAR) ga_step_kernel<ME_MAX_NPAR><<<grid_for(N), threads, smem, st>>>(gd, genes_in, chi2_in, N, t, genes_out);
    else ga_step_kernel<ME_NPAR><<<grid_for(N), threads, smem, st>>>(gd, genes_in, chi2_in, N, t, genes_out);
    return cudaGetLastError();
}

cudaError_t launch_ga_init(const GaDesc& gd, int npar, int64_t N, float* genes_out, cudaStream_t st) {
    const int64_t total = N * gd.pop;
    if (npar == ME_MAX_NPAR) ga_init_kernel<ME_MAX_NPAR><<<grid_for((total + 255) / 256), 256, 0, st>>>(gd, N, genes_out);
    else ga_init_kernel<ME_NPAR><<<grid_for((total + 255) / 256), 256, 0, st>>>(gd, N, genes_out);
    return cudaGetLastError();
}

// No allocation, no synchronisation: the kernel reads the offsets of the seed line from the descriptor it is passed.
cudaError_t launch_ga_prologue(const SynthDesc& sd, const GaDesc& gd, const float* obs, int64_t N, float* out, cudaStream_t st) {
    const size_t smem = (size_t)32 * ((sd.L + 1) / 2) + ME_PIX_WORDS * 4;
    ga_prologue_kernel<<<grid_for(N), 32, smem, st>>>(sd, gd, obs, N, out);
    return cudaGetLastError();
}

cudaError_t launch_philox(uint32_t k0, uint32_t k1, uint32_t c0_base, uint32_t c1, uint32_t c2, uint32_t c3, int64_t n,
                          uint32_t* out, cudaStream_t st) {
    philox_kernel<<<grid_for((n + 255) / 256), 256, 0, st>>>(k0, k1, c0_base, c1, c2, c3, n, reinterpret_cast<uint4*>(out));
    return cudaGetLastError();
}

cudaError_t launch_faddeeva(const float* v, const float* a, int64_t n, float* H, float* F, cudaStream_t st) {
    faddeeva_kernel<<<grid_for((n + 255) / 256), 256, 0, st>>>(v, a, n, H, F);
    return cudaGetLastError();
}

}  // namespace me
