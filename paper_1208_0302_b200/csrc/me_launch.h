// me_launch.h — host-side launch interface between me_api.cu (validation, descriptors) and me_kernels.cu.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace me {

struct SynthDesc;
struct GaDesc;

cudaError_t launch_ga_invert(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask, const float* mu,
                             int64_t N, float* out_params, float* out_chi2, cudaStream_t st);
cudaError_t launch_uncertainty(const SynthDesc& sd, const GaDesc& gd, const float* obs, const uint8_t* mask, const float* mu,
                               int64_t N, const float* params, float* out_sigma, float* out_chi2, cudaStream_t st);
cudaError_t launch_ga_fitness(const SynthDesc& sd, const GaDesc& gd, const float* genes, const float* obs, const float* mu,
                              int64_t N, float* chi2_out, cudaStream_t st);
cudaError_t launch_ga_step(const GaDesc& gd, int npar, const float* genes_in, const float* chi2_in, int64_t N, int t,
                           float* genes_out, cudaStream_t st);
cudaError_t launch_ga_init(const GaDesc& gd, int npar, int64_t N, float* genes_out, cudaStream_t st);
size_t synth_workspace_bytes(int64_t P);
cudaError_t launch_synth(const SynthDesc& sd, const float* params, const float* mu, int64_t P, float* out_stokes,
                         const float* obs_ref, const float* w2, float inv_nu, float* out_chi2, void* work, size_t work_bytes,
                         cudaStream_t st);
int64_t synth_static_max_vectors();
cudaError_t synth_static_scratch(void** ptr, size_t* bytes);     // the library's fixed scratch array on the current device
cudaError_t launch_philox(uint32_t k0, uint32_t k1, uint32_t c0_base, uint32_t c1, uint32_t c2, uint32_t c3, int64_t n,
                          uint32_t* out, cudaStream_t st);
cudaError_t launch_ga_prologue(const SynthDesc& sd, const GaDesc& gd, const float* obs, int64_t N, float* out, cudaStream_t st);
cudaError_t launch_probe(int kind, int iters, int blocks, float* out, cudaStream_t st);
cudaError_t launch_faddeeva(const float* v, const float* a, int64_t n, float* H, float* F, cudaStream_t st);

}  // namespace me
