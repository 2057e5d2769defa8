// me_probe.cu — instruction-throughput probes for the roofline denominators of the ALU-bound fitness loop
// (SURVEY.md par. 8(d): MEASURED_PEAKS.json has no FP32 / SFU peak, so they are measured on the box).
//
// Each probe is a register-only loop of independent dependency chains (8 per thread) of ONE instruction class, or
// a fixed mix, launched on every SM with full occupancy; the caller times it with CUDA events and divides the
// known instruction count by the time.  Nothing here touches memory except one guarded store that keeps the chains
// alive.  kinds (the product ABI carries only the three roofline denominators; the operand-form and mixing probes of round 1,
// whose findings are recorded in profiles/r1_history.md step r1c, are no longer exported):
//   0  FFMA   scalar fp32 fma                      (2 flop / lane-instruction)
//   1  FFMA2  packed fp32x2 fma                    (4 flop / lane-instruction; the form the fitness loop is written in)
//   3  MUFU.RCP / MUFU.EX2 alternating             (SFU / XU pipe)
#include <cuda_runtime.h>
#include <stdint.h>

#include "me_launch.h"

namespace me {

#define PROBE_CHAINS 8

template <int KIND>
__global__ void __launch_bounds__(256) probe_kernel(int iters, float seed, float* __restrict__ out) {
    float2 x[PROBE_CHAINS];
    float y[PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) {
        x[c] = make_float2(seed + (float)(threadIdx.x + c), seed - (float)c);
        y[c] = seed * (float)(c + 1) + (float)threadIdx.x;
    }
    const float2 a2 = make_float2(0.999f + seed, 1.001f - seed), b2 = make_float2(seed, -seed);
    const float a = 0.9995f + seed, b = seed;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
#pragma unroll
            for (int c = 0; c < PROBE_CHAINS; ++c) {
                if (KIND == 0) {
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(y[c]) : "f"(a), "f"(b));
                } else if (KIND == 1) {
                    x[c] = __ffma2_rn(x[c], a2, b2);
                } else if (KIND == 3) {       // rcp and ex2 alternate so that no pair of steps folds to the identity
                    if (u & 1) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(y[c]));
                    else asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(y[c]));
                }
            }
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < PROBE_CHAINS; ++c) s += x[c].x + x[c].y + y[c];
    if (s == 123.456f) out[blockIdx.x * blockDim.x + threadIdx.x] = s;     // never true in practice; keeps the chains
}

// Per thread and per loop iteration: 4 (unroll) x PROBE_CHAINS slots.
cudaError_t launch_probe(int kind, int iters, int blocks, float* out, cudaStream_t st) {
    const float seed = 1e-6f;
    switch (kind) {
        case 0: probe_kernel<0><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 1: probe_kernel<1><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 3: probe_kernel<3><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace me
