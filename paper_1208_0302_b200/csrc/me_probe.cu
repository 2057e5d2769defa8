// me_probe.cu — instruction-throughput probes for the roofline denominators of the ALU-bound fitness loop
// (SURVEY.md par. 8(d): MEASURED_PEAKS.json has no FP32 / SFU peak, so they are measured on the box).
//
// Each probe is a register-only loop of independent dependency chains (8 per thread) of ONE instruction class, or
// a fixed mix, launched on every SM with full occupancy; the caller times it with CUDA events and divides the
// known instruction count by the time.  Nothing here touches memory except one guarded store that keeps the chains
// alive.  kinds:
//   0  FFMA   scalar fp32 fma                      (2 flop / lane-instruction)
//   1  FFMA2  packed fp32x2 fma                    (4 flop / lane-instruction)
//   2  FFMA2 + FFMA alternating 1:1                (does the scalar fma issue beside the packed one?)
//   3  MUFU.RCP / MUFU.EX2 alternating             (SFU / XU pipe)
//   4  FMUL2  packed multiply                      (2 flop / lane-instruction)
//   5  FFMA2 + FFMA 2:1
//   6  FFMA2 + MUFU.RCP 8:1                        (the fitness loop's ratio, to see whether XU steals FMA issue)
//   7  FFMA2 pair x scalar + scalar   8  FFMA2 pair x pair + immediate   9  FFMA2 pair x scalar + pair   10  FADD2
//      (operand forms: three full register pairs cost more register-file bandwidth than broadcast scalars)
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
                } else if (KIND == 2) {
                    x[c] = __ffma2_rn(x[c], a2, b2);
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(y[c]) : "f"(a), "f"(b));
                } else if (KIND == 3) {       // rcp and ex2 alternate so that no pair of steps folds to the identity
                    if (u & 1) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(y[c]));
                    else asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(y[c]));
                } else if (KIND == 4) {
                    x[c] = __fmul2_rn(x[c], a2);
                } else if (KIND == 5) {
                    x[c] = __ffma2_rn(x[c], a2, b2);
                    if (c & 1) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(y[c]) : "f"(a), "f"(b));
                } else if (KIND == 7) {       // pair x broadcast scalar + broadcast scalar
                    x[c] = __ffma2_rn(x[c], make_float2(a, a), make_float2(b, b));
                } else if (KIND == 8) {       // pair x pair + immediate
                    x[c] = __ffma2_rn(x[c], a2, make_float2(0.001f, 0.001f));
                } else if (KIND == 9) {       // pair x broadcast scalar + pair
                    x[c] = __ffma2_rn(x[c], make_float2(a, a), b2);
                } else if (KIND == 10) {
                    x[c] = __fadd2_rn(x[c], b2);
                } else {
                    x[c] = __ffma2_rn(x[c], a2, b2);
                    if (c == 0) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(y[u]));
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
        case 2: probe_kernel<2><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 3: probe_kernel<3><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 4: probe_kernel<4><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 5: probe_kernel<5><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 6: probe_kernel<6><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 7: probe_kernel<7><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 8: probe_kernel<8><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 9: probe_kernel<9><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        case 10: probe_kernel<10><<<blocks, 256, 0, st>>>(iters, seed, out); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace me
