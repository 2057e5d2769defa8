// me_device.cuh — device-side building blocks of libme_b200.so (sm_100a, FP32).
//
//   faddeeva32      w(v + i a) = H + iF, two-region FP32 evaluator
//   Individual      per-parameter-vector constants hoisted out of the wavelength loop (eq. 14)
//   stokes_at       absorption matrix (eq. 8) + Unno-Rachkovsky solution (eq. 12-13, 15) at one wavelength
//   philox4x32_10   counter-based RNG keyed by (seed; pixel, generation, individual, block)
//   make_child      tournament selection, arithmetic crossover, bounded mutation
//
// Nothing here is shared with oracle/; the formulas are restated from the paper and DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/me.h"
#include "faddeeva_table.h"

namespace me {

// ------------------------------------------------------------------------------------------------------------
// Kernel-side descriptor, built on the host per call and passed by value as a __grid_constant__ parameter
// (it lands in the constant bank: every access below is warp-uniform).
// ------------------------------------------------------------------------------------------------------------
struct LineDesc {
    float lam0_over_c;      // lambda_l / c                        [A per km/s]
    float dld_scale;        // 1e-3 * lambda_l / lambda_ref         [A per mA]
    float zeeman;           // 4.66857e-13 * lambda_l^2             [A per G]
    float strength;         // r_l
    int kind_begin[4];      // components sorted by kind: [blue | pi | red], kind_begin[3] = end
    int triplet;            // 1 if exactly one component per kind with weight 1 and shifts (-g, 0, +g)
    float g;                // Lande factor of the triplet
    int pad[2];
};

struct SynthDesc {
    int L, n_lines, n_comp, all_triplets;
    LineDesc line[ME_MAX_LINES];
    float shift[ME_MAX_COMP];
    float weight[ME_MAX_COMP];
    float off[ME_MAX_LINES][ME_MAX_L];   // lambda_j - lambda_l, rounded once from double
};

struct GaDesc {
    int pop, generations, tournament_k, pad0;
    float p_cross, p_mut;
    uint32_t key0, key1;
    uint32_t pixel_base;
    float inv_nu;                       // 1 / (4L - M)
    float w2[4];                        // (w_s / sigma_s)^2
    float lo[ME_NPAR], span[ME_NPAR], log2ratio[ME_NPAR];
    int log_scale[ME_NPAR], periodic[ME_NPAR];
    float mut_scale[ME_MAX_GEN + 1];    // s_t, t = 0..generations
};

// ------------------------------------------------------------------------------------------------------------
// Small helpers
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// p <- p * Z + c   (complex p, complex Z, real c): 4 FP32 instructions
__device__ __forceinline__ void chorner(float& pr, float& pi, float zr, float zi, float c) {
    float nr = fmaf(pr, zr, c);
    nr = fmaf(-pi, zi, nr);
    float ni = pr * zi;
    ni = fmaf(pi, zr, ni);
    pr = nr; pi = ni;
}

// ------------------------------------------------------------------------------------------------------------
// Faddeeva function, FP32.  a2 = a*a and La = L + a, La2 = La*La are per-individual constants.
//   wing: w = (i/sqrt(pi)) s R(q), s = 1/z, q = s^2 (no cancellation: H keeps full relative accuracy)
//   core: Weideman N = 16
// ------------------------------------------------------------------------------------------------------------
struct FadConst { float a, a2, La, La2; };

__device__ __forceinline__ FadConst fad_const(float a) {
    FadConst f; f.a = a; f.a2 = a * a; f.La = FAD_L + a; f.La2 = f.La * f.La; return f;
}

__device__ __forceinline__ void faddeeva32(float v, const FadConst& f, float& wr, float& wi) {
    const float r2 = fmaf(v, v, f.a2);
    if (r2 >= FAD_CUT2) {
        const float r = rcp_approx(r2);
        const float sr = v * r, si = -f.a * r;
        const float qr = fmaf(sr, sr, -si * si), qi = 2.0f * sr * si;
        float pr = fmaf(FAD_C6, qr, FAD_C5), pi = FAD_C6 * qi;
        chorner(pr, pi, qr, qi, FAD_C4);
        chorner(pr, pi, qr, qi, FAD_C3);
        chorner(pr, pi, qr, qi, FAD_C2);
        chorner(pr, pi, qr, qi, FAD_C1);
        chorner(pr, pi, qr, qi, FAD_C0);
        wr = -fmaf(sr, pi, si * pr);
        wi = fmaf(sr, pr, -si * pi);
    } else {
        const float r = rcp_approx(fmaf(v, v, f.La2));
        const float dr = f.La * r, di = v * r;                 // D = 1 / (L - iz)
        const float zr = fmaf(FAD_2L, dr, -1.0f), zi = FAD_2L * di;   // Z = (L + iz) D = 2 L D - 1
        float pr = fmaf(FAD_A15, zr, FAD_A14), pi = FAD_A15 * zi;
        chorner(pr, pi, zr, zi, FAD_A13);
        chorner(pr, pi, zr, zi, FAD_A12);
        chorner(pr, pi, zr, zi, FAD_A11);
        chorner(pr, pi, zr, zi, FAD_A10);
        chorner(pr, pi, zr, zi, FAD_A9);
        chorner(pr, pi, zr, zi, FAD_A8);
        chorner(pr, pi, zr, zi, FAD_A7);
        chorner(pr, pi, zr, zi, FAD_A6);
        chorner(pr, pi, zr, zi, FAD_A5);
        chorner(pr, pi, zr, zi, FAD_A4);
        chorner(pr, pi, zr, zi, FAD_A3);
        chorner(pr, pi, zr, zi, FAD_A2);
        chorner(pr, pi, zr, zi, FAD_A1);
        chorner(pr, pi, zr, zi, FAD_A0);
        // w = D (p D + 1/sqrt(pi))   (the factor 2 is folded into the table)
        float tr = fmaf(pr, dr, FAD_INV_SQRTPI);
        tr = fmaf(-pi, di, tr);
        float ti = pr * di;
        ti = fmaf(pi, dr, ti);
        wr = fmaf(dr, tr, -di * ti);
        wi = fmaf(dr, ti, di * tr);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Per-individual constants (decode-time work, once per parameter vector).
// ------------------------------------------------------------------------------------------------------------
template <int NL>
struct Individual {
    FadConst fad;
    float invD[NL], v0[NL], vB[NL];   // 1/dlambdaD_l, -doppler_l/dlambdaD_l, Zeeman splitting in Doppler units
    float kA, kB, kC;                 // h sin^2(gamma), h (1 + cos^2 gamma)/2, h cos(gamma);  h = eta0 / (2 sqrt(pi))
    float c2x, s2x;                   // cos 2chi, sin 2chi
    float S0, muS1;
};

template <int NL>
__device__ __forceinline__ void setup_individual(Individual<NL>& ind, const float* p, float mu, const SynthDesc& d) {
    const float B = p[0], eta0 = p[3], dld = p[4], a = p[5], vlos = p[6];
    float sg, cg;
    sincospif(p[1] * (1.0f / 180.0f), &sg, &cg);
    sincospif(p[2] * (1.0f / 90.0f), &ind.s2x, &ind.c2x);
    const float h = eta0 * (0.5f * FAD_INV_SQRTPI);
    ind.kA = h * sg * sg;
    ind.kB = h * 0.5f * fmaf(cg, cg, 1.0f);
    ind.kC = h * cg;
    ind.fad = fad_const(a);
    ind.S0 = p[7];
    ind.muS1 = mu * p[8];
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        if (NL == ME_MAX_LINES && l >= d.n_lines) { ind.invD[l] = ind.v0[l] = ind.vB[l] = 0.f; continue; }
        const float inv = 1.0f / (dld * d.line[l].dld_scale);
        ind.invD[l] = inv;
        ind.v0[l] = -(d.line[l].lam0_over_c * vlos) * inv;
        ind.vB[l] = d.line[l].zeeman * B * inv;
    }
}

// Profile sums of one line at reduced wavelength v:  S_kind += r_l * sum_c weight_c * w(v - shift_c vB + i a)
template <bool TRIPLET>
__device__ __forceinline__ void line_profiles(float v, float vB, const FadConst& fad, const SynthDesc& d, int l,
                                              float& br, float& bi, float& pr, float& pi, float& rr, float& ri) {
    const float r = d.line[l].strength;
    if (TRIPLET) {
        const float gvB = d.line[l].g * vB;
        float w0r, w0i, w1r, w1i, w2r, w2i;
        faddeeva32(v, fad, w0r, w0i);
        faddeeva32(v + gvB, fad, w1r, w1i);      // sigma_blue sits at v = -g vB
        faddeeva32(v - gvB, fad, w2r, w2i);      // sigma_red  sits at v = +g vB
        pr = fmaf(r, w0r, pr); pi = fmaf(r, w0i, pi);
        br = fmaf(r, w1r, br); bi = fmaf(r, w1i, bi);
        rr = fmaf(r, w2r, rr); ri = fmaf(r, w2i, ri);
    } else {
        const int* kb = d.line[l].kind_begin;
        for (int c = kb[0]; c < kb[1]; ++c) {
            float wr, wi; faddeeva32(fmaf(-d.shift[c], vB, v), fad, wr, wi);
            const float s = r * d.weight[c]; br = fmaf(s, wr, br); bi = fmaf(s, wi, bi);
        }
        for (int c = kb[1]; c < kb[2]; ++c) {
            float wr, wi; faddeeva32(fmaf(-d.shift[c], vB, v), fad, wr, wi);
            const float s = r * d.weight[c]; pr = fmaf(s, wr, pr); pi = fmaf(s, wi, pi);
        }
        for (int c = kb[2]; c < kb[3]; ++c) {
            float wr, wi; faddeeva32(fmaf(-d.shift[c], vB, v), fad, wr, wi);
            const float s = r * d.weight[c]; rr = fmaf(s, wr, rr); ri = fmaf(s, wi, ri);
        }
    }
}

// Stokes vector at wavelength index j (eq. 8 + eq. 12-13 times I_c of eq. 15).
// The Unno-Rachkovsky solution is evaluated in the frame chi = 0 (eta_U = rho_U = 0) and Q,U are rotated by 2 chi.
template <int NL, bool TRIPLET>
__device__ __forceinline__ void stokes_at(const Individual<NL>& ind, const SynthDesc& d, int j,
                                          float& I, float& Q, float& U, float& V) {
    float br = 0.f, bi = 0.f, pr = 0.f, pi = 0.f, rr = 0.f, ri = 0.f;
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        if (NL == ME_MAX_LINES && l >= d.n_lines) break;      // NL == ME_MAX_LINES is the run-time-sized fallback
        const float v = fmaf(d.off[l][j], ind.invD[l], ind.v0[l]);
        line_profiles<TRIPLET>(v, ind.vB[l], ind.fad, d, l, br, bi, pr, pi, rr, ri);
    }
    const float sr = br + rr, si = bi + ri;                       // sigma sum
    const float eI = fmaf(ind.kA, pr, fmaf(ind.kB, sr, 1.0f));
    const float eL = ind.kA * fmaf(-0.5f, sr, pr);                // eta_Q in the chi = 0 frame
    const float rL = ind.kA * fmaf(-0.5f, si, pi);                // rho_Q in the chi = 0 frame
    const float eV = ind.kC * (rr - br);
    const float rV = ind.kC * (ri - bi);
    const float eI2 = eI * eI;
    const float Pi = fmaf(eL, rL, eV * rV);
    const float rho2 = fmaf(rL, rL, rV * rV);
    const float eta2 = fmaf(eL, eL, eV * eV);
    const float Delta = fmaf(eI2, eI2 + (rho2 - eta2), -Pi * Pi);
    const float t = ind.muS1 * rcp_approx(Delta);
    I = fmaf(t * eI, eI2 + rho2, ind.S0);
    const float Qp = -t * fmaf(eI2, eL, rL * Pi);
    const float Up = -t * eI * fmaf(eL, rV, -eV * rL);
    V = -t * fmaf(eI2, eV, rV * Pi);
    Q = fmaf(Qp, ind.c2x, -Up * ind.s2x);
    U = fmaf(Qp, ind.s2x, Up * ind.c2x);
}

// ------------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al. 2011): counter (c0..c3), key (k0,k1) -> 4 x u32.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// uniform in [0,1) from the top 24 bits (exact in binary32)
__device__ __forceinline__ float u01(uint32_t x) { return (float)(x >> 8) * (1.0f / 16777216.0f); }
// integer in [0, n): floor(u * n) in integer arithmetic
__device__ __forceinline__ int below(uint32_t x, int n) { return (int)__umulhi(x & 0xffffff00u, (uint32_t)n); }

__device__ __forceinline__ uint32_t lane_of(const uint4& r, int k) {
    return k == 0 ? r.x : (k == 1 ? r.y : (k == 2 ? r.z : r.w));
}

// ------------------------------------------------------------------------------------------------------------
// GA operators (readings G1-G3).  All gene arithmetic is single IEEE binary32 operations or one fma, written with
// intrinsics so that the compiler cannot re-associate or contract differently from the specification.
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float decode_gene(float g, const GaDesc& c, int j) {
    if (c.log_scale[j]) return c.lo[j] * exp2f(g * c.log2ratio[j]);
    return fmaf(c.span[j], g, c.lo[j]);
}

// generation 0, gene j: lane (j mod 4) of block floor(j / 4)
__device__ __forceinline__ void init_genes(float* g, uint32_t pixel, uint32_t i, const GaDesc& c) {
#pragma unroll
    for (int k = 0; k < (ME_NPAR + 3) / 4; ++k) {
        const uint4 r = philox4x32_10(pixel, 0u, i, (uint32_t)k, c.key0, c.key1);
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (4 * k + q < ME_NPAR) g[4 * k + q] = u01(lane_of(r, q));
    }
}

// k-way tournament with replacement on chi2[] (shared memory): smallest chi2 wins, ties -> smallest index.
__device__ __forceinline__ int tournament(const uint4& r, const float* chi2, const GaDesc& c) {
    int best = below(r.x, c.pop);
    float fb = chi2[best];
    for (int m = 1; m < c.tournament_k; ++m) {
        const int cand = below(lane_of(r, m), c.pop);
        const float fc = chi2[cand];
        if (fc < fb || (fc == fb && cand < best)) { best = cand; fb = fc; }
    }
    return best;
}

// Child i >= 1 of generation t from the previous population `genes` [pop][ME_NPAR] and its fitness `chi2` [pop].
__device__ __forceinline__ void make_child(float* child, const float* genes, const float* chi2, uint32_t pixel,
                                           uint32_t t, uint32_t i, float s_t, const GaDesc& c) {
    const int A = tournament(philox4x32_10(pixel, t, i, 0u, c.key0, c.key1), chi2, c);
    const int B = tournament(philox4x32_10(pixel, t, i, 1u, c.key0, c.key1), chi2, c);
    const uint4 rc = philox4x32_10(pixel, t, i, 2u, c.key0, c.key1);
    const bool cross = u01(rc.x) < c.p_cross;
    const float alpha = u01(rc.y);
    uint4 rm = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int j = 0; j < ME_NPAR; ++j) {
        const float gA = genes[A * ME_NPAR + j], gB = genes[B * ME_NPAR + j];
        float g = gA;
        if (cross) g = __fmaf_rn(alpha, __fsub_rn(gA, gB), gB);
        if ((j & 1) == 0) rm = philox4x32_10(pixel, t, i, (uint32_t)(3 + j / 2), c.key0, c.key1);
        const float um = u01((j & 1) ? rm.z : rm.x), ud = u01((j & 1) ? rm.w : rm.y);
        if (um < c.p_mut) g = __fmaf_rn(s_t, __fsub_rn(__fmul_rn(2.0f, ud), 1.0f), g);
        if (c.periodic[j]) g = __fsub_rn(g, floorf(g));
        else g = fminf(fmaxf(g, 0.0f), 1.0f);
        child[j] = g;
    }
}

}  // namespace me
