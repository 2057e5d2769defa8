// me_device.cuh — device-side building blocks of libme_b200.so (sm_100a, FP32).
//
//   faddeeva_pair   w(v + i a) = H + iF on two wavelengths, two-region FP32 evaluator
//   Individual      per-parameter-vector constants hoisted out of the wavelength loop (eq. 14)
//   stokes_pair     absorption matrix (eq. 8) + Unno-Rachkovsky solution (eq. 12-13, 15) at two wavelengths
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
    float smax;             // largest |shift| of the line's components (outermost Zeeman component, Lorentz units)
    int pad;
};

struct alignas(16) SynthDesc {
    int L, n_lines, n_comp, all_triplets;
    int npar, pad0;                       // 9, or 11 (fill fraction + stray light, reading F13)
    const float* nm_profile;              // device [L]: I_fixed of the 11-parameter model, else nullptr
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
    float lo[ME_MAX_NPAR], span[ME_MAX_NPAR], log2ratio[ME_MAX_NPAR];
    int log_scale[ME_MAX_NPAR], periodic[ME_MAX_NPAR];
    float mut_scale[ME_MAX_GEN + 1];    // s_t, t = 0..generations
    // per-pixel prologue (readings W1, P1, S1): bit 0 inverse-max weights, bit 1 polarity restriction, bit 2 seeds
    int prologue;
    int seed_line;                      // S1: the line with the largest g lambda^2
    float seed_hw;                      // half-width of its window (half the distance to the nearest other line, or +Inf)
    float seed_scale;                   // 1 / (2 C g lambda^2)   [G per A]
    float w_cfg[4], sigma[4];           // configured w_s and sigma_s (w2 above is (w_s / sigma_s)^2)
    // variant 1 (the paper's binary-coded GA, readings V0-V5 of DESIGN.md)
    int variant;                        // 0 real-coded operators, 1 binary-coded
    int n_samp;                         // restart period max(1, G / 4)
    uint32_t sobol_v[ME_MAX_NPAR][16];  // Sobol' direction numbers v_1..v_16 per dimension (point indices < 2^16)
};

// ------------------------------------------------------------------------------------------------------------
// Packed FP32 helpers.  Blackwell (sm_100) issues two FP32 FMAs per instruction (FFMA2 / FMUL2 / FADD2); the FMA
// pipe is as wide as before, so packing halves the ISSUE slots of the arithmetic.  The fitness loop is issue-bound
// (profiles/r1_history.md, step r1a), so everything per wavelength is written on pairs of adjacent wavelengths (j, j+1) held in float2.
// Scalars broadcast for free (SASS operand form R.F32), negation is an operand modifier.
// ------------------------------------------------------------------------------------------------------------
typedef float2 f2;
#define MEDEV __device__ __forceinline__

MEDEV f2 bc(float s) { return make_float2(s, s); }
MEDEV f2 neg(f2 a) { return make_float2(-a.x, -a.y); }
MEDEV f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
MEDEV f2 fma2(float a, f2 b, f2 c) { return __ffma2_rn(bc(a), b, c); }
MEDEV f2 fma2(f2 a, f2 b, float c) { return __ffma2_rn(a, b, bc(c)); }
MEDEV f2 fma2(float a, f2 b, float c) { return __ffma2_rn(bc(a), b, bc(c)); }
MEDEV f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
MEDEV f2 mul2(float a, f2 b) { return __fmul2_rn(bc(a), b); }
MEDEV f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
MEDEV f2 sub2(f2 a, f2 b) { return __fadd2_rn(a, neg(b)); }

MEDEV float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
MEDEV f2 rcp2(f2 a) { return make_float2(rcp_approx(a.x), rcp_approx(a.y)); }

// Real-coefficient polynomial at a complex argument x by the quadratic-factor recurrence
//   b_k = c_k + t b_{k+1} + m b_{k+2},  t = 2 Re x,  m = -|x|^2;   P(x) = (b_0 - b_1 Re x) + i b_1 Im x
// (x^2 = t x + m): two FMAs per coefficient instead of four for a complex Horner step.
#define ME_REC(bk, ck, b1, b2) const f2 bk = fma2(t, b1, fma2(m, b2, ck))

// ------------------------------------------------------------------------------------------------------------
// Faddeeva function w(v + i a) = H + iF on a pair of v, FP32, two regions.
//   wing |z|^2 >= CUT2: w = (i/sqrt(pi)) s R(q), s = 1/z, q = s^2, R = asymptotic series to q^5 (q^3, q^2 farther out).  H comes out as
//                       a/(sqrt(pi)|z|^2) x (1 + ...): no cancellation, full relative accuracy.
//   core |z|^2 <  CUT2: Weideman (1994), N = FAD_N terms in Z = (L + iz)/(L - iz).
// ------------------------------------------------------------------------------------------------------------
struct FadConst { float a, a2, m4a2, La, Lma, La2, Lma2, t4LLa; };

MEDEV FadConst fad_const(float a) {
    FadConst f;
    f.a = a; f.a2 = a * a; f.m4a2 = -4.0f * f.a2;
    f.La = FAD_L + a; f.Lma = FAD_L - a; f.La2 = f.La * f.La; f.Lma2 = f.Lma * f.Lma;
    f.t4LLa = 2.0f * FAD_2L * f.La;
    return f;
}

// Wing region.  With t = 2 Re q, m = -|q|^2 the recurrence gives R(q) = b0 - b1 conj(q); since s conj(q) = |s|^2 conj(s)
// and |s|^2 = r = 1/|z|^2:   w = i s R = r [ a (b0 + r b1) + i v (b0 - r b1) ]   (no cancellation in H).
// K = number of series terms beyond the leading one: 5 for |z| >= FAD_CUT, 2 for >= FAD_W2 (used as written only when
// a > FAD_FAR_AMAX; otherwise the far tier below).  An intermediate K = 3 tier (|z| >= 7.5) was measured and dropped: it
// saved 0.7 % of the arithmetic and cost more than that in code size (profiles/r1_history.md, step r1e).
template <int K>
MEDEV void faddeeva_wing(f2 v, f2 r2, const FadConst& f, f2& wr, f2& wi) {
    const f2 r = rcp2(r2);                                    // 1/|z|^2
    const f2 t = mul2(fma2(f.m4a2, r, 2.0f), r);              // 2 Re q = 2 (v^2 - a^2)/|z|^4 = (2 - 4 a^2 r) r
    const f2 m = mul2(neg(r), r);                             // -|q|^2 = -1/|z|^4
    f2 b0, b1;
    if (K == 2) {
        b1 = fma2(t, bc(FAD_C2), FAD_C1);
        b0 = fma2(t, b1, fma2(m, bc(FAD_C2), FAD_C0));
    } else if (K == 3) {
        const f2 b2 = fma2(t, bc(FAD_C3), FAD_C2);
        b1 = fma2(t, b2, fma2(m, bc(FAD_C3), FAD_C1));
        b0 = fma2(t, b1, fma2(m, b2, FAD_C0));
    } else {
        const f2 b4 = fma2(t, bc(FAD_C5), FAD_C4);
        const f2 b3 = fma2(t, b4, fma2(m, bc(FAD_C5), FAD_C3));
        ME_REC(b2, FAD_C2, b3, b4);
        b1 = fma2(t, b2, fma2(m, b3, FAD_C1));
        b0 = fma2(t, b1, fma2(m, b2, FAD_C0));
    }
    wr = mul2(mul2(f.a, r), fma2(r, b1, b0));
    wi = mul2(mul2(v, r), fma2(neg(r), b1, b0));
}

// Far tiers (|z| >= FAD_FAR, a <= FAD_FAR_AMAX): the asymptotic series regrouped as polynomials in r = 1/|z|^2 alone.
// With s = r (v - i a) and v^2 = 1/r - a^2 every term of (i/sqrt(pi)) c_k s^(2k+1) is a polynomial in r and A = a^2:
//   H = a r X(r; A),  X = C0 [1 + (3/2) r + (15/4 - 2 A) r^2 + (105/8 - 15 A) r^3 + ...]
//   F = v r Y(r; A),  Y = C0 [1 + (1/2) r + ( 3/4 - 2 A) r^2 + ( 15/8 -  9 A) r^3 + ...]
// and on r in [0, 1/T^2] the series is cut to a low degree by truncating its Chebyshev expansion on that interval
// (economisation; gen_faddeeva_table.py), which is a linear map of the series coefficients: the economised coefficients
// are again polynomials in A with tabulated constants (FAD_CUB_*, FAD_LIN_*), evaluated once per parameter vector.
//   cubic  tier, |z| >= FAD_FAR = 5:      max |dH| 1.5e-8, |dF| 5.9e-8 against scipy.special.wofz over a <= FAD_FAR_AMAX
//   linear tier, |z| >= FAD_FAR_LIN = 12: max |dH| 4.8e-8, |dF| 2.2e-7
// (rounds 1-2 cut the q^2 series by plain truncation: quadratics from |z| = 9 with 6.4e-8 / 4.0e-7, linear from |z| = 20, and
// a q^5 series evaluated per component between 5 and 9 at twice the cost of the cubic).  Each Horner step is FFMA2
// (pair x pair + scalar) -- the full-rate operand form (profiles/r1_history.md, step r1c: an FFMA2 whose ADDEND is a register
// pair runs at 0.77 of that rate) -- and the line strength r_l and the factor a are folded into the coefficients.
struct FarCoef { float x3, x2, x1, x0, y3, y2, y1, y0, lx1, lx0, ly1, ly0; };

// the economised coefficients for damping a, without the line strength: X rows carry the factor a
MEDEV FarCoef far_base(float a) {
    constexpr float CX[4][FAD_FAR_PA + 1] = FAD_CUB_X, CY[4][FAD_FAR_PA + 1] = FAD_CUB_Y;
    constexpr float LX[2][FAD_FAR_PA + 1] = FAD_LIN_X, LY[2][FAD_FAR_PA + 1] = FAD_LIN_Y;
    const float A = a * a;
    float cx[4], cy[4], lx[2], ly[2];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float x = CX[j][FAD_FAR_PA], y = CY[j][FAD_FAR_PA];
#pragma unroll
        for (int p = FAD_FAR_PA - 1; p >= 0; --p) { x = fmaf(x, A, CX[j][p]); y = fmaf(y, A, CY[j][p]); }
        cx[j] = a * x; cy[j] = y;
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        float x = LX[j][FAD_FAR_PA], y = LY[j][FAD_FAR_PA];
#pragma unroll
        for (int p = FAD_FAR_PA - 1; p >= 0; --p) { x = fmaf(x, A, LX[j][p]); y = fmaf(y, A, LY[j][p]); }
        lx[j] = a * x; ly[j] = y;
    }
    FarCoef c;
    c.x0 = cx[0]; c.x1 = cx[1]; c.x2 = cx[2]; c.x3 = cx[3]; c.y0 = cy[0]; c.y1 = cy[1]; c.y2 = cy[2]; c.y3 = cy[3];
    c.lx0 = lx[0]; c.lx1 = lx[1]; c.ly0 = ly[0]; c.ly1 = ly[1];
    return c;
}

MEDEV FarCoef far_scale(const FarCoef& b, float strength) {
    FarCoef c;
    c.x0 = strength * b.x0; c.x1 = strength * b.x1; c.x2 = strength * b.x2; c.x3 = strength * b.x3;
    c.y0 = strength * b.y0; c.y1 = strength * b.y1; c.y2 = strength * b.y2; c.y3 = strength * b.y3;
    c.lx0 = strength * b.lx0; c.lx1 = strength * b.lx1; c.ly0 = strength * b.ly0; c.ly1 = strength * b.ly1;
    return c;
}

// accumulates r_l w(v + i a) into (sr, si); LINEAR: the tier beyond FAD_FAR_LIN
template <bool LINEAR>
MEDEV void faddeeva_far_acc(f2 v, f2 r2, const FarCoef& c, f2& sr, f2& si) {
    const f2 r = rcp2(r2);
    const f2 X = LINEAR ? fma2(bc(c.lx1), r, c.lx0) : fma2(fma2(fma2(bc(c.x3), r, c.x2), r, c.x1), r, c.x0);
    const f2 Y = LINEAR ? fma2(bc(c.ly1), r, c.ly0) : fma2(fma2(fma2(bc(c.y3), r, c.y2), r, c.y1), r, c.y0);
    sr = fma2(r, X, sr);
    si = fma2(mul2(v, r), Y, si);
}

// The same coefficients parked in shared memory (three float4 rows per thread and line: the linear tier's, the cubic tier's X
// and Y) and re-loaded inside the far branch that uses them: in registers they do not fit next to the fitness loop's working
// set and the compiler rematerialises them with scalar FMULs on the FMA pipe (profiles/r1_history.md, step r1e); an LDS.128
// costs no FMA-pipe slot, and the linear tier (most line-pairs) needs one.
#define ME_FAR_ROWS 3
template <bool LINEAR>
MEDEV FarCoef far_load(unsigned addr, int stride_bytes) {
    FarCoef c;
    // "memory": the compiler must not sink or drop far_store's plain stores, which only these loads read.  addr is this
    // thread's column as a 32-bit shared address held in a register (keep_in_register below); stride_bytes is a constant.
    float4 x, y = make_float4(0.f, 0.f, 0.f, 0.f);
    if (LINEAR) {
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "r"(addr) : "memory");
        c.lx1 = x.x; c.lx0 = x.y; c.ly1 = x.z; c.ly0 = x.w;
        c.x3 = c.x2 = c.x1 = c.x0 = c.y3 = c.y2 = c.y1 = c.y0 = 0.f;
    } else {
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "r"(addr + stride_bytes) : "memory");
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(y.x), "=f"(y.y), "=f"(y.z), "=f"(y.w) : "r"(addr + 2 * stride_bytes) : "memory");
        c.x3 = x.x; c.x2 = x.y; c.x1 = x.z; c.x0 = x.w; c.y3 = y.x; c.y2 = y.y; c.y1 = y.z; c.y0 = y.w;
        c.lx1 = c.lx0 = c.ly1 = c.ly0 = 0.f;
    }
    return c;
}
// A loop-invariant value the compiler would otherwise RE-COMPUTE inside the wavelength loop to save a register (ncu r2c:
// S2R + LEA + 3 moves per far-tier branch for the shared address, FSETP + MOV + FSEL per pair for the far threshold =
// 6.4 of 112 instructions per wavelength point).  An empty asm with the value as in/out operand makes it opaque.
MEDEV void keep_in_register(unsigned& x) { asm volatile("" : "+r"(x)); }
MEDEV void keep_in_register(float& x) { asm volatile("" : "+f"(x)); }
MEDEV void far_store(float4* p, int stride, const FarCoef& c) {
    p[0] = make_float4(c.lx1, c.lx0, c.ly1, c.ly0);
    p[stride] = make_float4(c.x3, c.x2, c.x1, c.x0);
    p[2 * stride] = make_float4(c.y3, c.y2, c.y1, c.y0);
}

// Core region (Weideman).  D = 1/(L - iz) = r ((L+a) + i v), r = 1/|L - iz|^2, Z = (L + iz) D.  With t = 2 Re Z,
// m = -|Z|^2 the recurrence gives p(Z) = b0 - b1 conj(Z), and conj(Z) D = r conj(L + iz), so
//   p D = r [ (b0 (L+a) - b1 (L-a)) + i v (b0 + b1) ],     w = D (p D + 1/sqrt(pi)).
MEDEV void faddeeva_core(f2 v, const FadConst& f, f2& wr, f2& wi) {
    const f2 v2 = mul2(v, v);
    const f2 r = rcp2(add2(v2, bc(f.La2)));                   // 1/|L - iz|^2
    const f2 t = fma2(f.t4LLa, r, -2.0f);                     // 2 Re Z = 2 (2 L (L+a) r - 1)
    const f2 m = mul2(neg(add2(v2, bc(f.Lma2))), r);          // -|Z|^2 = -|L + iz|^2 / |L - iz|^2
    FAD_CORE_RECURRENCE(t, m)
    const f2 X = fma2(r, fma2(f.La, cb0, mul2(-f.Lma, cb1)), FAD_INV_SQRTPI);   // Re(p D) + 1/sqrt(pi)
    const f2 Y = mul2(mul2(r, v), add2(cb0, cb1));                                // Im(p D)
    wr = mul2(r, fma2(f.La, X, neg(mul2(v, Y))));
    wi = mul2(r, fma2(f.La, Y, mul2(v, X)));
}

MEDEV void faddeeva_pair(f2 v, const FadConst& f, f2& wr, f2& wi) {
    const f2 r2 = fma2(v, v, f.a2);
    const bool w0 = r2.x >= FAD_CUT2, w1 = r2.y >= FAD_CUT2;
    if (w0 || w1) faddeeva_wing<5>(v, r2, f, wr, wi);
    if (!(w0 && w1)) {
        f2 cr, ci;
        faddeeva_core(v, f, cr, ci);
        if (!w0) { wr.x = cr.x; wi.x = ci.x; }
        if (!w1) { wr.y = cr.y; wi.y = ci.y; }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Per-individual constants (decode-time work, once per parameter vector).
// ------------------------------------------------------------------------------------------------------------
template <int NL>
struct Individual {
    FadConst fad;
    FarCoef far[NL];                  // far-tier polynomial coefficients per line (strength and a folded in)
    float tfar;                       // far-tier threshold on dv = min|v| - g vB: FAD_FAR, or +Inf when a > FAD_FAR_AMAX
    float invD[NL], v0[NL], vB[NL];   // 1/dlambdaD_l, -doppler_l/dlambdaD_l, Zeeman splitting in Doppler units
    float kA, kB, kC;                 // h sin^2(gamma), h (1 + cos^2 gamma)/2, h cos(gamma);  h = eta0 / (2 sqrt(pi))
    float c2x, s2x;                   // cos 2chi, sin 2chi
    float S0, muS1;                   // 11-parameter model: (1-s) S0 and (1-s) alpha mu S1
    float k0, nmS1, stray;            // 11-parameter model only: eta0/sqrt(pi), (1-s)(1-alpha) mu S1, s
    unsigned far_addr;                // FARS: 32-bit shared address of this thread's far coefficients, [ME_FAR_ROWS l + {0,1,2}] * far_stride
    int far_stride;                   //       stride in BYTES between consecutive float4 rows (16 * threads per block)
};

// p: decoded parameter vector, M = 9 or 11 entries.  For M = 11 (reading F13)
//   I = (1-s)[alpha I^M + (1-alpha) I(B=0)] + s I_fixed
//     = (1-s) S0 + [(1-s) alpha mu S1] (K^-1 e)_I + [(1-s)(1-alpha) mu S1] / (1 + eta0 phi_nm) + s I_fixed,
// and Q, U, V carry the factor (1-s) alpha: both are obtained by rescaling S0 and mu S1 here.
// triplet: ind.vB[l] holds g_l vB_l, the sigma shift itself (the only form the triplet path uses; r2d: one FMUL per line and pair)
template <int NL, int M>
MEDEV void setup_individual(Individual<NL>& ind, const float* p, float mu, const SynthDesc& d, bool triplet = false) {
    const float B = p[0], eta0 = p[3], dld = p[4], a = p[5], vlos = p[6];
    float sg, cg;
    sincospif(p[1] * (1.0f / 180.0f), &sg, &cg);
    sincospif(p[2] * (1.0f / 90.0f), &ind.s2x, &ind.c2x);
    const float h = eta0 * (0.5f * FAD_INV_SQRTPI);
    ind.kA = h * sg * sg;
    ind.kB = h * 0.5f * fmaf(cg, cg, 1.0f);
    ind.kC = h * cg;
    ind.fad = fad_const(a);
    ind.tfar = a <= FAD_FAR_AMAX ? FAD_FAR : __int_as_float(0x7f800000);
    keep_in_register(ind.tfar);
    ind.S0 = p[7];
    ind.muS1 = mu * p[8];
    ind.k0 = ind.nmS1 = ind.stray = 0.f;
    if (M == ME_MAX_NPAR) {
        const float alpha = p[9], s = p[10], oms = 1.0f - s;
        ind.k0 = 2.0f * h;
        ind.nmS1 = oms * (1.0f - alpha) * ind.muS1;
        ind.muS1 = oms * alpha * ind.muS1;
        ind.S0 = oms * ind.S0;
        ind.stray = s;
    }
    const FarCoef fbase = far_base(a);
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        if (NL == ME_MAX_LINES && l >= d.n_lines) { ind.invD[l] = ind.v0[l] = ind.vB[l] = 0.f; ind.far[l] = far_scale(fbase, 0.f); continue; }
        ind.far[l] = far_scale(fbase, d.line[l].strength);
        const float inv = 1.0f / (dld * d.line[l].dld_scale);
        ind.invD[l] = inv;
        ind.v0[l] = -(d.line[l].lam0_over_c * vlos) * inv;
        ind.vB[l] = d.line[l].zeeman * B * inv;
        if (triplet) ind.vB[l] *= d.line[l].g;
    }
}

// Profile sums of one line at a pair of reduced wavelengths v:
//   S_kind += r_l * sum_c weight_c * w(v - shift_c vB + i a)
template <bool TRIPLET, bool FARS>
MEDEV void line_profiles(f2 v, float vB, const FadConst& fad, const FarCoef& far_r, unsigned far_addr, int far_stride,
                         float tfar, const SynthDesc& d, int l, f2& br, f2& bi, f2& pr, f2& pi, f2& rr, f2& ri) {
    const float r = d.line[l].strength;
    if (TRIPLET) {
        const float gvB = vB;                                      // g vB, formed once per individual (setup_individual)
        f2 w0r, w0i, w1r, w1i, w2r, w2i;
        const f2 vb = add2(v, bc(gvB)), vr = add2(v, bc(-gvB));   // sigma_blue sits at v = -g vB, sigma_red at +g vB
        // Tier of the whole line at this pair: the three components sit at 0, -+g vB, so the one nearest to either
        // wavelength is at distance >= dv = min(|v.x|, |v.y|) - g vB, and dv >= T guarantees |z| >= T for all six arguments.
        // (r2c: the minimum over the six |z|^2 cost 3 FMNMX + up to 4 FSETP per line and pair; this is 1 FMNMX + 1 FADD.)
        const float dv = fminf(fabsf(v.x), fabsf(v.y)) - gvB;
        // When all six arguments lie in one wing tier (the common case) the three evaluations are independent
        // straight-line code that the scheduler interleaves; the series shortens with distance from the line.
        if (dv >= tfar) {
            const f2 r2p = fma2(v, v, fad.a2), r2b = fma2(vb, vb, fad.a2), r2r = fma2(vr, vr, fad.a2);
            if (dv >= FAD_FAR_LIN) {
                const FarCoef far = FARS ? far_load<true>(far_addr + ME_FAR_ROWS * l * far_stride, far_stride) : far_r;
                faddeeva_far_acc<true>(v, r2p, far, pr, pi);
                faddeeva_far_acc<true>(vb, r2b, far, br, bi);
                faddeeva_far_acc<true>(vr, r2r, far, rr, ri);
            } else {
                const FarCoef far = FARS ? far_load<false>(far_addr + ME_FAR_ROWS * l * far_stride, far_stride) : far_r;
                faddeeva_far_acc<false>(v, r2p, far, pr, pi);
                faddeeva_far_acc<false>(vb, r2b, far, br, bi);
                faddeeva_far_acc<false>(vr, r2r, far, rr, ri);
            }
            return;
        }
        if (dv >= FAD_W2) {                                       // a > FAD_FAR_AMAX: the series itself, cut after q^2
            const f2 r2p = fma2(v, v, fad.a2), r2b = fma2(vb, vb, fad.a2), r2r = fma2(vr, vr, fad.a2);
            faddeeva_wing<2>(v, r2p, fad, w0r, w0i);
            faddeeva_wing<2>(vb, r2b, fad, w1r, w1i);
            faddeeva_wing<2>(vr, r2r, fad, w2r, w2i);
        } else if (dv >= FAD_CUT) {
            const f2 r2p = fma2(v, v, fad.a2), r2b = fma2(vb, vb, fad.a2), r2r = fma2(vr, vr, fad.a2);
            faddeeva_wing<5>(v, r2p, fad, w0r, w0i);
            faddeeva_wing<5>(vb, r2b, fad, w1r, w1i);
            faddeeva_wing<5>(vr, r2r, fad, w2r, w2i);
        } else {
            faddeeva_pair(v, fad, w0r, w0i);
            faddeeva_pair(vb, fad, w1r, w1i);
            faddeeva_pair(vr, fad, w2r, w2i);
        }
        pr = fma2(r, w0r, pr); pi = fma2(r, w0i, pi);
        br = fma2(r, w1r, br); bi = fma2(r, w1i, bi);
        rr = fma2(r, w2r, rr); ri = fma2(r, w2i, ri);
    } else {
        // General component list (full Zeeman patterns).  Every component sits within smax |vB| of the
        // line centre, so the smallest |z|^2 over all of them and both wavelengths is bounded below by
        // (max(0, min|v| - smax |vB|))^2 + a^2: one tier for the whole line, chosen without touching the components.
        const int* kb = d.line[l].kind_begin;
        const float dv = fminf(fabsf(v.x), fabsf(v.y)) - d.line[l].smax * fabsf(vB);
        const FarCoef far = far_r;
        const int tier = dv >= tfar ? 2 : (dv >= FAD_CUT ? 1 : 0);
#pragma unroll 1
        for (int k = 0; k < 3; ++k) {                              // k = 0 blue, 1 pi, 2 red
            f2 ar = bc(0.f), ai = bc(0.f);
            if (tier == 2) {
                for (int c = kb[k]; c < kb[k + 1]; ++c) {
                    const f2 vc = add2(v, bc(-d.shift[c] * vB));
                    const f2 rr_ = rcp2(fma2(vc, vc, fad.a2));                        // 1 / |z|^2
                    const f2 rw = mul2(d.weight[c], rr_);                             // weight_c / |z|^2
                    const f2 X = fma2(fma2(fma2(bc(far.x3), rr_, far.x2), rr_, far.x1), rr_, far.x0);
                    const f2 Y = fma2(fma2(fma2(bc(far.y3), rr_, far.y2), rr_, far.y1), rr_, far.y0);
                    ar = fma2(rw, X, ar);
                    ai = fma2(mul2(vc, rw), Y, ai);
                }
            } else if (tier == 1) {
                for (int c = kb[k]; c < kb[k + 1]; ++c) {
                    const f2 vc = add2(v, bc(-d.shift[c] * vB));
                    f2 wr, wi; faddeeva_wing<5>(vc, fma2(vc, vc, fad.a2), fad, wr, wi);
                    const float sw = r * d.weight[c]; ar = fma2(sw, wr, ar); ai = fma2(sw, wi, ai);
                }
            } else {
                for (int c = kb[k]; c < kb[k + 1]; ++c) {
                    f2 wr, wi; faddeeva_pair(add2(v, bc(-d.shift[c] * vB)), fad, wr, wi);
                    const float sw = r * d.weight[c]; ar = fma2(sw, wr, ar); ai = fma2(sw, wi, ai);
                }
            }
            if (k == 0) { br = add2(br, ar); bi = add2(bi, ai); }
            else if (k == 1) { pr = add2(pr, ar); pi = add2(pi, ai); }
            else { rr = add2(rr, ar); ri = add2(ri, ai); }
        }
    }
}

// Stokes vectors at the wavelength pair (j0, j1) (eq. 8 + eq. 12-13 times I_c of eq. 15).  j1 = j0 + 1 with j0 even
// in the main loop (one 8-byte constant-bank load per line); j1 = j0 for the odd tail.
// The Unno-Rachkovsky solution is evaluated in the frame chi = 0 (eta_U = rho_U = 0) and Q,U are rotated by 2 chi.
// M = 11: nmF = I_fixed at the two wavelengths; the field-free profile sum phi_nm = sum_l r_l H(a, v_l) is the pi sum of
// effective triplets (their pi component is unshifted with weight 1), else one extra Voigt per line.
// RES: on entry I, Q, U, V hold the OBSERVED values at the pair; on return they hold the residuals observed - model, formed
// by the last FMA of each Stokes parameter instead of a separate subtraction (the fused fitness needs nothing else).
template <int NL, bool TRIPLET, int M, bool FARS = false, bool RES = false>
MEDEV void stokes_pair(const Individual<NL>& ind, const SynthDesc& d, int j0, bool tail, f2 nmF, f2& I, f2& Q, f2& U, f2& V,
                       const f2* offp = nullptr, const f2* vpre = nullptr) {
    f2 br = bc(0.f), bi = bc(0.f), pr = bc(0.f), pi = bc(0.f), rr = bc(0.f), ri = bc(0.f), nr = bc(0.f);
#pragma unroll
    for (int l = 0; l < NL; ++l) {
        if (NL == ME_MAX_LINES && l >= d.n_lines) break;      // NL == ME_MAX_LINES is the run-time-sized fallback
        f2 v;
        if (vpre != nullptr) v = vpre[l];                     // reduced wavelengths formed by the caller (fused fitness)
        else {
            const f2 off = offp != nullptr ? offp[l] : (tail ? bc(d.off[l][j0]) : *reinterpret_cast<const f2*>(&d.off[l][j0]));
            v = fma2(ind.invD[l], off, ind.v0[l]);
        }
        line_profiles<TRIPLET, FARS>(v, ind.vB[l], ind.fad, ind.far[l], ind.far_addr, ind.far_stride, ind.tfar, d, l, br, bi,
                                     pr, pi, rr, ri);
        if (M == ME_MAX_NPAR && !TRIPLET) {
            f2 wr, wi;
            faddeeva_pair(v, ind.fad, wr, wi);
            nr = fma2(d.line[l].strength, wr, nr);
        }
    }
    if (M == ME_MAX_NPAR && TRIPLET) nr = pr;
    const f2 sr = add2(br, rr), si = add2(bi, ri);                // sigma sums
    const f2 eI = fma2(ind.kA, pr, fma2(ind.kB, sr, 1.0f));
    const f2 eL = mul2(ind.kA, fma2(-0.5f, sr, pr));              // eta_Q in the chi = 0 frame
    const f2 rL = mul2(ind.kA, fma2(-0.5f, si, pi));              // rho_Q in the chi = 0 frame
    const f2 eV = mul2(ind.kC, sub2(rr, br));
    const f2 rV = mul2(ind.kC, sub2(ri, bi));
    // r2d: this tail is the largest consumer of the FMA pipe, which limits the kernel (31 % of its lane-slots, two thirds of
    // them bare FMUL2 / FADD2).  eI^2 + rho^2 and eI^2 + rho^2 - eta^2 are formed by chained FMAs, -mu S1 eI / Delta is shared
    // between I and U, and in RES mode the subtraction from the observation is the last FMA of each Stokes parameter.
    const f2 E2 = mul2(eI, eI);
    const f2 A = fma2(rL, rL, fma2(rV, rV, E2));                  // eta_I^2 + rho_Q^2 + rho_V^2
    const f2 Bq = fma2(neg(eL), eL, fma2(neg(eV), eV, A));        // ... - eta_Q^2 - eta_V^2
    const f2 Pi = fma2(eL, rL, mul2(eV, rV));
    const f2 Delta = fma2(E2, Bq, neg(mul2(Pi, Pi)));
    const f2 nt = mul2(-ind.muS1, rcp2(Delta));                   // -mu S1 / Delta
    const f2 nteI = mul2(nt, eI);
    const f2 Qp = mul2(nt, fma2(E2, eL, mul2(rL, Pi)));
    const f2 Up = mul2(nteI, fma2(eL, rV, neg(mul2(eV, rL))));
    const f2 Vn = fma2(E2, eV, mul2(rV, Pi));
    if (!RES) {
        I = fma2(neg(nteI), A, ind.S0);
        V = mul2(nt, Vn);
        Q = fma2(ind.c2x, Qp, mul2(-ind.s2x, Up));
        U = fma2(ind.s2x, Qp, mul2(ind.c2x, Up));
        if (M == ME_MAX_NPAR) {
            const f2 rn = rcp2(fma2(ind.k0, nr, 1.0f));           // 1 / (1 + eta0 phi_nm): pin P1
            I = fma2(ind.nmS1, rn, fma2(ind.stray, nmF, I));
        }
    } else {
        I = add2(fma2(nteI, A, I), bc(-ind.S0));                  // obs_I - (S0 - nt eI A)
        V = fma2(neg(nt), Vn, V);
        Q = fma2(-ind.c2x, Qp, fma2(ind.s2x, Up, Q));
        U = fma2(-ind.s2x, Qp, fma2(-ind.c2x, Up, U));
        if (M == ME_MAX_NPAR) {
            const f2 rn = rcp2(fma2(ind.k0, nr, 1.0f));
            I = fma2(-ind.nmS1, rn, fma2(-ind.stray, nmF, I));
        }
    }
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

// Gene value in [0,1] from the stored gene: the real-coded variant stores it; the binary-coded variant stores the 16-bit
// code k as an integer-valued float and decodes g = k / (2^16 - 1) (eq. 5) with one IEEE division.
__device__ __forceinline__ float gene_value(float stored, const GaDesc& c) {
    return c.variant ? __fdiv_rn(stored, 65535.0f) : stored;
}

// ---- variant 1: Sobol' points (Bratley & Fox 1988 as the paper uses them) -----------------------
// Point n of dimension j in Gray-code order, top 16 bits, xor the per-pixel digital shift (reading V1).
template <int M>
__device__ __forceinline__ void sobol_genes(float* g, uint32_t pixel, uint32_t n, const GaDesc& c) {
    const uint32_t gray = n ^ (n >> 1);
    uint4 r = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int j = 0; j < M; ++j) {
        if ((j & 3) == 0) r = philox4x32_10(pixel, 0u, 0xFFFFFFFFu, (uint32_t)(j >> 2), c.key0, c.key1);
        uint32_t x = 0, q = gray;
        while (q) {
            const int b = __ffs(q) - 1;
            x ^= c.sobol_v[j][b];
            q &= q - 1;
        }
        g[j] = (float)(((x >> 16) ^ (lane_of(r, j & 3) >> 16)) & 0xFFFFu);
    }
}

__device__ __forceinline__ int tournament(const uint4& r, const float* chi2, const GaDesc& c);

// k-way tournament among the n_live best (order[rank] = member index); reading V2/V3.
__device__ __forceinline__ int tournament_live(const uint4& r, const float* chi2, const uint16_t* order, int n_live,
                                               const GaDesc& c) {
    int best = order[below(r.x, n_live)];
    float fb = chi2[best];
    for (int m = 1; m < c.tournament_k; ++m) {
        const int cand = order[below(lane_of(r, m), n_live)];
        const float fc = chi2[cand];
        if (fc < fb || (fc == fb && cand < best)) { best = cand; fb = fc; }
    }
    return best;
}

// Child i >= 1 of generation t, binary-coded (readings V2, V4, V5).  order == nullptr: every member is live.
template <int M>
__device__ __forceinline__ void make_child_binary(float* child, const float* genes, const float* chi2,
                                                  const uint16_t* order, int n_live, uint32_t pixel, uint32_t t,
                                                  uint32_t i, const GaDesc& c) {
    if ((int)i >= n_live) {                                   // restart: the next points of the shifted Sobol' sequence
        const int n_dead = c.pop - n_live;
        sobol_genes<M>(child, pixel, (uint32_t)(c.pop + ((int)t / c.n_samp - 1) * n_dead + ((int)i - n_live) + 1), c);
        return;
    }
    const uint32_t key = 2u * ((i + 1u) >> 1) - 1u;           // the pair (2q-1, 2q) shares its parents and its cut
    int A, B;
    if (order != nullptr) {
        A = tournament_live(philox4x32_10(pixel, t, key, 0u, c.key0, c.key1), chi2, order, n_live, c);
        B = tournament_live(philox4x32_10(pixel, t, key, 1u, c.key0, c.key1), chi2, order, n_live, c);
    } else {
        A = tournament(philox4x32_10(pixel, t, key, 0u, c.key0, c.key1), chi2, c);
        B = tournament(philox4x32_10(pixel, t, key, 1u, c.key0, c.key1), chi2, c);
    }
    const uint4 rc = philox4x32_10(pixel, t, key, 2u, c.key0, c.key1);
    const bool cross = u01(rc.x) < c.p_cross;
    const int cut = 1 + below(rc.y, 16 * M - 1);
    const int first = (i & 1u) ? A : B, second = (i & 1u) ? B : A;
    uint4 rm = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int j = 0; j < M; ++j) {
        const uint32_t k1 = (uint32_t)genes[first * M + j], k2 = (uint32_t)genes[second * M + j];
        uint32_t k = k1;
        if (cross) {
            const int nhead = min(max(cut - 16 * j, 0), 16);  // bits taken from the first parent, MSB side
            const uint32_t mask = (0xFFFFu << (16 - nhead)) & 0xFFFFu;
            k = (k1 & mask) | (k2 & ~mask & 0xFFFFu);
        }
        if ((j & 1) == 0) rm = philox4x32_10(pixel, t, i, (uint32_t)(3 + j / 2), c.key0, c.key1);
        const uint32_t xm = (j & 1) ? rm.z : rm.x, xd = (j & 1) ? rm.w : rm.y;
        if (u01(xm) < c.p_mut) k ^= ((xd & 0xFFFFu) & (xd >> 16)) >> (xm & 15u);
        child[j] = (float)k;
    }
}

// Rank of member i by (chi2, index): the number of members that come before it.  O(pop) shared-memory reads.
__device__ __forceinline__ int rank_of(const float* chi2, int pop, int i) {
    const float fi = chi2[i];
    int r = 0;
    for (int k = 0; k < pop; ++k) {
        const float fk = chi2[k];
        r += (fk < fi || (fk == fi && k < i)) ? 1 : 0;
    }
    return r;
}

// generation 0, gene j: lane (j mod 4) of block floor(j / 4)
template <int M>
__device__ __forceinline__ void init_genes(float* g, uint32_t pixel, uint32_t i, const GaDesc& c) {
#pragma unroll
    for (int k = 0; k < (M + 3) / 4; ++k) {
        const uint4 r = philox4x32_10(pixel, 0u, i, (uint32_t)k, c.key0, c.key1);
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (4 * k + q < M) g[4 * k + q] = u01(lane_of(r, q));
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

// Child i >= 1 of generation t from the previous population `genes` [pop][M] and its fitness `chi2` [pop].
template <int M>
__device__ __forceinline__ void make_child(float* child, const float* genes, const float* chi2, uint32_t pixel,
                                           uint32_t t, uint32_t i, float s_t, const GaDesc& c) {
    const int A = tournament(philox4x32_10(pixel, t, i, 0u, c.key0, c.key1), chi2, c);
    const int B = tournament(philox4x32_10(pixel, t, i, 1u, c.key0, c.key1), chi2, c);
    const uint4 rc = philox4x32_10(pixel, t, i, 2u, c.key0, c.key1);
    const bool cross = u01(rc.x) < c.p_cross;
    const float alpha = u01(rc.y);
    uint4 rm = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int j = 0; j < M; ++j) {
        const float gA = genes[A * M + j], gB = genes[B * M + j];
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

// Stage obs[n] ([4][L] in HBM, rows contiguous) into shared memory, pair-interleaved:
// element (s, j) -> word 8 (j/2) + 2 s + (j & 1).  Shared size: 8 * ceil(L/2) floats.
// L % 4 == 0 (and a 16-byte aligned cube): one coalesced LDG.128 per thread (streaming, read once: no L1 allocation)
// and two 8-byte shared stores; otherwise element-wise.
__device__ __forceinline__ void stage_obs(float* obs_s, const float* obs_n, int L, int tid, int nthreads) {
    if ((L & 3) == 0 && (reinterpret_cast<uintptr_t>(obs_n) & 15) == 0) {
        for (int k4 = tid; k4 < L; k4 += nthreads) {
            const int k = 4 * k4, s = k / L, j = k - s * L;     // the four values sit in one Stokes row (L % 4 == 0)
            float4 x;
            asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "l"(obs_n + k));
            *reinterpret_cast<float2*>(obs_s + 8 * (j >> 1) + 2 * s) = make_float2(x.x, x.y);
            *reinterpret_cast<float2*>(obs_s + 8 * ((j >> 1) + 1) + 2 * s) = make_float2(x.z, x.w);
        }
        return;
    }
    for (int k = tid; k < 4 * L; k += nthreads) {
        const int s = k / L, j = k - s * L;
        obs_s[8 * (j >> 1) + 2 * s + (j & 1)] = __ldg(obs_n + k);
    }
}

// Per-pixel prologue (readings W1, P1; eq. 20-23, polarity PAPER.md:278), run by ONE warp on the staged
// observation (pair-interleaved layout of stage_obs).  pix[0..3] = (w_s / sigma_s)^2, pix[4] = gamma_lo, pix[5] = gamma
// span, pix[6] = gamma_hi; without flags these are the configured values.  Bit 2 (reading S1): pix[7],
// pix[8] = stored genes (B, gamma) of the centre-of-gravity member, pix[9] = B_los [G]; `off` = sd.off[gd.seed_line].
#define ME_PIX_WORDS 16
__device__ __forceinline__ void pixel_prologue(const float* obs_s, int L, const GaDesc& gd, float* pix, bool writer,
                                               const float* off = nullptr) {
    const int lane = threadIdx.x & 31;
    const float INF = __int_as_float(0x7f800000);
    float imax = -INF, imin = INF, mq = 0.f, mu_ = 0.f, mv = 0.f, vmax = -INF, vmin = INF;
    int jmax = 0x7fffffff, jmin = 0x7fffffff;
#pragma unroll 1
    for (int j = lane; j < L; j += 32) {                        // ascending j per lane: strict compare keeps the first
        const float* o = obs_s + 8 * (j >> 1) + (j & 1);
        const float I = o[0], Q = o[2], U = o[4], V = o[6];
        imax = fmaxf(imax, I); imin = fminf(imin, I);
        mq = fmaxf(mq, fabsf(Q)); mu_ = fmaxf(mu_, fabsf(U)); mv = fmaxf(mv, fabsf(V));
        if (V > vmax) { vmax = V; jmax = j; }
        if (V < vmin) { vmin = V; jmin = j; }
    }
#pragma unroll 1
    for (int s = 16; s > 0; s >>= 1) {
        imax = fmaxf(imax, __shfl_xor_sync(0xffffffffu, imax, s)); imin = fminf(imin, __shfl_xor_sync(0xffffffffu, imin, s));
        mq = fmaxf(mq, __shfl_xor_sync(0xffffffffu, mq, s)); mu_ = fmaxf(mu_, __shfl_xor_sync(0xffffffffu, mu_, s));
        mv = fmaxf(mv, __shfl_xor_sync(0xffffffffu, mv, s));
        const float ov = __shfl_xor_sync(0xffffffffu, vmax, s); const int oj = __shfl_xor_sync(0xffffffffu, jmax, s);
        if (ov > vmax || (ov == vmax && oj < jmax)) { vmax = ov; jmax = oj; }
        const float pv = __shfl_xor_sync(0xffffffffu, vmin, s); const int pj = __shfl_xor_sync(0xffffffffu, jmin, s);
        if (pv < vmin || (pv == vmin && pj < jmin)) { vmin = pv; jmin = pj; }
    }
    if (writer) {
        float glo = gd.lo[1], ghi = __fadd_rn(gd.lo[1], gd.span[1]);
        if (gd.prologue & 1) {
            const float den[4] = {fmaxf(imax - imin, gd.sigma[0]), fmaxf(mq, gd.sigma[1]), fmaxf(mu_, gd.sigma[2]), fmaxf(mv, gd.sigma[3])};
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const float w = __fdiv_rn(__fdiv_rn(1.0f, den[s]), gd.sigma[s]);
                pix[s] = w * w;
            }
        } else {
#pragma unroll
            for (int s = 0; s < 4; ++s) pix[s] = gd.w2[s];
        }
        if (gd.prologue & 2) {
            if (jmax < jmin) ghi = fminf(ghi, 90.0f);
            else glo = fmaxf(glo, 90.0f);
        }
        pix[4] = glo; pix[5] = (gd.prologue & 2) ? ghi - glo : gd.span[1]; pix[6] = ghi;
    }
    if ((gd.prologue & 4) && off != nullptr) {               // S1: centre of gravity of I +- V (Rees & Semel 1979)
        float sp = 0.f, sm = 0.f, lp = 0.f, lm = 0.f;
#pragma unroll 1
        for (int j = lane; j < L; j += 32) {
            const float dl = off[j];
            if (fabsf(dl) > gd.seed_hw) continue;
            const float* o = obs_s + 8 * (j >> 1) + (j & 1);
            const float ap = imax - (o[0] + o[6]), am = imax - (o[0] - o[6]);
            sp += ap; sm += am; lp = fmaf(dl, ap, lp); lm = fmaf(dl, am, lm);
        }
#pragma unroll 1
        for (int s = 16; s > 0; s >>= 1) {
            sp += __shfl_xor_sync(0xffffffffu, sp, s); sm += __shfl_xor_sync(0xffffffffu, sm, s);
            lp += __shfl_xor_sync(0xffffffffu, lp, s); lm += __shfl_xor_sync(0xffffffffu, lm, s);
        }
        if (writer) {
            float blos = 0.f;
            if (sp > 0.f && sm > 0.f) blos = (lp / sp - lm / sm) * gd.seed_scale;
            const float hiB = gd.log_scale[0] ? gd.lo[0] * exp2f(gd.log2ratio[0]) : gd.lo[0] + gd.span[0];
            const float b = fminf(fmaxf(fabsf(blos), gd.lo[0]), hiB);
            float u = 0.f;
            if (gd.log_scale[0]) { if (gd.log2ratio[0] != 0.f) u = log2f(b / gd.lo[0]) / gd.log2ratio[0]; }
            else if (gd.span[0] != 0.f) u = (b - gd.lo[0]) / gd.span[0];
            const float qb = rintf(u * 1023.0f), qg = blos >= 0.f ? 0.f : 1023.0f;
            pix[7] = gd.variant ? 64.0f * qb : __fdiv_rn(qb, 1023.0f);
            pix[8] = gd.variant ? 64.0f * qg : __fdiv_rn(qg, 1023.0f);
            pix[9] = blos;
        }
    }
}

// Reading S2: the weak-field member "as in Auer et al. (1977)", prologue bit 8, run like
// pixel_prologue by every warp on the staged observation; the writer fills pix[10..12] = stored genes (B, gamma, chi) and
// pix[13] = B_los [G].  pix[4], pix[6] (the pixel's inclination box) must have been written by the same thread before.
//   B_los from the separation of the I+V and I-V line cores (parabola vertex at the first minimum), chi and gamma from the
//   maxima of Q^2 + U^2, |V|, |I'|, |I''| on the interior samples of the seed line's window; off = lambda_j - lambda_0.
__device__ __forceinline__ void pixel_seed_auer(const float* obs_s, int L, const GaDesc& gd, float* pix, bool writer,
                                                const float* off) {
    const int lane = threadIdx.x & 31;
    const float INF = __int_as_float(0x7f800000), hw = gd.seed_hw;
    const int NONE = 0x7fffffff;
    float yp = INF, ym = INF, D1 = 0.f, D2 = 0.f, Vm = 0.f, L2m = -1.f;
    int jp = NONE, jm = NONE, jL = NONE;
#pragma unroll 1
    for (int j = lane; j < L; j += 32) {                         // ascending j per lane: strict compares keep the first
        const float dj = off[j];
        if (fabsf(dj) > hw) continue;
        const float* o = obs_s + 8 * (j >> 1) + (j & 1);
        const float I = o[0], V = o[6];
        const float a = I + V, b = I - V;
        if (a < yp) { yp = a; jp = j; }
        if (b < ym) { ym = b; jm = j; }
        if (j >= 1 && j + 1 < L && fabsf(off[j - 1]) <= hw && fabsf(off[j + 1]) <= hw) {       // interior sample
            const float hm = dj - off[j - 1], hp = off[j + 1] - dj;
            const float Im = obs_s[8 * ((j - 1) >> 1) + ((j - 1) & 1)], Ip = obs_s[8 * ((j + 1) >> 1) + ((j + 1) & 1)];
            const float d1 = (Ip - Im) / (hm + hp);
            const float d2 = 2.0f * ((Ip - I) / hp - (I - Im) / hm) / (hm + hp);
            D1 = fmaxf(D1, fabsf(d1)); D2 = fmaxf(D2, fabsf(d2)); Vm = fmaxf(Vm, fabsf(V));
            const float l2 = fmaf(o[2], o[2], o[4] * o[4]);
            if (l2 > L2m) { L2m = l2; jL = j; }
        }
    }
#pragma unroll 1
    for (int s = 16; s > 0; s >>= 1) {
        D1 = fmaxf(D1, __shfl_xor_sync(0xffffffffu, D1, s)); D2 = fmaxf(D2, __shfl_xor_sync(0xffffffffu, D2, s));
        Vm = fmaxf(Vm, __shfl_xor_sync(0xffffffffu, Vm, s));
        float ov = __shfl_xor_sync(0xffffffffu, yp, s); int oj = __shfl_xor_sync(0xffffffffu, jp, s);
        if (ov < yp || (ov == yp && oj < jp)) { yp = ov; jp = oj; }
        ov = __shfl_xor_sync(0xffffffffu, ym, s); oj = __shfl_xor_sync(0xffffffffu, jm, s);
        if (ov < ym || (ov == ym && oj < jm)) { ym = ov; jm = oj; }
        ov = __shfl_xor_sync(0xffffffffu, L2m, s); oj = __shfl_xor_sync(0xffffffffu, jL, s);
        if (ov > L2m || (ov == L2m && oj < jL)) { L2m = ov; jL = oj; }
    }
    if (!writer) return;
    pix[10] = pix[11] = pix[12] = pix[13] = 0.f;
    if (jp == NONE) return;                                      // empty window
    auto at = [&](int st, int j) { return obs_s[8 * (j >> 1) + 2 * st + (j & 1)]; };
    auto interior = [&](int j) { return j >= 1 && j + 1 < L && fabsf(off[j - 1]) <= hw && fabsf(off[j]) <= hw && fabsf(off[j + 1]) <= hw; };
    float core[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {                                // 1. line cores of I + V (k = 0) and I - V (k = 1)
        const float sg = k == 0 ? 1.0f : -1.0f, y1 = k == 0 ? yp : ym;
        const int j = k == 0 ? jp : jm;
        float x = off[j];
        if (interior(j)) {                                       // vertex of the parabola through the minimum and its neighbours
            const float y0 = at(0, j - 1) + sg * at(3, j - 1), y2 = at(0, j + 1) + sg * at(3, j + 1);
            const float a0 = x - off[j - 1], a2 = x - off[j + 1];
            const float num = a0 * a0 * (y1 - y2) - a2 * a2 * (y1 - y0), den = a0 * (y1 - y2) - a2 * (y1 - y0);
            if (den != 0.f) x -= 0.5f * num / den;
        }
        core[k] = x;
    }
    const float blos = (core[0] - core[1]) * gd.seed_scale;      // seed_scale = 1 / (2 C g lambda0^2)
    float QL = 0.f, UL = 0.f, d2L = 0.f;                         // 3. azimuth at the maximum of the linear polarisation
    if (jL != NONE) {
        const float hm = off[jL] - off[jL - 1], hp = off[jL + 1] - off[jL];
        d2L = 2.0f * ((at(0, jL + 1) - at(0, jL)) / hp - (at(0, jL) - at(0, jL - 1)) / hm) / (hm + hp);
        QL = at(1, jL); UL = at(2, jL);
    } else L2m = 0.f;
    const float s = d2L >= 0.f ? -1.0f : 1.0f;
    float chi = 0.5f * atan2f(s * UL, s * QL) * 57.29577951308232f;
    if (chi < 0.f) chi += 180.0f;
    if (chi >= 180.0f) chi -= 180.0f;
    float gp = 90.0f;                                            // 4. inclination from the L / V amplitude ratio
    if (Vm > 0.f && D2 > 0.f) gp = atanf(2.0f * sqrtf(sqrtf(L2m)) * D1 / (Vm * sqrtf(D2))) * 57.29577951308232f;
    const float glo = pix[4], ghi = pix[6];
    float gam = blos >= 0.f ? gp : 180.0f - gp;
    if (gam < glo || gam > ghi) gam = 180.0f - gam;              // the seed is checked against the polarity box
    gam = fminf(fmaxf(gam, glo), ghi);
    const float cg = fmaxf(fabsf(cospif(gam * (1.0f / 180.0f))), 0.125f);      // 5. field strength
    const float hiB = gd.log_scale[0] ? gd.lo[0] * exp2f(gd.log2ratio[0]) : gd.lo[0] + gd.span[0];
    const float b = fminf(fmaxf(fabsf(blos) / cg, gd.lo[0]), hiB);
    float uB = 0.f;
    if (gd.log_scale[0]) { if (gd.log2ratio[0] != 0.f) uB = log2f(b / gd.lo[0]) / gd.log2ratio[0]; }
    else if (gd.span[0] != 0.f) uB = (b - gd.lo[0]) / gd.span[0];
    const float ug = ghi > glo ? (gam - glo) / (ghi - glo) : 0.f;
    const float chic = fminf(fmaxf(chi, gd.lo[2]), gd.lo[2] + gd.span[2]);
    const float uc = gd.span[2] > 0.f ? (chic - gd.lo[2]) / gd.span[2] : 0.f;
    const float q[3] = {rintf(fminf(fmaxf(uB, 0.f), 1.f) * 1023.0f), rintf(fminf(fmaxf(ug, 0.f), 1.f) * 1023.0f),
                        rintf(fminf(fmaxf(uc, 0.f), 1.f) * 1023.0f)};
#pragma unroll
    for (int k = 0; k < 3; ++k) pix[10 + k] = gd.variant ? 64.0f * q[k] : __fdiv_rn(q[k], 1023.0f);
    pix[13] = blos;
}

// Block-wide argmin of (value, index) with ties -> lowest index. Values must be >= 0 or +Inf.
// scratch: 2 * 32 words of shared memory. Every thread returns the same (value, index).
__device__ __forceinline__ void block_argmin(float v, int idx, uint32_t* scratch, float& vmin, int& imin) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    uint32_t bits = __float_as_uint(v);
    uint32_t m = __reduce_min_sync(0xffffffffu, bits);
    uint32_t i = __reduce_min_sync(0xffffffffu, bits == m ? (uint32_t)idx : 0xffffffffu);
    if (lane == 0) { scratch[warp] = m; scratch[32 + warp] = i; }
    __syncthreads();
    const uint32_t mb = lane < nwarps ? scratch[lane] : 0xffffffffu;
    const uint32_t ib = lane < nwarps ? scratch[32 + lane] : 0xffffffffu;
    m = __reduce_min_sync(0xffffffffu, mb);
    i = __reduce_min_sync(0xffffffffu, mb == m ? ib : 0xffffffffu);
    vmin = __uint_as_float(m);
    imin = (int)i;
    __syncthreads();          // scratch may be reused by the next call
}

}  // namespace me
