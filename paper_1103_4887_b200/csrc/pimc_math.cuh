// Branch-free double-precision elementary functions for the PIMC kernels.
//
// Why not libdevice: exp/tanh/log/sincos/division from the CUDA math library carry special-case branches
// (BSSY/BSYNC/BRA), materialise every polynomial coefficient with two UMOVs and serialise the three
// independent gate evaluations of the Hodgkin-Huxley right-hand side.  In the v1 profile
// (profiles/r01_v1_baseline.md) only 34 % of the executed warp instructions were FP64-pipe instructions.
// These versions assume what the sampler guarantees (finite, range-limited arguments), keep coefficients in
// constant memory (a free DFMA operand) and contain no branches, so the compiler can interleave independent
// chains.  Each is accurate to about 1 ulp, far inside the 1e-12 Delta-A tolerance; tests/test_gpu_math.py
// checks them against the host libm through the pimc_math_selftest entry point.
#pragma once
#include <cuda_runtime.h>

namespace pimc {

#define PIMC_COEF(name, n) static __constant__ double name[n]      // one copy per translation unit
#include "pimc_math_coef.inc"
#undef PIMC_COEF

__device__ __forceinline__ double rcp_seed(double d) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    return y;
}
__device__ __forceinline__ double rsqrt_seed(double d) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));
    return y;
}

// 1/d for normal d (no zero / inf / nan handling): MUFU seed (~20 bits) + two Newton steps.
__device__ __forceinline__ double rcp_fast(double d) {
    double y = rcp_seed(d);
    double e = fma(-d, y, 1.0);
    y = fma(y, e, y);
    e = fma(-d, y, 1.0);
    y = fma(y, e, y);
    return y;
}
// n/d with one residual correction of the quotient.
__device__ __forceinline__ double div_fast(double n, double d) {
    const double y = rcp_fast(d);
    const double q = n * y;
    const double r = fma(-d, q, n);
    return fma(r, y, q);
}

// e^r - 1 for |r| <= ~0.36: r + r^2 P(r), P of degree 9 evaluated by Estrin's scheme (dependent depth 5 instead of 11).
__device__ __forceinline__ double expm1_small(double r) {
    const double r2 = r * r;
    const double a0 = fma(kExpP[1], r, kExpP[0]);
    const double a1 = fma(kExpP[3], r, kExpP[2]);
    const double a2 = fma(kExpP[5], r, kExpP[4]);
    const double a3 = fma(kExpP[7], r, kExpP[6]);
    const double a4 = fma(kExpP[9], r, kExpP[8]);
    const double r4 = r2 * r2;
    const double b0 = fma(a1, r2, a0);
    const double b1 = fma(a3, r2, a2);
    const double r8 = r4 * r4;
    const double c0 = fma(b1, r4, b0);
    const double p = fma(a4, r8, c0);
    return fma(p, r2, r);
}

// exp(x) for |x| <= 700: x = k ln2 + r, |r| <= ln2/2; scale by 2^k through the exponent field.
__device__ __forceinline__ double exp_fast(double x) {
    constexpr double kMagic = 6755399441055744.0;                 // 1.5 * 2^52: adds round-to-nearest-integer
    constexpr double kLog2e = 1.4426950408889634074;
    constexpr double kLn2Hi = 0x1.62e42fefa39efp-1, kLn2Lo = 0x1.abc9e3b39803fp-56;
    const double t = fma(x, kLog2e, kMagic);
    const int k = __double2loint(t);
    const double kd = t - kMagic;
    double r = fma(kd, -kLn2Hi, x);
    r = fma(kd, -kLn2Lo, r);
    const double e = expm1_small(r);                               // e^r - 1
    const double s = __hiloint2double((k + 1023) << 20, 0);        // 2^k
    return fma(e, s, s);
}

// exp(c1 V + c0) for any finite V with the result SATURATED to [2^-300, 2^301): used where only e/(1+e)-type
// ratios of the result matter (the Hodgkin-Huxley gates), which are exact to rounding long before saturation.
// The clamp is integer arithmetic on k, off the floating-point dependency chain.  Requires |c1 V + c0| < 2^31 ln 2
// (the caller guards).
template <int KMAX> __device__ __forceinline__ double exp_affine_sat_k(double V, double c1, double c0);
__device__ __forceinline__ double exp_affine_sat(double V, double c1, double c0) { return exp_affine_sat_k<300>(V, c1, c0); }
// the same with the scale clamped to 2^+-KMAX
template <int KMAX> __device__ __forceinline__ double exp_affine_sat_k(double V, double c1, double c0) {
    constexpr double kMagic = 6755399441055744.0;
    constexpr double kLog2e = 1.4426950408889634074;
    constexpr double kLn2Hi = 0x1.62e42fefa39efp-1, kLn2Lo = 0x1.abc9e3b39803fp-56;
    const double x = fma(V, c1, c0);
    const double t = fma(x, kLog2e, kMagic);
    int k = __double2loint(t);
    const double kd = t - kMagic;
    double r = fma(kd, -kLn2Hi, x);
    r = fma(kd, -kLn2Lo, r);
    const double e = expm1_small(r);
    k = min(max(k, -KMAX), KMAX);
    const double s = __hiloint2double((k + 1023) << 20, 0);
    return fma(e, s, s);
}

// num / den for normal den: MUFU seed y0 (measured relative error ~2^-13), then
// num y0 (1 + e + e^2 + e^3 + e^4) with e = 1 - den y0 (relative error e^5 < 2^-64): four dependent FP64 operations
// after the seed, and the numerator rides along for free.
__device__ __forceinline__ double div_series(double num, double den) {
    const double y0 = rcp_seed(den);
    const double e = fma(-den, y0, 1.0);
    const double t = num * y0;
    const double p = fma(e, e, e);
    const double e2 = e * e;
    const double S = fma(p, e2, p);
    return fma(t, S, t);
}

// exp(x) - 1 for |x| <= 700, accurate near 0: same reduction as exp_fast; with k = 0 the result is the polynomial itself,
// otherwise 2^k (1 + e) - 1 = e 2^k + (2^k - 1) with 2^k - 1 exact (|k| <= 52) or absorbed (larger |k|).
__device__ __forceinline__ double expm1_fast(double x) {
    constexpr double kMagic = 6755399441055744.0;
    constexpr double kLog2e = 1.4426950408889634074;
    constexpr double kLn2Hi = 0x1.62e42fefa39efp-1, kLn2Lo = 0x1.abc9e3b39803fp-56;
    const double t = fma(x, kLog2e, kMagic);
    const int k = __double2loint(t);
    const double kd = t - kMagic;
    double r = fma(kd, -kLn2Hi, x);
    r = fma(kd, -kLn2Lo, r);
    const double e = expm1_small(r);
    const double s = __hiloint2double((k + 1023) << 20, 0);
    return fma(e, s, s - 1.0);
}
// u / (1 - exp(-u)) with its removable singularity at u = 0 (value 1); |u| <= 700
__device__ __forceinline__ double u_over_1mexp(double u) {
    const double d = -expm1_fast(-u);
    const double q = div_fast(u, d);
    return u == 0.0 ? 1.0 : q;
}

// ---- single precision (the fp32 variant of config 3) -----------------------------------------------------------
// exp(x) SATURATED to [2^-60, 2^61) (so that its square stays finite in fp32): x = k ln2 + r, |r| <= ln2/2,
// e^r = 1 + r + r^2 Q(r) with Q of degree 5 (truncation < 2e-8 relative); k clamped in integer arithmetic.
template <int KMAX> __device__ __forceinline__ float expf_sat_k(float x);
__device__ __forceinline__ float expf_sat(float x) { return expf_sat_k<60>(x); }
template <int KMAX> __device__ __forceinline__ float expf_sat_k(float x) {
    constexpr float kMagic = 12582912.0f;                          // 1.5 * 2^23
    constexpr float kLog2e = 1.44269504088896341f;
    constexpr float kLn2Hi = 0.693145751953125f, kLn2Lo = 1.42860682030941723e-6f;   // hi has 12 trailing zero bits
    const float t = fmaf(x, kLog2e, kMagic);
    int k = __float_as_int(t) - __float_as_int(kMagic);
    const float kd = t - kMagic;
    float r = fmaf(kd, -kLn2Hi, x);
    r = fmaf(kd, -kLn2Lo, r);
    const float r2 = r * r;
    const float a0 = fmaf(1.0f / 6.0f, r, 0.5f);
    const float a1 = fmaf(1.0f / 120.0f, r, 1.0f / 24.0f);
    const float a2 = fmaf(1.0f / 5040.0f, r, 1.0f / 720.0f);
    const float r4 = r2 * r2;
    const float b = fmaf(a1, r2, a0);
    const float p = fmaf(a2, r4, b);
    const float e = fmaf(p, r2, r);                                // e^r - 1
    k = min(max(k, -KMAX), KMAX);
    const float s = __int_as_float((k + 127) << 23);               // 2^k
    return fmaf(e, s, s);
}
// num / den for normal den: MUFU reciprocal (1 ulp) + one Newton step
__device__ __forceinline__ float divf_fast(float num, float den) {
    float y0;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(den));
    const float e = fmaf(-den, y0, 1.0f);
    const float y = fmaf(y0, e, y0);
    return num * y;
}

// log(u) for normal positive u (here u in (0,1)): u = m 2^e, m in [sqrt(1/2), sqrt(2)); log m = 2 atanh((m-1)/(m+1)).
__device__ __forceinline__ double log_fast(double u) {
    constexpr double kLn2Hi = 6.93147180369123816490e-01, kLn2Lo = 1.90821492927058770002e-10;   // hi has 21 trailing zero bits
    int hi = __double2hiint(u);
    const int lo = __double2loint(u);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000FFFFF) | 0x3FF00000;                           // m in [1,2)
    const int big = hi >= 0x3FF6A09F ? 1 : 0;                      // m >= ~sqrt(2): halve it
    hi -= big << 20;
    e += big;
    const double m = __hiloint2double(hi, lo);
    const double f = div_fast(m - 1.0, m + 1.0);
    const double w = f * f;
    double L = kLogL[8];
#pragma unroll
    for (int i = 7; i >= 0; --i) L = fma(L, w, kLogL[i]);
    const double lm = fma(f * w, L, f + f);                        // 2 f + f^3 L(w)
    const double ed = (double)e;
    return fma(ed, kLn2Hi, fma(ed, kLn2Lo, lm));
}

// sqrt(x) for normal positive x: MUFU seed, two coupled Newton steps on (sqrt, 1/(2 sqrt)), one residual correction.
__device__ __forceinline__ double sqrt_fast(double x) {
    const double y = rsqrt_seed(x);
    double g = x * y, h = 0.5 * y;
    double r = fma(-h, g, 0.5);
    g = fma(g, r, g); h = fma(h, r, h);
    r = fma(-h, g, 0.5);
    g = fma(g, r, g); h = fma(h, r, h);
    const double d = fma(-g, g, x);
    return fma(d, h, g);
}

// sin and cos of a in [0, 8): a = k pi/2 + r, |r| <= pi/4.
__device__ __forceinline__ void sincos_fast(double a, double& s_out, double& c_out) {
    constexpr double kMagic = 6755399441055744.0;
    constexpr double kTwoOverPi = 0.63661977236758134308;
    constexpr double kPio2Hi = 0x1.921fb54442d18p+0, kPio2Lo = 0x1.1a62633145c07p-54;
    const double t = fma(a, kTwoOverPi, kMagic);
    const int k = __double2loint(t);
    const double kd = t - kMagic;
    double r = fma(kd, -kPio2Hi, a);
    r = fma(kd, -kPio2Lo, r);
    const double w = r * r;
    double S = kSinS[5], C = kCosC[5];
#pragma unroll
    for (int i = 4; i >= 0; --i) { S = fma(S, w, kSinS[i]); C = fma(C, w, kCosC[i]); }
    const double s = fma(r * w, S, r);
    const double c = fma(w * w, C, fma(w, -0.5, 1.0));
    const double sa = (k & 1) ? c : s, ca = (k & 1) ? s : c;
    s_out = (k & 2) ? -sa : sa;
    c_out = ((k + 1) & 2) ? -ca : ca;
}

}  // namespace pimc
