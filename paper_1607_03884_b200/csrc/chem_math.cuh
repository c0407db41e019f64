// chem_math.cuh -- compact fp64 elementary functions shared by all kernels of the path.
#pragma once
#include <cuda_runtime.h>

namespace chem {

__device__ __forceinline__ double rcp_nr(double x)   // 1/x for normal x: MUFU seed + two Newton steps
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
}


constexpr double kLn10 = 2.302585092994045684, kInvLn10 = 0.4342944819032518277;

// Compact fp64 elementary functions for normal, finite arguments (the rates, temperatures and step-size ratios of
// this path).  Polynomial coefficients sit in constant memory so that each Horner step is ONE DFMA with a constant-bank
// operand (the libdevice versions spend two UMOVs per coefficient and are 2-3x larger, which matters for the 32 KB
// instruction cache).  Accuracy ~1-2 ulp; no special-case handling beyond what is stated.
static __constant__ double kExpC[14] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
                                 1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};
static __constant__ double kAtanhC[11] = {2.0, 2.0 / 3, 2.0 / 5, 2.0 / 7, 2.0 / 9, 2.0 / 11, 2.0 / 13, 2.0 / 15, 2.0 / 17, 2.0 / 19, 2.0 / 21};

// 1/x for normal x (rcp_nr above): hardware seed + two Newton steps; no denormal / zero / inf handling
__device__ __forceinline__ double rcp_f(double x) { return rcp_nr(x); }
// a / b with one residual correction (<= 1 ulp for normal operands)
__device__ __forceinline__ double div_f(double a, double b)
{
    const double r = rcp_f(b);
    const double q = a * r;
    return fma(fma(-b, q, a), r, q);
}
// sqrt(x) for normal x > 0: rsqrt seed + Newton, final Heron correction
__device__ __forceinline__ double sqrt_f(double x)
{
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double h = 0.5 * r;
    double g = x * r;                       // ~sqrt(x)
    double e = fma(-g, h, 0.5);
    g = fma(g, e, g);
    const double h2 = fma(h, e, h);
    e = fma(-g, g, x);
    return fma(e, h2, g);
}
// sqrt for x >= 0 including 0; NaN / negative -> NaN, inf -> NaN (both "non-finite" for the controller, R11)
__device__ __forceinline__ double sqrt_s(double x)
{
    return x > 1e-300 ? sqrt_f(x) : (x >= 0.0 ? 0.0 : __longlong_as_double(0x7ff8000000000000LL));
}
// exp(x): x = n ln2 + r, |r| <= ln2/2, Taylor degree 13; returns 0 below -700, inf above 709
__device__ __forceinline__ double exp_f(double x)
{
    const double t = fma(x, 1.4426950408889634074, 6755399441055744.0);      // round(x / ln2) in the low word
    const int n = __double2loint(t);
    const double fn = t - 6755399441055744.0;
    double r = fma(fn, -6.93147180369123816490e-01, x);
    r = fma(fn, -1.90821492927058770002e-10, r);
    double p = kExpC[13];
#pragma unroll
    for (int k = 12; k >= 0; k--) p = fma(p, r, kExpC[k]);
    // scale by 2^n in two steps so that n down to -1074 + ... stays correct enough; clamp the far tails
    const int n1 = n >> 1, n2 = n - n1;
    p *= __hiloint2double((1023 + n1) << 20, 0);
    p *= __hiloint2double((1023 + n2) << 20, 0);
    if (x < -700.0) p = 0.0;
    if (x > 709.0) p = __longlong_as_double(0x7ff0000000000000LL);
    return p;
}
// log(x) for normal x > 0: x = 2^e m, m in [sqrt(1/2), sqrt(2)), log m = 2 atanh((m-1)/(m+1)), 11 odd terms
__device__ __forceinline__ double log_f(double x)
{
    int hi = __double2hiint(x);
    const int lo = __double2loint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;
    double m = __hiloint2double(hi, lo);
    if (m > 1.4142135623730951) { m *= 0.5; e += 1; }
    const double s = div_f(m - 1.0, m + 1.0);
    const double z = s * s;
    double p = kAtanhC[10];
#pragma unroll
    for (int k = 9; k >= 1; k--) p = fma(p, z, kAtanhC[k]);
    const double fe = (double)e;
    // log x = e ln2_hi + (2 s + (s z p + e ln2_lo))
    return fma(fe, 6.93147180369123816490e-01, fma(2.0, s, fma(s * z, p, fe * 1.90821492927058770002e-10)));
}

}  // namespace chem
