// ep_math.cuh -- fp64 device math for the cell-model kernels (sm_100a).
//
// The B200 fp64 pipe (64 lanes/SM) is the co-limiting resource of the fused step, so the
// transcendental and division sequences are written out here with exactly the work the cell model needs:
//   - ep_rcp / ep_div: MUFU.RCP64H seed + two Newton steps, no special-case slow path (arguments are finite, normal
//     and far from the ends of the exponent range in every call site);
//   - ep_exp: Cody-Waite reduction + degree-13 polynomial, argument clamped to [-700, 700] (no overflow, underflow
//     or NaN handling: call sites pass finite arguments);
//   - ep_log: frexp by bit manipulation + atanh series in s = (m-1)/(m+1).
// Accuracy of each is <= 2 ulp over the ranges used (tests/test_gpu_math.py measures it against numpy on the GPU box),
// four orders of magnitude inside the 1e-11 one-step parity tolerance.
#pragma once
#include <cstdint>

namespace epk {

#ifndef EP_LIBM
#define EP_LIBM 0   // 1: route everything through the CUDA math library (debug / A-B comparison builds only)
#endif

__device__ __forceinline__ double ep_rcp(double b) {
#if EP_LIBM
    return 1.0 / b;
#else
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));   // ~20 good bits
    double e = fma(-b, r, 1.0);
    r = fma(r, e, r);                                         // ~40 bits
    e = fma(-b, r, 1.0);
    r = fma(r, e, r);                                         // full
    return r;
#endif
}

__device__ __forceinline__ double ep_div(double a, double b) {
#if EP_LIBM
    return a / b;
#else
    const double r = ep_rcp(b);
    const double q = a * r;
    return fma(fma(-b, q, a), r, q);                          // one residual correction: <= 1 ulp
#endif
}

__device__ __forceinline__ double ep_exp(double x) {
#if EP_LIBM
    return exp(x);
#else
    x = fmin(fmax(x, -700.0), 700.0);
    // k = round(x / ln 2) by the 2^52+2^51 shift trick
    const double shift = 6755399441055744.0;
    const double t = fma(x, 1.4426950408889634, shift);
    const double kd = t - shift;
    const int k = __double2loint(t);
    double r = fma(kd, -6.93147180369123816490e-01, x);       // ln2 high part (low 21 bits zero)
    r = fma(kd, -1.90821492927058770002e-10, r);              // ln2 low part
    // e^r on |r| <= ln2/2: Taylor coefficients 1/n!, degree 13 (remainder r^14/14! < 2^-57 relative)
    double p = 1.60590438368216145994e-10;                    // 1/13!
    p = fma(p, r, 2.08767569878680989792e-09);                // 1/12!
    p = fma(p, r, 2.50521083854417187751e-08);                // 1/11!
    p = fma(p, r, 2.75573192239858906526e-07);                // 1/10!
    p = fma(p, r, 2.75573192239858906526e-06);                // 1/9!
    p = fma(p, r, 2.48015873015873015873e-05);                // 1/8!
    p = fma(p, r, 1.98412698412698412698e-04);                // 1/7!
    p = fma(p, r, 1.38888888888888888889e-03);                // 1/6!
    p = fma(p, r, 8.33333333333333333333e-03);                // 1/5!
    p = fma(p, r, 4.16666666666666666667e-02);                // 1/4!
    p = fma(p, r, 1.66666666666666666667e-01);                // 1/3!
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    // scale by 2^k through the exponent field (|k| <= 1010; result stays normal for |x| <= 700)
    const int hi = __double2hiint(p) + k * 1048576;
    return __hiloint2double(hi, __double2loint(p));
#endif
}

__device__ __forceinline__ double ep_log(double x) {
#if EP_LIBM
    return log(x);
#else
    // x = m * 2^e with m in [sqrt(1/2), sqrt(2)); x is positive and normal at every call site
    int hi = __double2hiint(x);
    const int lo = __double2loint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;
    double m = __hiloint2double(hi, lo);
    if (hi > 0x3ff6a09e) { m *= 0.5; e += 1; }
    const double s = ep_div(m - 1.0, m + 1.0);                // |s| <= 0.1716
    const double z = s * s;
    // log m = 2 s (1 + z/3 + z^2/5 + ... + z^10/21); z^11/23 term < 2^-58 relative
    double p = 1.0 / 21.0;
    p = fma(p, z, 1.0 / 19.0);
    p = fma(p, z, 1.0 / 17.0);
    p = fma(p, z, 1.0 / 15.0);
    p = fma(p, z, 1.0 / 13.0);
    p = fma(p, z, 1.0 / 11.0);
    p = fma(p, z, 1.0 / 9.0);
    p = fma(p, z, 1.0 / 7.0);
    p = fma(p, z, 1.0 / 5.0);
    p = fma(p, z, 1.0 / 3.0);
    const double ed = (double)e;
    // log x = e ln2 + 2s + 2 s z p, summed small to large
    double res = (2.0 * s) * (z * p);
    res = fma(ed, 1.90821492927058770002e-10, res);
    res += 2.0 * s;
    return fma(ed, 6.93147180369123816490e-01, res);
#endif
}

__device__ __forceinline__ double ep_sqrt(double x) { return sqrt(x); }

}  // namespace epk
