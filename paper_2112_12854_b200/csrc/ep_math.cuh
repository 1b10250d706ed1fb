// ep_math.cuh -- fp64 device math for the cell-model kernels (sm_100a).
//
// The B200 fp64 pipe (64 lanes/SM, one warp instruction per 2 cycles per SM sub-partition) and the issue slots are the
// co-limiting resources of the fused step.  The ncu capture of the first version
// (profiles/r1a_*.md) showed three things this file is built around:
//   * 64-bit literals cost two extra issue slots each (UMOV pairs) unless they come from the constant bank through
//     LDCU.128 into uniform registers  ->  polynomial coefficients live in __constant__ arrays;
//   * 60 inlined exponentials made the kernel 86 KB of SASS, far beyond the 32 KB instruction cache (top stall:
//     no_instruction)  ->  exponentials and logarithms are evaluated in BATCHES: a thread writes its arguments into
//     its own column of a shared-memory slot array and one rolled loop (two arguments per trip for ILP) replaces
//     them by their exponentials; the loop body exists once in the kernel and its constants stay in uniform registers;
//   * IEEE division is ~10 fp64 instructions plus a slow-path call  ->  ep_rcp: MUFU.RCP64H seed + one third-order
//     step (3 DFMA), arguments are finite, normal and far from the ends of the exponent range at every call site.
// Accuracy, measured on the GPU by tests/test_gpu_math.py through ep_math_eval(): exp <= 1 ulp on [-700, 700]
// (polynomial error 2e-17), log <= 1 ulp where |log x| > 1 (the concentrations it is used on) and <= 2.5 ulp near
// x = 1, rcp <= 1 ulp, rsqrt <= 2 ulp, hence a*rcp(b) <= 2 ulp.  No lookup tables (north_star: "precomputed-free exp paths").
#pragma once
#include <cstdint>

namespace epk {

// e^r = 1 + r + r^2 q(r) on |r| <= ln2/2; q = degree-9 Chebyshev interpolant of (e^r - 1 - r)/r^2
// (max relative error of the reconstructed e^r: 1.6e-17, computed in 60-digit arithmetic).
__constant__ double EXP_Q[10] = {0.5000000000000001,     0.16666666666666669,   0.04166666666662396,
                                 0.00833333333333005,    0.0013888888917294928, 0.00019841269863116068,
                                 2.48015211698282e-05,   2.755726836300438e-06, 2.762014840966706e-07,
                                 2.5100431608666542e-08};
// log m = 2 s (1 + z/3 + z^2/5 + ... + z^9/19), s = (m-1)/(m+1), z = s^2 <= 0.0295 (next term z^10/21 < 2.4e-17)
__constant__ double LOG_C[9] = {1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0, 1.0 / 13.0, 1.0 / 15.0,
                                1.0 / 17.0, 1.0 / 19.0};

__device__ __forceinline__ double ep_rcp(double b) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));   // MUFU.RCP64H: >= 20 good bits
    const double e = fma(-b, r, 1.0);
    const double t = fma(e, e, e);                            // e + e^2; remainder e^3 <= 2^-60
    return fma(r, t, r);
}

__device__ __forceinline__ double ep_rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));  // MUFU.RSQ64H
    const double h = x * y;
    const double e = fma(-h, y, 1.0);                         // 1 - x y^2
    const double t = fma(0.375, e, 0.5) * e;                  // e/2 + 3e^2/8
    return fma(y, t, y);
}

// exp of a finite argument with |x| <= 700 (callers clamp); no overflow / underflow / NaN handling
__device__ __forceinline__ double ep_exp_core(double x) {
    const double shift = 6755399441055744.0;                  // 2^52 + 2^51: round-to-nearest-integer trick
    const double t = fma(x, 1.4426950408889634, shift);
    const int k = __double2loint(t);
    const double kd = t - shift;
    double r = fma(kd, -6.93147180369123816490e-01, x);       // ln2 high part (low bits zero: kd*hi is exact)
    r = fma(kd, -1.90821492927058770002e-10, r);              // ln2 low part
    double q = EXP_Q[9];
#pragma unroll
    for (int i = 8; i >= 0; --i) q = fma(q, r, EXP_Q[i]);
    double p = fma(r, q, 1.0);
    p = fma(r, p, 1.0);
    return __hiloint2double(__double2hiint(p) + k * 1048576, __double2loint(p));   // * 2^k via the exponent field
}

// log of a positive normal argument
__device__ __forceinline__ double ep_log_core(double x) {
    int hi = __double2hiint(x);
    const int lo = __double2loint(x);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;
    if (hi > 0x3ff6a09e) { hi -= 0x00100000; e += 1; }        // m in [sqrt(1/2), sqrt(2))
    const double m = __hiloint2double(hi, lo);
    const double s = (m - 1.0) * ep_rcp(m + 1.0);
    const double z = s * s;
    double p = LOG_C[8];
#pragma unroll
    for (int i = 7; i >= 0; --i) p = fma(p, z, LOG_C[i]);
    const double ed = (double)e;
    const double s2 = s + s;
    double res = s2 * (z * p);                                // summed small to large
    res = fma(ed, 1.90821492927058770002e-10, res);
    res += s2;
    return fma(ed, 6.93147180369123816490e-01, res);
}

// W exponentials at once, written stage by stage so that the W dependency chains are interleaved in issue order
// (the fp64 pipe needs several independent chains per warp to stay busy).  Same arithmetic as ep_exp_core.
template <int W>
__device__ __forceinline__ void ep_exp_wide(double (&x)[W]) {
    const double shift = 6755399441055744.0;
    double t[W], r[W], q[W];
    int k[W];
#pragma unroll
    for (int j = 0; j < W; ++j) t[j] = fma(x[j], 1.4426950408889634, shift);
#pragma unroll
    for (int j = 0; j < W; ++j) { k[j] = __double2loint(t[j]); t[j] -= shift; }
#pragma unroll
    for (int j = 0; j < W; ++j) r[j] = fma(t[j], -6.93147180369123816490e-01, x[j]);
#pragma unroll
    for (int j = 0; j < W; ++j) r[j] = fma(t[j], -1.90821492927058770002e-10, r[j]);
#pragma unroll
    for (int j = 0; j < W; ++j) q[j] = fma(EXP_Q[9], r[j], EXP_Q[8]);
#pragma unroll
    for (int i = 7; i >= 0; --i) {
#pragma unroll
        for (int j = 0; j < W; ++j) q[j] = fma(q[j], r[j], EXP_Q[i]);
    }
#pragma unroll
    for (int j = 0; j < W; ++j) q[j] = fma(r[j], q[j], 1.0);
#pragma unroll
    for (int j = 0; j < W; ++j) q[j] = fma(r[j], q[j], 1.0);
#pragma unroll
    for (int j = 0; j < W; ++j) x[j] = __hiloint2double(__double2hiint(q[j]) + k[j] * 1048576, __double2loint(q[j]));
}

// Batched evaluation over a thread's own column of a shared-memory slot array xs[slot][BLOCK]; col = &xs[0][tid].
// N must be a multiple of W.  The loops stay rolled on purpose (instruction-cache footprint).
// n <= N (a multiple of W, the same for every lane of the warp) lets a caller skip trailing slots it does not need.
template <int N, int BLOCK, int W>
__device__ __forceinline__ void ep_exp_slots(double* col, int n = N) {
    static_assert(N % W == 0, "pad the slot list to a multiple of W");
#pragma unroll 1
    for (int s = 0; s < n; s += W) {
        double x[W];
#pragma unroll
        for (int j = 0; j < W; ++j) x[j] = col[(s + j) * BLOCK];
        ep_exp_wide<W>(x);
#pragma unroll
        for (int j = 0; j < W; ++j) col[(s + j) * BLOCK] = x[j];
    }
}

// W logarithms at once, stage by stage (same arithmetic as ep_log_core); arguments positive and normal.
template <int W>
__device__ __forceinline__ void ep_log_wide(double (&x)[W]) {
    double m[W], s[W], z[W], p[W], ed[W];
#pragma unroll
    for (int j = 0; j < W; ++j) {
        int hi = __double2hiint(x[j]);
        const int lo = __double2loint(x[j]);
        int e = (hi >> 20) - 1023;
        hi = (hi & 0x000fffff) | 0x3ff00000;
        if (hi > 0x3ff6a09e) { hi -= 0x00100000; e += 1; }    // m in [sqrt(1/2), sqrt(2))
        m[j] = __hiloint2double(hi, lo);
        ed[j] = (double)e;
    }
#pragma unroll
    for (int j = 0; j < W; ++j) s[j] = ep_rcp(m[j] + 1.0);
#pragma unroll
    for (int j = 0; j < W; ++j) { s[j] *= (m[j] - 1.0); z[j] = s[j] * s[j]; }
#pragma unroll
    for (int j = 0; j < W; ++j) p[j] = fma(LOG_C[8], z[j], LOG_C[7]);
#pragma unroll
    for (int i = 6; i >= 0; --i) {
#pragma unroll
        for (int j = 0; j < W; ++j) p[j] = fma(p[j], z[j], LOG_C[i]);
    }
#pragma unroll
    for (int j = 0; j < W; ++j) {
        const double s2 = s[j] + s[j];
        double res = s2 * (z[j] * p[j]);                      // summed small to large
        res = fma(ed[j], 1.90821492927058770002e-10, res);
        res += s2;
        x[j] = fma(ed[j], 6.93147180369123816490e-01, res);
    }
}

// 8-byte asynchronous global -> shared copy (LDGSTS) into the thread's own slot column: no destination register is
// held while the load is in flight.  ep_cp_async_wait() makes every copy this thread has issued visible to it.
__device__ __forceinline__ void ep_cp_async8(double* smem_dst, const double* gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void ep_cp_async_wait() {
    asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}

__device__ __forceinline__ double ep_clamp(double x, double lo, double hi) { return fmin(fmax(x, lo), hi); }

}  // namespace epk
