// ep_math.cuh -- fp64 device math for the cell-model kernels (sm_100a).
//
// The B200 fp64 pipe (64 lanes/SM, one warp instruction per 2 cycles per SM sub-partition) and the issue slots are the
// co-limiting resources of the fused step.  The ncu capture of the first version
// (profiles/r1a_*.md) showed three things this file is built around:
//   * 64-bit literals cost two extra issue slots each (UMOV pairs) unless they come from the constant bank through
//     LDCU.128 into uniform registers  ->  polynomial coefficients live in __constant__ arrays;
//   * 60 inlined exponentials of ~70 instructions each made the first kernel 86 KB of SASS (top stall: no_instruction).
//     Round 1 answered with rolled loops over arguments parked in shared memory; round 2 found that traffic to be the next
//     limiter and went back to inline evaluation, but of 35 shared exponentials of ~14 fp64 instructions each, FOUR AT A TIME
//     (ep_exp2_wide<4>: four interleaved dependency chains, coefficients in uniform registers), each group placed right
//     before its consumers (ep_tp06.cuh); the kernel is 43 KB of SASS and no_instruction stalls stay below 1 %;
//   * IEEE division is ~10 fp64 instructions plus a slow-path call  ->  ep_rcp: MUFU.RCP64H seed + one third-order
//     step (3 DFMA), arguments are finite, normal and far from the ends of the exponent range at every call site.
//   * every exponential of the cell models has an argument of the form (compile-time constant) x (run-time value), so the
//     factor log2(e) is folded into those constants and the primitive is 2^x: the reduction x = k + r is one exact
//     subtraction instead of the two-constant Cody-Waite pair of a natural exponential (one fp64 instruction less per
//     call, 36 calls per TP06 cell-step).
// Accuracy, measured on the GPU by tests/test_gpu_math.py through ep_math_eval(): 2^x relative error <= 4.2e-16 on [-1000, 1000]
// (<= 3.1 ulp; polynomial error 3e-16), log <= 1 ulp where |log x| > 1 (the concentrations it is used on) and <= 2.5 ulp near
// x = 1, rcp <= 1 ulp, rsqrt <= 2 ulp, hence a*rcp(b) <= 2 ulp.  No lookup tables (north_star: "precomputed-free exp paths").
#pragma once
#include <cstdint>

namespace epk {

// 2^r = 1 + r P(r) on |r| <= 1/2.  P = the degree-9 MINIMAX polynomial for the relative error of the reconstructed 2^r
// (Remez exchange with weight r / 2^r, 60-digit arithmetic): 2.96e-16; measured on the GPU, with the rounding of the Horner
// chain: relative error <= 4.2e-16, i.e. <= 3.1 ulp just below a power of two and <= 1.9 ulp just above one
// (tests/test_gpu_math.py).  EP_EXP2_DEG = 10 selects the degree-10 Chebyshev interpolant (8.4e-18: <= 1 ulp, one DFMA more per
// call); round 1 shipped that one, round 2 measured the difference on the fused kernel (175.7 vs 177.8 us on config 3)
// against a one-step tolerance of 1e-11 and a run tolerance of 1e-6 mV that both keep three orders of margin.
#ifndef EP_EXP2_DEG
#define EP_EXP2_DEG 9
#endif
constexpr double L2E = 1.4426950408889634;   // log2(e): folded into the compile-time slopes of every exponent
#if EP_EXP2_DEG == 10
__constant__ double EXP2_P[11] = {0.6931471805599453,     0.24022650695910097,   0.0555041086648216,
                                  0.009618129107606888,   0.0013333558146416936, 0.0001540353044173605,
                                  1.525273382983612e-05,  1.321544258792169e-06, 1.0178062445845774e-07,
                                  7.072585949269223e-09,  4.4549605981865186e-10};
#else
__constant__ double EXP2_P[10] = {0.6931471805599516,     0.24022650695910472,   0.05550410866434658,
                                  0.009618129107380715,   0.001333355824648072,  0.00015403530800818256,
                                  1.525264774769592e-05,  1.321523563477604e-06, 1.0210506458816145e-07,
                                  7.111758687557852e-09};
#endif
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

// 2^x of a finite argument with |x| <= 1000 (callers clamp); no overflow / underflow / NaN handling
__device__ __forceinline__ double ep_exp2_core(double x) {
    const double shift = 6755399441055744.0;                  // 2^52 + 2^51: round-to-nearest-integer trick
    const double t = x + shift;
    const int k = __double2loint(t);
    const double r = x - (t - shift);                         // exact: |r| <= 1/2
    double q = EXP2_P[EP_EXP2_DEG];
#pragma unroll
    for (int i = EP_EXP2_DEG - 1; i >= 0; --i) q = fma(q, r, EXP2_P[i]);
    const double p = fma(r, q, 1.0);
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

// W powers of two at once, written stage by stage so that the W dependency chains are interleaved in issue order
// (the fp64 pipe needs several independent chains per warp to stay busy).  Same arithmetic as ep_exp2_core.
template <int W>
__device__ __forceinline__ void ep_exp2_wide(double (&x)[W]) {
    const double shift = 6755399441055744.0;
    double t[W], r[W], q[W];
    int k[W];
#pragma unroll
    for (int j = 0; j < W; ++j) t[j] = x[j] + shift;
#pragma unroll
    for (int j = 0; j < W; ++j) { k[j] = __double2loint(t[j]); t[j] -= shift; }
#pragma unroll
    for (int j = 0; j < W; ++j) r[j] = x[j] - t[j];
#pragma unroll
    for (int j = 0; j < W; ++j) q[j] = fma(EXP2_P[EP_EXP2_DEG], r[j], EXP2_P[EP_EXP2_DEG - 1]);
#pragma unroll
    for (int i = EP_EXP2_DEG - 2; i >= 0; --i) {
#pragma unroll
        for (int j = 0; j < W; ++j) q[j] = fma(q[j], r[j], EXP2_P[i]);
    }
#pragma unroll
    for (int j = 0; j < W; ++j) q[j] = fma(r[j], q[j], 1.0);
#pragma unroll
    for (int j = 0; j < W; ++j) x[j] = __hiloint2double(__double2hiint(q[j]) + k[j] * 1048576, __double2loint(q[j]));
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

// Streaming loads: data that is read once per step (stencil tables, state rows, the node table) does not allocate in L1,
// which then keeps the gather targets (node values, neighbour potentials) that neighbouring cells share.  Streaming stores
// (st.global.cs: evict-first) for the state rows, which nothing reads before the next step, so that L2 keeps the new Vm for
// the node kernel that follows (node kernel 33.7 -> 31.3 us on config 3).  ld.global.cs instead of no_allocate: no difference.
#ifndef EP_STREAM_LOADS
#define EP_STREAM_LOADS 1
#endif
#ifndef EP_STREAM_STORES
#define EP_STREAM_STORES 1
#endif
__device__ __forceinline__ double ep_ldg_stream(const double* q) {   // read-only for the lifetime of the kernel
#if EP_STREAM_LOADS
    double v;
    asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(q));
    return v;
#else
    return __ldg(q);
#endif
}
__device__ __forceinline__ int32_t ep_ldg_stream(const int32_t* q) {
#if EP_STREAM_LOADS
    int32_t v;
    asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(q));
    return v;
#else
    return __ldg(q);
#endif
}
__device__ __forceinline__ double ep_ld_stream(const double* q) {    // state rows: read here, overwritten later by the same thread
#if EP_STREAM_LOADS
    double v;
    asm volatile("ld.global.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(q) : "memory");
    return v;
#else
    return *q;
#endif
}

__device__ __forceinline__ void ep_st_stream(double* q, double v) {   // state rows: not read again before the next step
#if EP_STREAM_STORES
    asm volatile("st.global.cs.f64 [%0], %1;" ::"l"(q), "d"(v) : "memory");
#else
    *q = v;
#endif
}

__device__ __forceinline__ double ep_clamp(double x, double lo, double hi) { return fmin(fmax(x, lo), hi); }

}  // namespace epk
