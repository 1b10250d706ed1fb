// ep_tp06.cuh -- ten Tusscher-Panfilov 2006 ventricular cell model, one explicit step of one cell (device code).
//
// PAPER.md:126, :174, :256 name the model (ref [3]: 19 states, 13 of them advanced by Rush-Larsen);
// the equations and constants are restated from the published model in DESIGN.md Appendix A.  Readings B1..B9 of
// DESIGN.md section 3 apply (13 RL variables = 12 gates + Rbar; buffer factors + forward Euler for the three calcium
// pools; v >= -40 mV takes the high-voltage h/j branch; removable singularity of I_CaL handled by a series).
// Everything on the right-hand side is taken at t^n.
//
// This is the production form.  It computes the same functions as Appendix A, rearranged for the fp64 pipe
// (DESIGN.md section 7): exponentials with commensurate slopes are integer powers of one exponential
// (v/600 -> slopes 1/200, 1/24, 1/20, 1/15, 1/10, 1/7.5, 1/6, 1/5; v/14 -> 1/14, 1/7; vF/20RT -> 0.1, 0.65, 0.9, 1 vF/RT;
// 0.02(v-E_K) -> 0.06, 0.1, 0.5; (v+27)^2/3600 -> /240, /225), every sigmoid product is written as one rational function
// with a single reciprocal, and the remaining 35 exponentials are evaluated four at a time (interleaved dependency chains,
// ep_math.cuh) in nine groups, each right before the quantities that consume it, so that arguments and results stay in
// registers; shared memory only parks the gate values at t^n and the stencil coefficients.  Relative differences from the literal formulas are <= ~5e-14 (120-fold powers of a value good to 4.2e-16),
// three orders of magnitude inside the 1e-11 one-step tolerance.  (The literal transcription was the first kernel of
// this repo -- profiles/r01a_baseline_direct_kernel.md -- and lives on only in the CPU oracle.)
//
// Units: mV, ms, mM, currents uA/uF, conductances nS/pF.
#pragma once
#include "ep_math.cuh"

// A 64-bit literal costs two issue slots (UMOV pair) each time it is used; a double non-type template argument (C++20)
// instantiates one __constant__ word per distinct value, which ptxas reads with LDC.64 / LDCU.128 instead.
// Values whose low 32 mantissa bits are zero (1.0, 0.25, 1400.0 ...) stay literals: they are free DFMA immediates.
template <double V>
__device__ __constant__ double EPK_CONST = V;
#define CK(x) (::EPK_CONST<(x)>)

namespace epk {

enum { TP06_S = 19 };
// state order at the ABI (ep_read_state var): v m h j xr1 xr2 xs r s d f f2 fCass Rbar Ca_i Ca_SR Ca_SS Na_i K_i
enum { Y_V = 0, Y_M, Y_H, Y_J, Y_XR1, Y_XR2, Y_XS, Y_R, Y_S, Y_D, Y_F, Y_F2, Y_FCASS, Y_RBAR, Y_CAI, Y_CASR, Y_CASS,
       Y_NAI, Y_KI };

__device__ __constant__ const double TP06_REST_STATE[TP06_S] = {
    -86.2, 0.0, 0.75, 0.75, 0.0, 1.0, 0.0, 0.0, 1.0, 0.0, 1.0, 1.0, 1.0, 1.0, 7e-5, 1.3, 7e-5, 7.67, 138.3};

namespace tp06 {
constexpr double R = 8314.472, T = 310.0, F = 96485.3415;
constexpr double RTF = R * T / F;          // mV
constexpr double FRT = F / (R * T);        // 1/mV
constexpr double Ko = 5.4, Cao = 2.0, Nao = 140.0;
constexpr double Vc = 0.016404, Vsr = 0.001094, Vss = 0.00005468, Cap = 0.185;
constexpr double GNa = 14.838, GK1 = 5.405, GKr = 0.153, GCaL = 3.980e-5, GbNa = 2.9e-4, GbCa = 5.92e-4;
constexpr double GpCa = 0.1238, KpCa = 5e-4, GpK = 0.0146, pKNa = 0.03;
constexpr double PNaK = 2.724, KmK = 1.0, KmNa = 40.0;
constexpr double kNaCa = 1000.0, KmNai = 87.5, KmCa = 1.38, ksat = 0.1, alpha = 2.5;   // gamma = 0.35 = 7/20
constexpr double Vmaxup = 0.006375, Kup = 2.5e-4, Vrel = 0.102, k1p = 0.15, k2p = 0.045, k3 = 0.060, k4 = 0.005;
constexpr double EC = 1.5, maxsr = 2.5, minsr = 1.0, Vleak = 3.6e-4, Vxfer = 0.0038;
constexpr double Bufc = 0.2, Kbufc = 0.001, Bufsr = 10.0, Kbufsr = 0.3, Bufss = 0.4, Kbufss = 2.5e-4;
// natural logarithms of the extracellular concentrations
constexpr double LN_KO = 1.6863989535702288, LN_NAO = 4.941642422609304, LN_KO_PNAO = 2.2617630984737906,
                 LN_CAO = 0.6931471805599453;
// e^c constants produced when (v + a)/b exponents are split into e^(v/b) e^(a/b)
constexpr double EM12 = 6.14421235332821e-06;     // e^(-12)
constexpr double E7C = 1096.6331584284585;        // e^(7)
constexpr double EM025 = 0.7788007830714049;      // e^(-0.25)
constexpr double EM32 = 0.04076220397836622;      // e^(-3.2)
constexpr double EM45 = 0.011108996538242306;     // e^(-4.5)
constexpr double EM26_7 = 0.0243728440732796;     // e^(-26/7)
constexpr double E88_24 = 39.12128399815322;      // e^(88/24)
constexpr double EM3 = 0.049787068367863944;      // e^(-3)
constexpr double EM5_14 = 0.6996725373751304;     // e^(-5/14)
constexpr double E5_6 = 2.300975890892825;        // e^(5/6)
constexpr double EM35_15 = 0.09697196786440507;   // e^(-35/15)
constexpr double E20_6 = 28.031624894526136;      // e^(20/6)
constexpr double E56 = 270.42640742615265;        // e^(5.6)
constexpr double E4 = 54.598150033144236;         // e^(4)
constexpr double EM4 = 0.01831563888873418;       // e^(-4)
constexpr double EM8_75 = 0.34415378686541237;    // e^(-8/7.5)
constexpr double E1 = 2.718281828459045;          // e
constexpr double E25 = 12.182493960703473;        // e^(2.5)
constexpr double E20_7 = 17.41170806332765;       // e^(20/7)
constexpr double E13 = 3.669296667619244;         // e^(1.3)
constexpr double E3 = 20.085536923187668;         // e^(3)
constexpr double E5C = 148.4131591025766;         // e^(5)
constexpr double EM1 = 0.36787944117144233;       // e^(-1)

// shared-memory slots (one column of BLOCK doubles per thread): the gate values at t^n, parked by asynchronous copies
constexpr int EXP_W = 4;     // exponentials evaluated side by side (four interleaved dependency chains)
constexpr int N_RLB = 11;    // Rush-Larsen variables with voltage-driven rates: m h j xr1 xr2 xs r s d f f2 (fCass and Rbar: rates need no exp)
constexpr int G_OLD0 = 0;    // 11 gate values at t^n, parked from the first load to the Rush-Larsen update, slots 0..10
constexpr int G_RBAR = 11;   // Rbar at t^n
constexpr int N_SLOTS = 12;
static_assert(G_OLD0 + N_RLB <= G_RBAR && G_RBAR < N_SLOTS, "slot layout");
}  // namespace tp06

// One step of one cell, everything on the right-hand side at t^n.  v = Vm^n of this cell, ycol = &y[0][cell] (state
// row k at ycol[k*stride]; rows 1..18 are read and overwritten), type: 0 endo, 1 mid, 2 epi, stimulus() returns
// I_s/C_m [uA/uF] of this cell and step.
// The diffusion term D_c/(chi C_m) [mV/ms] comes from two callables so that its gathers are in flight while the
// logarithms and the first exponential batch run: issue_gather() starts the loads, finish_gather() returns the sum.
// col = this thread's column of the block's slot array (stride BLOCK doubles, tp06::N_SLOTS slots).  Returns Vm^{n+1}.
//
// ORDER == 2 (reading H1): second-order Adams-Bashforth for v and the five concentrations, and the
// gates relax towards y_inf(*) with tau(*), (*) = arguments extrapolated to t^{n+1/2} (v* = 3/2 v^n - 1/2 v^{n-1}, likewise
// Ca_SS*, Ca_SR* for fCass and Rbar); the stimulus is piecewise constant on steps and is integrated exactly, outside the
// extrapolation.  hist.have == 0 (first step after an initialisation): the first-order step, history recorded.
struct O2Hist {
    double* hcol = nullptr;   // this cell's column of the history rows: 0..5 f^{n-1} of v Ca_i Ca_SR Ca_SS Na_i K_i, 6 Ca_SS^{n-1}, 7 Ca_SR^{n-1}
    int64_t stride = 0;
    double v_prev = 0.0;      // v^{n-1}
    int have = 0;
};
template <int ORDER, int BLOCK, class Stim, class Issue, class Finish>
__device__ __forceinline__ double tp06_step(double v, double* ycol, int64_t stride, int type, double dt, Stim stimulus,
                                            Issue issue_gather, Finish finish_gather, double* col, O2Hist hist = O2Hist()) {
    using namespace tp06;
    // Argument of every transcendental (reading T2).  TP06 lives in [-100, +60] mV; for |v| <= 200 mV every
    // exponent stays below 90 in magnitude, so the clamp is inert there and the kernel follows the (unclamped) oracle;
    // beyond it the exponentials are frozen at their +-200 mV values while the ohmic factors (v - E) keep the true v.
    // Inside that range four Rush-Larsen rates can exceed 700/dt (m: 8e12, h: 3e6, j: 5e4, xr1: 2e5 per ms at -200 mV):
    // their base-2 exponents are clamped to -1000 below (2^-1000 = 1e-301 stands for the oracle's underflow to 0).
    const double vg = ep_clamp(v, -200.0, 200.0);
    const double dtl = dt * L2E;   // Rush-Larsen exponents -dt/tau in base-2 units (the exponential primitive is 2^x)
    const double Cai = ep_ld_stream(ycol + Y_CAI * stride), CaSR = ep_ld_stream(ycol + Y_CASR * stride),
                 CaSS = ep_ld_stream(ycol + Y_CASS * stride), Nai = ep_ld_stream(ycol + Y_NAI * stride),
                 Ki = ep_ld_stream(ycol + Y_KI * stride);
    // arguments of the gate functions: the values at t^n (first order) or extrapolated to t^{n+1/2} (second order)
    double vs = v, vgs = vg, CaSSs = CaSS, CaSRs = CaSR;
    double fprev[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if constexpr (ORDER == 2) {
#pragma unroll
        for (int k = 0; k < 6; ++k) fprev[k] = hist.hcol[k * hist.stride];
        if (hist.have) {
            vs = fma(1.5, v, -0.5 * hist.v_prev);
            CaSSs = fma(1.5, CaSS, -0.5 * hist.hcol[6 * hist.stride]);
            CaSRs = fma(1.5, CaSR, -0.5 * hist.hcol[7 * hist.stride]);
            vgs = ep_clamp(vs, -200.0, 200.0);
        }
    }
    // The 11 voltage-driven gates and Rbar are copied into shared memory asynchronously (no registers held, nothing waits
    // for them here); they are first touched after the first exponential batch, which hides their latency.
#pragma unroll
    for (int k = 0; k < N_RLB; ++k) ep_cp_async8(col + (G_OLD0 + k) * BLOCK, ycol + (1 + k) * stride);
    ep_cp_async8(col + G_RBAR * BLOCK, ycol + Y_RBAR * stride);
    const double fCass = ep_ld_stream(ycol + Y_FCASS * stride);

    // ---- batch 1: the four logarithms of the reversal potentials, side by side in registers
    double lg[4] = {Ki, Nai, fma(CK(pKNa), Nai, Ki), Cai};
    ep_log_wide<4>(lg);
    issue_gather();   // the stencil indices were requested before the concentrations: they are here by now
    const double EK = CK(RTF) * (CK(LN_KO) - lg[0]);
    const double ENa = CK(RTF) * (CK(LN_NAO) - lg[1]);
    const double EKs = CK(RTF) * (CK(LN_KO_PNAO) - lg[2]);
    const double ECa = CK(0.5 * RTF) * (CK(LN_CAO) - lg[3]);
    const double u = v - EK;
    const double ug = ep_clamp(u, -150.0, 300.0);
    const bool hi = (vs >= -40.0);   // reading B7 (on the gates' own argument)

    double h_exp;   // e^{(v+71.55)/7.43}: evaluated with group 2, used for h_inf = j_inf with the last group
    // ---- streaming form: the exponentials are evaluated in nine groups of EXP_W, each group right before the quantities that
    // consume it, so that their arguments AND results stay in registers; the slot array only parks the gate values at t^n and
    // the stencil coefficients (profiles/r02_cell_kernel.md: shared-memory traffic, not the fp64 pipe, was what the batch form
    // of this kernel ran into).
    // fCass and Rbar: their Rush-Larsen rates need no exponential, so exp(-dt/tau) rides in this batch
    const double c2 = CaSR * CaSR, css2 = CaSS * CaSS, ci2 = Cai * Cai;
    const double kcasr = fma(-(maxsr - minsr) * c2, ep_rcp(c2 + EC * EC), maxsr);
    double kcasr_s = kcasr, css2_s = css2;      // the same at the gates' arguments (second order: Ca_SR*, Ca_SS*)
    if constexpr (ORDER == 2) {
        const double c2s = CaSRs * CaSRs;
        kcasr_s = fma(-(maxsr - minsr) * c2s, ep_rcp(c2s + EC * EC), maxsr);
        css2_s = CaSSs * CaSSs;
    }
    const double qf = ep_rcp(fma(400.0, css2_s, 1.0));              // 1/(1 + (CaSS/0.05)^2)
    const double fCass_inf = fma(CK(0.6), qf, CK(0.4));
    const double Rbar_rate = fma(CK(k2p) * kcasr_s, CaSSs, CK(k4));   // dR/dt = k4 (1 - R) - k2 CaSS R (reading B1)
    const double Rbar_inf = CK(k4) * ep_rcp(Rbar_rate);
    // group 0: the two shared gate exponentials and the two current exponentials that are raised to powers
    double x0[EXP_W] = {vgs * CK(L2E / 600.0), vgs * CK(L2E / 14.0), vg * CK(0.05 * FRT * L2E),
                        fma(vg, CK(2.0 * FRT * L2E), CK(-30.0 * FRT * L2E))};
    const double xcal = (vg - 15.0) * CK(2.0 * FRT);
    ep_exp2_wide<EXP_W>(x0);
    // group 1: I_pK, the two I_K1 exponentials, the Gaussian of tau_f / tau_f2
    double x1[EXP_W] = {fma(vg, CK(-L2E / 5.98), CK(25.0 * L2E / 5.98)), fma(ug, CK(0.0002 * L2E), CK(0.02 * L2E)),
                        ug * CK(0.02 * L2E), (vgs + 27.0) * (vgs + 27.0) * CK(-L2E / 3600.0)};
    ep_exp2_wide<EXP_W>(x1);
    const double dv_diff = finish_gather();   // the gathers have landed by now: 12 values -> 1
    const double istim = stimulus();          // late on purpose: its first instruction waits for the cell's stimulus mask
    ep_cp_async_wait();                       // the parked gate values have landed too
    double gNa, gCaL, gto, gKr, gKs;
    const double Rbar = col[G_RBAR * BLOCK];
    {
        double g[N_RLB];
#pragma unroll
        for (int k = 0; k < N_RLB; ++k) g[k] = col[(G_OLD0 + k) * BLOCK];
        gNa = (g[Y_M - 1] * g[Y_M - 1] * g[Y_M - 1]) * g[Y_H - 1] * g[Y_J - 1];
        gCaL = (g[Y_D - 1] * g[Y_F - 1]) * (g[Y_F2 - 1] * fCass);
        gto = g[Y_R - 1] * g[Y_S - 1];
        gKr = g[Y_XR1 - 1] * g[Y_XR2 - 1];
        gKs = g[Y_XS - 1] * g[Y_XS - 1];
    }
    // ---- integer powers
    double E200, E24, E20, E15, E10, E7p5, E6, E5;
    {
        const double B = x0[0];
        const double B2 = B * B, B3 = B2 * B, B5 = B2 * B3, B10 = B5 * B5, B20 = B10 * B10, B40 = B20 * B20;
        const double B30 = B20 * B10, B60 = B30 * B30;
        E200 = B3; E24 = B20 * B5; E20 = B30; E15 = B40; E10 = B60; E7p5 = B40 * B40; E6 = B60 * B40; E5 = B60 * B60;
    }
    const double E14 = x0[1], E7 = E14 * E14;
    double W13, W18, W20;
    {
        const double W = x0[2];
        const double W2 = W * W, W4 = W2 * W2, W8 = W4 * W4, W16 = W8 * W8;
        W13 = W8 * W4 * W; W18 = W16 * W2; W20 = W18 * W2;
    }
    double Gf, Gf2;   // exp(-(v+27)^2/225), exp(-(v+27)^2/240)
    {
        const double b = x1[3];
        const double b2 = b * b, b4 = b2 * b2, b8 = b4 * b4;
        Gf = b8 * b8; Gf2 = (b8 * b4) * (b2 * b);
    }

    // ---- membrane currents
    const double INa = CK(GNa) * gNa * (v - ENa);
    double ICaL;
    {
        const double ex = x0[3];
        // x/(e^x - 1), with the series 1 - x/2 inside |x| < 1e-7 (reading B6)
        const double xo = (fabs(xcal) < 1e-7) ? fma(-0.5, xcal, 1.0) : xcal * ep_rcp(ex - 1.0);
        ICaL = CK(GCaL * 2.0 * F) * gCaL * xo * fma(0.25 * CaSS, ex, -Cao);
    }
    const double Gto = (type == 0) ? CK(0.073) : CK(0.294);
    const double GKs = (type == 1) ? CK(0.098) : CK(0.392);
    const double Ito = Gto * gto * u;
    const double IKr = CK(GKr) * gKr * u;     // sqrt(Ko/5.4) = 1
    const double IKs = GKs * gKs * (v - EKs);
    double IK1;
    {
        const double q = x1[1], Q = x1[2];
        const double Q2 = Q * Q, Q3 = Q2 * Q, Q5 = Q2 * Q3, Q10 = Q5 * Q5, Q25 = Q10 * Q10 * Q5;
        const double t1 = fma(CK(0.1), Q25, CK(0.1));                                       // 0.1 (1 + e^{-0.5u}) Q^25
        const double t2 = fma(CK(EM1), Q5, 3.0 * q) * fma(CK(EM12), Q3, 1.0) * Q25;         // (3q + e^{0.1(u-10)})(1 + e^{0.06(u-200)}) Q^25
        IK1 = CK(GK1) * u * t1 * ep_rcp(t1 + t2);
    }
    const double Nai3 = Nai * Nai * Nai;
    const double INaCa = CK(kNaCa / ((KmNai * KmNai * KmNai + Nao * Nao * Nao) * (KmCa + Cao)))
                         * fma(W20, Nai3 * Cao, CK(-(Nao * Nao * Nao * alpha)) * Cai) * ep_rcp(W13 + CK(ksat));
    const double INaK = CK(PNaK * Ko / (Ko + KmK)) * Nai * W20
                        * ep_rcp((Nai + KmNa) * fma(CK(0.1245), W18, W20 + CK(0.0353)));
    const double IpCa = CK(GpCa) * Cai * ep_rcp(CK(KpCa) + Cai);
    const double IpK = CK(GpK) * u * ep_rcp(1.0 + x1[0]);
    const double IbNa = CK(GbNa) * (v - ENa);
    const double IbCa = CK(GbCa) * (v - ECa);
    const double iion = INa + ICaL + Ito + IKr + IKs + IK1 + INaCa + INaK + IpCa + IpK + IbNa + IbCa;

    // ---- sarcoplasmic-reticulum fluxes, buffer factors (reading B3), concentration derivatives
    const double O = CK(k1p) * css2 * Rbar * ep_rcp(fma(CK(k3), kcasr, CK(k1p) * css2));
    const double Irel = CK(Vrel) * O * (CaSR - CaSS);
    const double Ileak = CK(Vleak) * (CaSR - Cai);
    const double Iup = CK(Vmaxup) * ci2 * ep_rcp(ci2 + CK(Kup * Kup));
    const double Ixfer = CK(Vxfer) * (CaSS - Cai);
    const double ti = (Cai + CK(Kbufc)) * (Cai + CK(Kbufc)), tsr = (CaSR + CK(Kbufsr)) * (CaSR + CK(Kbufsr)),
                 tss = (CaSS + CK(Kbufss)) * (CaSS + CK(Kbufss));
    const double bi = ti * ep_rcp(ti + CK(Bufc * Kbufc));
    const double bsr = tsr * ep_rcp(tsr + Bufsr * Kbufsr);
    const double bss = tss * ep_rcp(tss + CK(Bufss * Kbufss));
    const double dCai = bi * ((Ileak - Iup) * CK(Vsr / Vc) + Ixfer - (IbCa + IpCa - 2.0 * INaCa) * CK(Cap / (2.0 * Vc * F)));
    const double dCaSR = bsr * (Iup - Ileak - Irel);
    const double dCaSS = bss * (-ICaL * CK(Cap / (2.0 * Vss * F)) + Irel * CK(Vsr / Vss) - Ixfer * CK(Vc / Vss));
    const double dNai = -(INa + IbNa + 3.0 * INaK + 3.0 * INaCa) * CK(Cap / (Vc * F));
    double v_new;
    if constexpr (ORDER == 1) {
        const double dKi = -(IK1 + Ito + IKr + IKs - 2.0 * INaK + IpK + istim) * CK(Cap / (Vc * F));   // reading B8
        v_new = fma(dt, dv_diff - iion - istim, v);            // eq. (7); explicit increment :172
        ep_st_stream(ycol + Y_CAI * stride, fma(dt, dCai, Cai));             // forward Euler
        ep_st_stream(ycol + Y_CASR * stride, fma(dt, dCaSR, CaSR));
        ep_st_stream(ycol + Y_CASS * stride, fma(dt, dCaSS, CaSS));
        ep_st_stream(ycol + Y_NAI * stride, fma(dt, dNai, Nai));
        ep_st_stream(ycol + Y_KI * stride, fma(dt, dKi, Ki));
    } else {
        // right-hand sides without the stimulus; AB2 where there is a history, the stimulus added as its exact integral
        const double f[6] = {dv_diff - iion, dCai, dCaSR, dCaSS, dNai,
                             -(IK1 + Ito + IKr + IKs - 2.0 * INaK + IpK) * CK(Cap / (Vc * F))};
        double w[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            w[k] = hist.have ? fma(1.5, f[k], -0.5 * fprev[k]) : f[k];
            hist.hcol[k * hist.stride] = f[k];
        }
        hist.hcol[6 * hist.stride] = CaSS;
        hist.hcol[7 * hist.stride] = CaSR;
        v_new = fma(dt, w[0] - istim, v);
        ep_st_stream(ycol + Y_CAI * stride, fma(dt, w[1], Cai));
        ep_st_stream(ycol + Y_CASR * stride, fma(dt, w[2], CaSR));
        ep_st_stream(ycol + Y_CASS * stride, fma(dt, w[3], CaSS));
        ep_st_stream(ycol + Y_NAI * stride, fma(dt, w[4], Nai));
        ep_st_stream(ycol + Y_KI * stride, fma(dt, w[5] - istim * CK(Cap / (Vc * F)), Ki));      // reading B8
    }

    // one Rush-Larsen group: y <- inf + (y_old - inf) 2^e for four gates (gate index g = state row - 1; g < 0: pad)
    auto rush_larsen4 = [&](double (&e)[EXP_W], const double (&in)[EXP_W], int g0, int g1, int g2, int g3) {
        const int gi[EXP_W] = {g0, g1, g2, g3};
        double yo[EXP_W];
#pragma unroll
        for (int j = 0; j < EXP_W; ++j) yo[j] = col[(G_OLD0 + (gi[j] < 0 ? 0 : gi[j])) * BLOCK];
        ep_exp2_wide<EXP_W>(e);
#pragma unroll
        for (int j = 0; j < EXP_W; ++j)
            if (gi[j] >= 0) ep_st_stream(ycol + (1 + gi[j]) * stride, fma(yo[j] - in[j], e[j], in[j]));
    };
    // ---- group 2: m, h_inf, xr1, d; gates m, xr1, xr2, d
    {
        double x2[EXP_W] = {fma(vgs, CK(-L2E / 9.03), CK(-56.86 * L2E / 9.03)), fma(vgs, CK(L2E / 7.43), CK(71.55 * L2E / 7.43)),
                            fma(vgs, CK(L2E / 11.5), CK(30.0 * L2E / 11.5)), fma(vgs, CK(-L2E / 13.0), CK(-35.0 * L2E / 13.0))};
        ep_exp2_wide<EXP_W>(x2);
        double in[EXP_W], e[EXP_W];
        {   // m: tau = s(-60-v;5) [0.1 s(v+35;5) + 0.1 s(v-50;200)],  s(z) = 1/(1+e^z)
            const double sm = ep_rcp(1.0 + x2[0]);
            in[0] = sm * sm;
            const double P = fma(CK(E7C), E5, 1.0), Q = fma(CK(EM025), E200, 1.0);
            e[0] = fmax(-dtl * ((E5 + CK(EM12)) * P * Q * ep_rcp(CK(0.1) * E5 * (P + Q))), -1000.0);
        }
        in[1] = E7 * ep_rcp(E7 + CK(EM26_7));                                                          // xr1
        e[1] = fmax(-dtl * ((E10 + CK(EM45)) * (1.0 + x2[2]) * ep_rcp(2700.0 * E10)), -1000.0);
        in[2] = ep_rcp(fma(CK(E88_24), E24, 1.0));                                                     // xr2
        e[2] = -dtl * ((E20 + CK(EM3)) * fma(CK(EM3), E20, 1.0) * ep_rcp(CK(3.36) * E20));
        {   // d
            in[3] = E7p5 * ep_rcp(E7p5 + CK(EM8_75));
            const double D = 1.0 + x2[3], P5 = fma(CK(E1), E5, 1.0), Q20 = E20 + CK(E25);
            e[3] = -dtl * (D * P5 * Q20 * ep_rcp(fma(fma(0.25, D, CK(1.4)) * CK(1.4), Q20, E20 * D * P5)));
        }
        h_exp = x2[1];
        rush_larsen4(e, in, Y_M - 1, Y_XR1 - 1, Y_XR2 - 1, Y_D - 1);
    }
    // ---- group 3: the Gaussians of tau_r and tau_s, exp(-dt/tau) of fCass and Rbar; gates xs, r, s, f
    {
        double x3[EXP_W] = {(vgs + 40.0) * (vgs + 40.0) * CK(-L2E / 1800.0),
                            (type == 0) ? (vgs + 67.0) * (vgs + 67.0) * CK(-L2E / 1000.0)
                                        : (vgs + 45.0) * (vgs + 45.0) * CK(-L2E / 320.0),
                            -dtl * ep_rcp(fma(80.0, qf, 2.0)),              // tau_fCass >= 2 ms
                            fmax(-dtl * Rbar_rate, -1000.0)};               // rate grows with Ca_SS: keep the clamp
        ep_exp2_wide<EXP_W>(x3);
        ep_st_stream(ycol + Y_FCASS * stride, fma(fCass - fCass_inf, x3[2], fCass_inf));   // Rush-Larsen
        ep_st_stream(ycol + Y_RBAR * stride, fma(Rbar - Rbar_inf, x3[3], Rbar_inf));
        double in[EXP_W], e[EXP_W];
        {   // xs
            in[0] = E14 * ep_rcp(E14 + CK(EM5_14));
            const double t = ep_rsqrt((E6 + CK(E5_6)) * E6) * E6;          // 1/sqrt(1 + e^{(5-v)/6})
            const double P15 = fma(CK(EM35_15), E15, 1.0);
            e[0] = -dtl * (P15 * ep_rcp(fma(1400.0, t, 80.0 * P15)));
        }
        in[1] = E6 * ep_rcp(E6 + CK(E20_6));                                // r
        e[1] = -dtl * ep_rcp(fma(9.5, x3[0], CK(0.8)));
        if (type == 0) {                                                    // s (reading B5: endo has its own curves)
            in[2] = ep_rcp(fma(CK(E56), E5, 1.0));
            e[2] = -dtl * ep_rcp(fma(1000.0, x3[1], 8.0));
        } else {
            in[2] = ep_rcp(fma(CK(E4), E5, 1.0));
            const double P = fma(CK(EM4), E5, 1.0);
            e[2] = -dtl * (P * ep_rcp(fma(fma(85.0, x3[1], 3.0), P, 5.0)));
        }
        {   // f
            const double Qa = E10 + CK(E13), Qb = fma(CK(E3), E10, 1.0);
            in[3] = ep_rcp(fma(CK(E20_7), E7, 1.0));
            e[3] = -dtl * (Qa * Qb * ep_rcp(fma(fma(1102.5, Gf, 20.0), Qa * Qb, fma(200.0 * E10, Qb, 180.0 * Qa))));
        }
        rush_larsen4(e, in, Y_XS - 1, Y_R - 1, Y_S - 1, Y_F - 1);
    }
    // ---- groups 4, 5: the h / j rate exponentials (the four that only the low-voltage branch needs are skipped when every
    // cell of the warp is above -40 mV: warp-uniform); gates h, j, f2
    {
        double x4[EXP_W], x5[EXP_W] = {1.0, 1.0, 1.0, 1.0};
        const bool all_hi = __all_sync(__activemask(), hi);
        if (hi) {
            x4[0] = fma(vgs, CK(-L2E / 11.1), CK(-10.66 * L2E / 11.1));
            x4[1] = vgs * CK(0.057 * L2E);
            x4[2] = 0.0; x4[3] = 0.0;
        } else {
            x4[0] = fma(vgs, CK(-L2E / 6.8), CK(-80.0 * L2E / 6.8));
            x4[1] = vgs * CK(0.079 * L2E);
            x4[2] = vgs * CK(0.3485 * L2E);
            x4[3] = vgs * CK(0.2444 * L2E);
        }
        ep_exp2_wide<EXP_W>(x4);
        if (!all_hi) {
            x5[0] = vgs * CK(-0.04391 * L2E);
            x5[1] = fma(vgs, CK(0.311 * L2E), CK(0.311 * 79.23 * L2E));
            x5[2] = vgs * CK(-0.01052 * L2E);
            x5[3] = fma(vgs, CK(-0.1378 * L2E), CK(-0.1378 * 40.14 * L2E));
            ep_exp2_wide<EXP_W>(x5);
        }
        double in[EXP_W], e[EXP_W];
        const double sh = ep_rcp(1.0 + h_exp);
        in[0] = in[1] = sh * sh;                                            // h, j share the steady state
        if (hi) {
            e[0] = fmax(-dtl * (CK(0.77 / 0.13) * ep_rcp(1.0 + x4[0])), -1000.0);
            e[1] = fmax(-dtl * (CK(0.6) * x4[1] * E10 * ep_rcp(E10 + CK(EM32))), -1000.0);
        } else {
            e[0] = fmax(-dtl * fma(CK(0.057), x4[0], fma(CK(2.7), x4[1], 3.1e5 * x4[2])), -1000.0);
            const double N1 = fma(-2.5428e4, x4[3], CK(-6.948e-6) * x5[0]) * (vgs + CK(37.78)), D1 = 1.0 + x5[1];
            const double N2 = CK(0.02424) * x5[2], D2 = 1.0 + x5[3];
            e[1] = fmax(-dtl * (fma(N1, D2, N2 * D1) * ep_rcp(D1 * D2)), -1000.0);
        }
        {   // f2
            const double Qb = fma(CK(E3), E10, 1.0), Qc = E10 + CK(E25);
            in[2] = fma(CK(0.67), ep_rcp(fma(CK(E5C), E7, 1.0)), CK(0.33));
            e[2] = -dtl * (Qc * Qb * ep_rcp(fma(562.0 * Gf2, Qc * Qb, fma(31.0 * E10, Qb, 80.0 * Qc))));
        }
        in[3] = 0.0; e[3] = 0.0;
        rush_larsen4(e, in, Y_H - 1, Y_J - 1, Y_F2 - 1, -1);
    }
    return v_new;
}

}  // namespace epk
