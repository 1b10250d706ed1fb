// ep_stewart.cuh -- Stewart et al. 2009 human Purkinje-fibre cell model, one explicit step of one cell (device code).
//
// PAPER.md:126, :174, :256 and Table 2 (:271) name the model (ref [2]: 20 states, 13 of them gating variables advanced by
// Rush-Larsen); equations and constants are restated from the published model in DESIGN.md Appendix C (reading B13): ten
// Tusscher-Panfilov 2006 with the hyperpolarisation-activated current I_f (gate y), the sustained current I_sus, a
// time-independent I_K1, its own I_to kinetics and its own conductances.  Reading B12: the 13 Rush-Larsen variables are the
// 13 Hodgkin-Huxley gates; R' and the five concentrations are advanced by forward Euler.
//
// Production form, same rearrangements as ep_tp06.cuh: exponentials with commensurate slopes are integer
// powers of one exponential (v/600 -> 1/200, 1/25 (I_f), 1/24, 1/20, 1/15, 1/10, 1/7.5, 1/6, 1/5 and 0.11 (I_f);
// -(v+35)/13 serves tau_d, r_inf and s_inf), every sigmoid product is one rational function with a single reciprocal, the
// exponentials are evaluated four at a time right before their consumers (streaming form, see ep_tp06.cuh).  Units: mV, ms, mM, currents uA/uF.
#pragma once
#include "ep_tp06.cuh"   // CK(), the shared TP06 constants (tp06::), ep_math.cuh

namespace epk {

enum { STW_S = 20 };
// state order at the ABI: V y xr1 xr2 xs m h j d f f2 fCass s r R' Ca_i Ca_SR Ca_SS Na_i K_i
enum { W_V = 0, W_Y, W_XR1, W_XR2, W_XS, W_M, W_H, W_J, W_D, W_F, W_F2, W_FCASS, W_S, W_R, W_RP, W_CAI, W_CASR, W_CASS,
       W_NAI, W_KI };

__device__ __constant__ const double STW_INIT_STATE[STW_S] = {
    -69.1370441635924, 0.0457562667986602, 0.00550281999719088, 0.313213286437995, 0.00953708522974789,
    0.0417391656294997, 0.190678733735145, 0.238219836154029, 0.000287906256206415, 0.989328560287987,
    0.995474890442185, 0.999955429598213, 0.96386101799501, 0.00103618091196912, 0.991580051907845,
    0.000101878186157052, 3.10836886659417, 0.000446818714055411, 8.80420286531673, 136.781894160227};

namespace stw {
// constants the model shares with ten Tusscher-Panfilov 2006 (physical constants, concentrations, volumes, pump / exchanger /
// SR / buffer constants, e^c factors of the inherited gates)
using tp06::F, tp06::RTF, tp06::FRT, tp06::Ko, tp06::Cao, tp06::Nao, tp06::Vc, tp06::Vsr, tp06::Vss, tp06::Cap;
using tp06::GCaL, tp06::GbNa, tp06::GbCa, tp06::GpCa, tp06::KpCa, tp06::GpK, tp06::pKNa, tp06::PNaK, tp06::KmK, tp06::KmNa;
using tp06::kNaCa, tp06::KmNai, tp06::KmCa, tp06::ksat, tp06::alpha, tp06::Vmaxup, tp06::Kup, tp06::Vrel, tp06::k1p, tp06::k2p;
using tp06::k3, tp06::k4, tp06::EC, tp06::maxsr, tp06::minsr, tp06::Vleak, tp06::Vxfer, tp06::Bufc, tp06::Kbufc, tp06::Bufsr;
using tp06::Kbufsr, tp06::Bufss, tp06::Kbufss, tp06::LN_KO, tp06::LN_NAO, tp06::LN_KO_PNAO, tp06::LN_CAO, tp06::EM12, tp06::E7C, tp06::EM025;
using tp06::EM32, tp06::EM45, tp06::EM26_7, tp06::E88_24, tp06::EM3, tp06::EM5_14, tp06::E5_6, tp06::EM35_15, tp06::EM8_75, tp06::E1;
using tp06::E25, tp06::E20_7, tp06::E13, tp06::E3, tp06::E5C;
constexpr double GfNa = 0.0145654, GfK = 0.0234346, GK1s = 0.065, GKrs = 0.0918, GKss = 0.2352, GNas = 130.5744,
                 Gtos = 0.08184, Gsus = 0.0227;
constexpr double E06_68 = 1.092245090640267;       // e^(0.6/6.8)
constexpr double EM29 = 0.05502322005640723;       // e^(-2.9)
constexpr double E36 = 36.59823444367799;          // e^(3.6)
constexpr double E7544 = 1889.3724199964838;       // e^(7.544)
constexpr double E55_13 = 68.77011191896699;       // e^(55/13)
constexpr double EM8_13 = 0.5404329964865341;      // e^(-8/13)
constexpr double EM8 = 0.00033546262790251185;     // e^(-8)
constexpr double E5_17 = 1.3419417698828804;       // e^(5/17)

// shared-memory slots (one column of BLOCK doubles per thread): the 12 voltage-driven gate values at t^n, parked by asynchronous copies
constexpr int EXP_W = 4;     // exponentials evaluated side by side
constexpr int N_RLB = 12;    // Rush-Larsen list: 0 y, 1 xr1, 2 xr2, 3 xs, 4 m, 5 h, 6 j, 7 d, 8 f, 9 f2 (rows 1..10), 10 s, 11 r (rows 12, 13)
constexpr int G_OLD0 = 0;
constexpr int N_SLOTS = 12;
__device__ __forceinline__ constexpr int rl_row(int g) { return g < 10 ? 1 + g : 2 + g; }   // skips fCass (row 11)
}  // namespace stw

// One step of one cell (same contract as tp06_step, without cell types).  Returns Vm^{n+1}.
template <int BLOCK, class Stim, class Issue, class Finish>
__device__ __forceinline__ double stw_step(double v, double* ycol, int64_t stride, double dt, Stim stimulus,
                                           Issue issue_gather, Finish finish_gather, double* col) {
    using namespace stw;
    const double vg = ep_clamp(v, -200.0, 200.0);   // argument of every transcendental (reading T2, as TP06)
    const double dtl = dt * L2E;
    const double Cai = ep_ld_stream(ycol + W_CAI * stride), CaSR = ep_ld_stream(ycol + W_CASR * stride),
                 CaSS = ep_ld_stream(ycol + W_CASS * stride),
                 Nai = ep_ld_stream(ycol + W_NAI * stride), Ki = ep_ld_stream(ycol + W_KI * stride);
#pragma unroll
    for (int k = 0; k < N_RLB; ++k) ep_cp_async8(col + (G_OLD0 + k) * BLOCK, ycol + rl_row(k) * stride);
    const double fCass = ep_ld_stream(ycol + W_FCASS * stride), Rp = ep_ld_stream(ycol + W_RP * stride);

    // ---- batch 1: logarithms of the reversal potentials
    double lg[4] = {Ki, Nai, fma(CK(pKNa), Nai, Ki), Cai};
    ep_log_wide<4>(lg);
    issue_gather();
    const double EK = CK(RTF) * (CK(LN_KO) - lg[0]);
    const double ENa = CK(RTF) * (CK(LN_NAO) - lg[1]);
    const double EKs = CK(RTF) * (CK(LN_KO_PNAO) - lg[2]);
    const double ECa = CK(0.5 * RTF) * (CK(LN_CAO) - lg[3]);
    const double u = v - EK;
    const bool hi = (v >= -40.0);   // reading B7

    // ---- streaming form (see tp06_step): nine groups of EXP_W exponentials, each evaluated right before its consumers, so that
    // arguments and results stay in registers; the slot array only parks the 12 gate values at t^n and the stencil coefficients
    const double c2 = CaSR * CaSR, css2 = CaSS * CaSS, ci2 = Cai * Cai;
    const double kcasr = fma(-(maxsr - minsr) * c2, ep_rcp(c2 + EC * EC), maxsr);
    const double qf = ep_rcp(fma(400.0, css2, 1.0));
    const double fCass_inf = fma(CK(0.6), qf, CK(0.4));
    // group 0: the two shared gate exponentials and the two current exponentials that are raised to powers
    double x0[EXP_W] = {vg * CK(L2E / 600.0), vg * CK(L2E / 14.0), vg * CK(0.05 * FRT * L2E),
                        fma(vg, CK(2.0 * FRT * L2E), CK(-30.0 * FRT * L2E))};
    const double xcal = (vg - 15.0) * CK(2.0 * FRT);
    ep_exp2_wide<EXP_W>(x0);
    // group 1: I_pK, the Gaussian of tau_f / tau_f2, e^{-(v+80)/6.8} (y_inf, alpha_h below -40 mV), e^{-v/17} (I_sus)
    double x1[EXP_W] = {fma(vg, CK(-L2E / 5.98), CK(25.0 * L2E / 5.98)), (vg + 27.0) * (vg + 27.0) * CK(-L2E / 3600.0),
                        fma(vg, CK(-L2E / 6.8), CK(-80.0 * L2E / 6.8)), vg * CK(-L2E / 17.0)};
    ep_exp2_wide<EXP_W>(x1);
    const double dv_diff = finish_gather();
    const double istim = stimulus();          // late on purpose: see tp06_step
    ep_cp_async_wait();
    double gNa, gCaL, gto, gKr, gKs, gy;
    {
        double g[N_RLB];
#pragma unroll
        for (int k = 0; k < N_RLB; ++k) g[k] = col[(G_OLD0 + k) * BLOCK];
        // g index = position in the Rush-Larsen list: 0 y, 1 xr1, 2 xr2, 3 xs, 4 m, 5 h, 6 j, 7 d, 8 f, 9 f2, 10 s, 11 r
        gy = g[0];
        gKr = g[1] * g[2];
        gKs = g[3] * g[3];
        gNa = (g[4] * g[4] * g[4]) * g[5] * g[6];
        gCaL = (g[7] * g[8]) * (g[9] * fCass);
        gto = g[10] * g[11];
    }
    // ---- integer powers
    double E200, E24, E20, E15, E10, E7p5, E6, E5, B24, B90;
    {
        const double B = x0[0];
        const double B2 = B * B, B3 = B2 * B, B5 = B2 * B3, B10 = B5 * B5, B20 = B10 * B10, B40 = B20 * B20;
        const double B30 = B20 * B10, B60 = B30 * B30;
        E200 = B3; E24 = B20 * B5; E20 = B30; E15 = B40; E10 = B60; E7p5 = B40 * B40; E6 = B60 * B40; E5 = B60 * B60;
        B24 = B20 * (B3 * B);      // e^{0.04 v}
        B90 = B60 * B30;           // e^{0.15 v}
    }
    const double E14 = x0[1], E7 = E14 * E14;
    double W13, W18, W20;
    {
        const double W = x0[2];
        const double W2 = W * W, W4 = W2 * W2, W8 = W4 * W4, W16 = W8 * W8;
        W13 = W8 * W4 * W; W18 = W16 * W2; W20 = W18 * W2;
    }
    double Gf, Gf2;
    {
        const double b = x1[1];
        const double b2 = b * b, b4 = b2 * b2, b8 = b4 * b4;
        Gf = b8 * b8; Gf2 = (b8 * b4) * (b2 * b);
    }
    const double Y68 = x1[2];     // e^{-(v+80)/6.8}

    // ---- membrane currents
    const double INa = CK(GNas) * gNa * (v - ENa);
    double ICaL;
    {
        const double ex = x0[3];
        const double xo = (fabs(xcal) < 1e-7) ? fma(-0.5, xcal, 1.0) : xcal * ep_rcp(ex - 1.0);   // reading B6
        ICaL = CK(GCaL * 2.0 * F) * gCaL * xo * fma(0.25 * CaSS, ex, -Cao);
    }
    const double IfNa = CK(GfNa) * gy * (v - ENa);
    const double IfK = CK(GfK) * gy * u;
    const double Ito = CK(Gtos) * gto * u;
    const double IKr = CK(GKrs) * gKr * u;     // sqrt(Ko/5.4) = 1
    const double IKs = CK(GKss) * gKs * (v - EKs);
    const double IK1 = CK(GK1s) * (u - 8.0) * ep_rcp(fma(CK(E7544), E10, 1.0));     // 1/(1 + e^{0.1 (v + 75.44)})
    const double Isus = CK(Gsus) * u * ep_rcp(fma(CK(E5_17), x1[3], 1.0));   // 1/(1 + e^{(5 - v)/17})
    const double Nai3 = Nai * Nai * Nai;
    const double INaCa = CK(kNaCa / ((KmNai * KmNai * KmNai + Nao * Nao * Nao) * (KmCa + Cao)))
                         * fma(W20, Nai3 * Cao, CK(-(Nao * Nao * Nao * alpha)) * Cai) * ep_rcp(W13 + CK(ksat));
    const double INaK = CK(PNaK * Ko / (Ko + KmK)) * Nai * W20
                        * ep_rcp((Nai + KmNa) * fma(CK(0.1245), W18, W20 + CK(0.0353)));
    const double IpCa = CK(GpCa) * Cai * ep_rcp(CK(KpCa) + Cai);
    const double IpK = CK(GpK) * u * ep_rcp(1.0 + x1[0]);
    const double IbNa = CK(GbNa) * (v - ENa);
    const double IbCa = CK(GbCa) * (v - ECa);
    const double iion = IK1 + Ito + Isus + IKr + IKs + ICaL + INaK + INa + IbNa + INaCa + IbCa + IpK + IpCa + IfNa + IfK;

    // ---- sarcoplasmic-reticulum fluxes, buffer factors (reading B3), derivatives of the 7 forward-Euler states
    const double O = CK(k1p) * css2 * Rp * ep_rcp(fma(CK(k3), kcasr, CK(k1p) * css2));
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
    const double dNai = -(INa + IbNa + IfNa + 3.0 * INaK + 3.0 * INaCa) * CK(Cap / (Vc * F));
    const double dKi = -(IK1 + Ito + IfK + Isus + IKr + IKs + IpK + istim - 2.0 * INaK) * CK(Cap / (Vc * F));
    const double dRp = fma(-CK(k2p) * kcasr * CaSS, Rp, CK(k4) * (1.0 - Rp));     // reading B12: forward Euler
    const double v_new = fma(dt, dv_diff - iion - istim, v);   // eq. (7)
    ep_st_stream(ycol + W_RP * stride, fma(dt, dRp, Rp));
    ep_st_stream(ycol + W_CAI * stride, fma(dt, dCai, Cai));
    ep_st_stream(ycol + W_CASR * stride, fma(dt, dCaSR, CaSR));
    ep_st_stream(ycol + W_CASS * stride, fma(dt, dCaSS, CaSS));
    ep_st_stream(ycol + W_NAI * stride, fma(dt, dNai, Nai));
    ep_st_stream(ycol + W_KI * stride, fma(dt, dKi, Ki));

    // one Rush-Larsen group: y <- inf + (y_old - inf) 2^e for four gates (g = position in the Rush-Larsen list)
    auto rush_larsen4 = [&](double (&e)[EXP_W], const double (&in)[EXP_W], int g0, int g1, int g2, int g3) {
        const int gi[EXP_W] = {g0, g1, g2, g3};
        double yo[EXP_W];
#pragma unroll
        for (int j = 0; j < EXP_W; ++j) yo[j] = col[(G_OLD0 + gi[j]) * BLOCK];
        ep_exp2_wide<EXP_W>(e);
#pragma unroll
        for (int j = 0; j < EXP_W; ++j) ep_st_stream(ycol + rl_row(gi[j]) * stride, fma(yo[j] - in[j], e[j], in[j]));
    };
    // m, h, j, xr1 can be faster than 700/dt inside the clamp range (see the note in tp06_step), and so can y: its rate reaches
    // 3e7 per ms at +200 mV (2 per ms at +50 mV).  Their exponents are clamped to -1000: 2^-1000 stands for the oracle's 0.
    double D13, h_exp;
    // ---- group 2: m, h_inf, xr1, tau_d / r_inf / s_inf; gates y, xr1, m, d
    {
        double x2[EXP_W] = {fma(vg, CK(-L2E / 9.03), CK(-56.86 * L2E / 9.03)), fma(vg, CK(L2E / 7.43), CK(71.55 * L2E / 7.43)),
                            fma(vg, CK(L2E / 11.5), CK(30.0 * L2E / 11.5)), fma(vg, CK(-L2E / 13.0), CK(-35.0 * L2E / 13.0))};
        ep_exp2_wide<EXP_W>(x2);
        h_exp = x2[1];
        D13 = x2[3];                                                       // e^{-(v+35)/13}
        double in[EXP_W], e[EXP_W];
        in[0] = Y68 * ep_rcp(Y68 + CK(E06_68));                            // y: 1/(1 + e^{(v+80.6)/6.8})
        e[0] = fmax(-dtl * (fma(CK(E36), B90, CK(EM29)) * ep_rcp(4000.0 * B24)), -1000.0);   // tau = 4000/(e^{-2.9-0.04v} + e^{3.6+0.11v})
        in[1] = E7 * ep_rcp(E7 + CK(EM26_7));                              // xr1
        e[1] = fmax(-dtl * ((E10 + CK(EM45)) * (1.0 + x2[2]) * ep_rcp(2700.0 * E10)), -1000.0);
        {   // m
            const double sm = ep_rcp(1.0 + x2[0]);
            in[2] = sm * sm;
            const double P = fma(CK(E7C), E5, 1.0), Q = fma(CK(EM025), E200, 1.0);
            e[2] = fmax(-dtl * ((E5 + CK(EM12)) * P * Q * ep_rcp(CK(0.1) * E5 * (P + Q))), -1000.0);
        }
        {   // d
            in[3] = E7p5 * ep_rcp(E7p5 + CK(EM8_75));
            const double D = 1.0 + D13, P5 = fma(CK(E1), E5, 1.0), Q20 = E20 + CK(E25);
            e[3] = -dtl * (D * P5 * Q20 * ep_rcp(fma(fma(0.25, D, CK(1.4)) * CK(1.4), Q20, E20 * D * P5)));
        }
        rush_larsen4(e, in, 0, 1, 4, 7);
    }
    // ---- group 3: the Gaussians of tau_r and tau_s, exp(-dt/tau) of fCass; gates xr2, xs, s, r
    {
        double x3[EXP_W] = {(vg + 40.0) * (vg + 40.0) * CK(-L2E / 1800.0), (vg + 25.0) * (vg + 25.0) * CK(-L2E / 320.0),
                            -dtl * ep_rcp(fma(80.0, qf, 2.0)), 0.0};
        ep_exp2_wide<EXP_W>(x3);
        ep_st_stream(ycol + W_FCASS * stride, fma(fCass - fCass_inf, x3[2], fCass_inf));   // Rush-Larsen
        double in[EXP_W], e[EXP_W];
        in[0] = ep_rcp(fma(CK(E88_24), E24, 1.0));                                                     // xr2
        e[0] = -dtl * ((E20 + CK(EM3)) * fma(CK(EM3), E20, 1.0) * ep_rcp(CK(3.36) * E20));
        {   // xs
            in[1] = E14 * ep_rcp(E14 + CK(EM5_14));
            const double t = ep_rsqrt((E6 + CK(E5_6)) * E6) * E6;
            const double P15 = fma(CK(EM35_15), E15, 1.0);
            e[1] = -dtl * (P15 * ep_rcp(fma(1400.0, t, 80.0 * P15)));
        }
        {   // s, r of the Purkinje transient outward current
            in[2] = D13 * ep_rcp(D13 + CK(EM8_13));                        // 1/(1 + e^{(v+27)/13})
            const double P = fma(CK(EM8), E5, 1.0);                        // 1 + e^{(v-40)/5}
            e[2] = -dtl * (P * ep_rcp(fma(fma(85.0, x3[1], 42.0), P, 5.0)));
            in[3] = ep_rcp(fma(CK(E55_13), D13, 1.0));                     // 1/(1 + e^{(20-v)/13})
            e[3] = -dtl * ep_rcp(fma(10.45, x3[0], CK(7.3)));
        }
        rush_larsen4(e, in, 2, 3, 10, 11);
    }
    // ---- groups 4, 5: the h / j rate exponentials (the second group is skipped when every cell of the warp is above -40 mV);
    // gates h, j, f, f2
    {
        double x4[EXP_W], x5[EXP_W] = {1.0, 1.0, 1.0, 1.0};
        const bool all_hi = __all_sync(__activemask(), hi);
        if (hi) {
            x4[0] = fma(vg, CK(-L2E / 11.1), CK(-10.66 * L2E / 11.1));
            x4[1] = vg * CK(0.057 * L2E);
            x4[2] = 0.0; x4[3] = 0.0;
        } else {
            x4[0] = vg * CK(0.079 * L2E);
            x4[1] = vg * CK(0.3485 * L2E);
            x4[2] = vg * CK(0.2444 * L2E);
            x4[3] = vg * CK(-0.04391 * L2E);
        }
        ep_exp2_wide<EXP_W>(x4);
        if (!all_hi) {
            x5[0] = fma(vg, CK(0.311 * L2E), CK(0.311 * 79.23 * L2E));
            x5[1] = vg * CK(-0.01052 * L2E);
            x5[2] = fma(vg, CK(-0.1378 * L2E), CK(-0.1378 * 40.14 * L2E));
            x5[3] = 0.0;
            ep_exp2_wide<EXP_W>(x5);
        }
        double in[EXP_W], e[EXP_W];
        const double sh = ep_rcp(1.0 + h_exp);
        in[0] = in[1] = sh * sh;
        if (hi) {
            e[0] = fmax(-dtl * (CK(0.77 / 0.13) * ep_rcp(1.0 + x4[0])), -1000.0);
            e[1] = fmax(-dtl * (CK(0.6) * x4[1] * E10 * ep_rcp(E10 + CK(EM32))), -1000.0);
        } else {
            e[0] = fmax(-dtl * fma(CK(0.057), Y68, fma(CK(2.7), x4[0], 3.1e5 * x4[1])), -1000.0);
            const double N1 = fma(-2.5428e4, x4[2], CK(-6.948e-6) * x4[3]) * (vg + CK(37.78)), D1 = 1.0 + x5[0];
            const double N2 = CK(0.02424) * x5[1], D2 = 1.0 + x5[2];
            e[1] = fmax(-dtl * (fma(N1, D2, N2 * D1) * ep_rcp(D1 * D2)), -1000.0);
        }
        {   // f, f2 (as TP06)
            const double Qa = E10 + CK(E13), Qb = fma(CK(E3), E10, 1.0), Qc = E10 + CK(E25);
            in[2] = ep_rcp(fma(CK(E20_7), E7, 1.0));
            e[2] = -dtl * (Qa * Qb * ep_rcp(fma(fma(1102.5, Gf, 20.0), Qa * Qb, fma(200.0 * E10, Qb, 180.0 * Qa))));
            in[3] = fma(CK(0.67), ep_rcp(fma(CK(E5C), E7, 1.0)), CK(0.33));
            e[3] = -dtl * (Qc * Qb * ep_rcp(fma(562.0 * Gf2, Qc * Qb, fma(31.0 * E10, Qb, 80.0 * Qc))));
        }
        rush_larsen4(e, in, 5, 6, 8, 9);
    }
    return v_new;
}

}  // namespace epk
