// ep_oracle.cpp -- CPU ORACLE. TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct fp64 implementation of the explicit monodomain time step of
// arXiv 2112.12854 (section 3.2) on a tetrahedral cell-centred finite-volume mesh, with the
// ten Tusscher-Panfilov 2006 ventricular cell model (ref [3]) -- and the Courtemanche atrial model
// (ref [1], config 5) -- integrated by Rush-Larsen
// (gates) and forward Euler (everything else).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use this file.
// It shares no code, header, table or helper with the CUDA path (paper_2112_12854_b200/csrc) and neither
// includes the other. It follows the paper's Fig. 8 pipeline a->e literally: no operator
// collapsing, no blocking, no fusion. Readings of silent/ambiguous points are the ones listed in DESIGN.md
// section 3 (A1..A18, B1..B9). Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC.
// The OpenMP loops are all over independent cells / nodes / faces (no reductions), so results are
// bit-identical for any thread count; the default is ONE thread.
//
// Parity pins (tests/test_oracle_*.py): row sums, conservation, linear-field exactness, Gauss-Green identity,
// dense brute force vs an independent numpy assembly, RL closed form, single-cell rest/AP facts from
// PAPER.md:256, 1st-order-in-time trend, CV refinement trend. Unpinned: Niederer activation-time table
// (values not available) -- "parity unpinned" for that comparison only.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------------------------------------
// TP06 (ref [3] of the paper; statement in DESIGN.md Appendix A). Units: mV, ms, mM, uA/uF, nS/pF.
// State order: 0 v, 1 m, 2 h, 3 j, 4 xr1, 5 xr2, 6 xs, 7 r, 8 s, 9 d, 10 f, 11 f2, 12 fCass, 13 Rbar,
//              14 Ca_i, 15 Ca_SR, 16 Ca_SS, 17 Na_i, 18 K_i.
const int TP06_S = 19;
const double R_gas = 8314.472, T_abs = 310.0, F_far = 96485.3415;
const double RTF = R_gas * T_abs / F_far;
const double K_o = 5.4, Ca_o = 2.0, Na_o = 140.0;
const double V_c = 0.016404, V_sr = 0.001094, V_ss = 0.00005468, Cap = 0.185;
const double G_Na = 14.838, G_K1 = 5.405, G_Kr = 0.153, G_CaL = 3.980e-5, G_bNa = 2.9e-4, G_bCa = 5.92e-4;
const double G_pCa = 0.1238, K_pCa = 5e-4, G_pK = 0.0146, p_KNa = 0.03;
const double P_NaK = 2.724, K_mK = 1.0, K_mNa = 40.0;
const double k_NaCa = 1000.0, K_mNai = 87.5, K_mCa = 1.38, k_sat = 0.1, gam = 0.35, alp = 2.5;
const double V_maxup = 0.006375, K_up = 2.5e-4, V_rel = 0.102, k1p = 0.15, k2p = 0.045, k3 = 0.060, k4 = 0.005;
const double EC = 1.5, max_sr = 2.5, min_sr = 1.0, V_leak = 3.6e-4, V_xfer = 0.0038;
const double Buf_c = 0.2, K_bufc = 0.001, Buf_sr = 10.0, K_bufsr = 0.3, Buf_ss = 0.4, K_bufss = 2.5e-4;

const double TP06_REST[TP06_S] = {-86.2, 0.0, 0.75, 0.75, 0.0, 1.0, 0.0, 0.0, 1.0, 0.0, 1.0, 1.0, 1.0, 1.0,
                                  7e-5, 1.3, 7e-5, 7.67, 138.3};

inline double sig(double z) { return 1.0 / (1.0 + std::exp(z)); }  // sigma(z) = 1/(1+e^z)

// Steady states and time constants of the 13 Rush-Larsen variables (reading B1: 12 HH gates + Rbar).
// Index g = state index - 1 (0 m ... 11 fCass, 12 Rbar).
void tp06_gates(double v, int type, double Ca_SS, double Ca_SR, double* inf, double* tau) {
    // m
    { double s = sig((-56.86 - v) / 9.03); inf[0] = s * s;
      tau[0] = sig((-60.0 - v) / 5.0) * (0.1 * sig((v + 35.0) / 5.0) + 0.1 * sig((v - 50.0) / 200.0)); }
    // h, j (reading B7: v >= -40 takes the high-voltage branch)
    { double s = sig((v + 71.55) / 7.43); inf[1] = s * s; inf[2] = s * s;
      double ah, bh, aj, bj;
      if (v >= -40.0) {
          ah = 0.0; bh = 0.77 / (0.13 * (1.0 + std::exp(-(v + 10.66) / 11.1)));
          aj = 0.0; bj = 0.6 * std::exp(0.057 * v) / (1.0 + std::exp(-0.1 * (v + 32.0)));
      } else {
          ah = 0.057 * std::exp(-(v + 80.0) / 6.8);
          bh = 2.7 * std::exp(0.079 * v) + 3.1e5 * std::exp(0.3485 * v);
          aj = (-2.5428e4 * std::exp(0.2444 * v) - 6.948e-6 * std::exp(-0.04391 * v)) * (v + 37.78)
               / (1.0 + std::exp(0.311 * (v + 79.23)));
          bj = 0.02424 * std::exp(-0.01052 * v) / (1.0 + std::exp(-0.1378 * (v + 40.14)));
      }
      tau[1] = 1.0 / (ah + bh); tau[2] = 1.0 / (aj + bj); }
    // xr1, xr2, xs
    inf[3] = sig((-26.0 - v) / 7.0);
    tau[3] = 450.0 * sig((-45.0 - v) / 10.0) * 6.0 * sig((v + 30.0) / 11.5);
    inf[4] = sig((v + 88.0) / 24.0);
    tau[4] = 3.0 * sig((-60.0 - v) / 20.0) * 1.12 * sig((v - 60.0) / 20.0);
    inf[5] = sig((-5.0 - v) / 14.0);
    tau[5] = 1400.0 / std::sqrt(1.0 + std::exp((5.0 - v) / 6.0)) * sig((v - 35.0) / 15.0) + 80.0;
    // r, s (reading B5: endo has its own s curves)
    inf[6] = sig((20.0 - v) / 6.0);
    tau[6] = 9.5 * std::exp(-(v + 40.0) * (v + 40.0) / 1800.0) + 0.8;
    if (type == 0) {
        inf[7] = sig((v + 28.0) / 5.0);
        tau[7] = 1000.0 * std::exp(-(v + 67.0) * (v + 67.0) / 1000.0) + 8.0;
    } else {
        inf[7] = sig((v + 20.0) / 5.0);
        tau[7] = 85.0 * std::exp(-(v + 45.0) * (v + 45.0) / 320.0) + 5.0 * sig((v - 20.0) / 5.0) + 3.0;
    }
    // d, f, f2
    inf[8] = sig((-8.0 - v) / 7.5);
    tau[8] = (1.4 * sig((-35.0 - v) / 13.0) + 0.25) * (1.4 * sig((v + 5.0) / 5.0)) + sig((50.0 - v) / 20.0);
    inf[9] = sig((v + 20.0) / 7.0);
    tau[9] = 1102.5 * std::exp(-(v + 27.0) * (v + 27.0) / 225.0) + 200.0 * sig((13.0 - v) / 10.0)
             + 180.0 * sig((v + 30.0) / 10.0) + 20.0;
    inf[10] = 0.67 * sig((v + 35.0) / 7.0) + 0.33;
    tau[10] = 562.0 * std::exp(-(v + 27.0) * (v + 27.0) / 240.0) + 31.0 * sig((25.0 - v) / 10.0)
              + 80.0 * sig((v + 30.0) / 10.0);
    // fCass
    { double q = 1.0 + (Ca_SS / 0.05) * (Ca_SS / 0.05);
      inf[11] = 0.6 / q + 0.4; tau[11] = 80.0 / q + 2.0; }
    // Rbar: dR/dt = k4 (1-R) - k2 Ca_SS R  (linear in R at frozen Ca)
    { double kcasr = max_sr - (max_sr - min_sr) / (1.0 + (EC / Ca_SR) * (EC / Ca_SR));
      double k2 = k2p * kcasr;
      inf[12] = k4 / (k2 * Ca_SS + k4); tau[12] = 1.0 / (k2 * Ca_SS + k4); }
}

struct Tp06Currents {
    double INa, ICaL, Ito, IKr, IKs, IK1, INaCa, INaK, IpCa, IpK, IbNa, IbCa, iion;
    double Irel, Ileak, Iup, Ixfer;
};

void tp06_currents(const double* y, int type, Tp06Currents& c) {
    const double v = y[0], m = y[1], h = y[2], j = y[3], xr1 = y[4], xr2 = y[5], xs = y[6], r = y[7], s = y[8];
    const double d = y[9], f = y[10], f2 = y[11], fcass = y[12], Rbar = y[13];
    const double Ca_i = y[14], Ca_SR = y[15], Ca_SS = y[16], Na_i = y[17], K_i = y[18];
    const double G_Ks = (type == 1) ? 0.098 : 0.392;
    const double G_to = (type == 0) ? 0.073 : 0.294;
    const double E_K = RTF * std::log(K_o / K_i);
    const double E_Na = RTF * std::log(Na_o / Na_i);
    const double E_Ks = RTF * std::log((K_o + p_KNa * Na_o) / (K_i + p_KNa * Na_i));
    const double E_Ca = 0.5 * RTF * std::log(Ca_o / Ca_i);
    c.INa = G_Na * m * m * m * h * j * (v - E_Na);
    {   // reading B6: x/(e^x-1) -> 1 - x/2 for |x| < 1e-7
        const double x = 2.0 * (v - 15.0) / RTF;
        const double ex = std::exp(x);
        double xo;  // x / (e^x - 1)
        if (std::fabs(x) < 1e-7) xo = 1.0 - 0.5 * x; else xo = x / (ex - 1.0);
        // 4 (v-15) F/RTF * (0.25 Ca_SS e^x - Ca_o)/(e^x - 1) = 2 F * [x/(e^x-1)] * (0.25 Ca_SS e^x - Ca_o)
        c.ICaL = G_CaL * d * f * f2 * fcass * 2.0 * F_far * xo * (0.25 * Ca_SS * ex - Ca_o);
    }
    c.Ito = G_to * r * s * (v - E_K);
    c.IKr = G_Kr * std::sqrt(K_o / 5.4) * xr1 * xr2 * (v - E_K);
    c.IKs = G_Ks * xs * xs * (v - E_Ks);
    {
        const double a = 0.1 / (1.0 + std::exp(0.06 * (v - E_K - 200.0)));
        const double b = (3.0 * std::exp(0.0002 * (v - E_K + 100.0)) + std::exp(0.1 * (v - E_K - 10.0)))
                         / (1.0 + std::exp(-0.5 * (v - E_K)));
        c.IK1 = G_K1 * (a / (a + b)) * (v - E_K);
    }
    {
        const double e1 = std::exp(gam * v / RTF), e2 = std::exp((gam - 1.0) * v / RTF);
        c.INaCa = k_NaCa * (e1 * Na_i * Na_i * Na_i * Ca_o - e2 * Na_o * Na_o * Na_o * Ca_i * alp)
                  / ((K_mNai * K_mNai * K_mNai + Na_o * Na_o * Na_o) * (K_mCa + Ca_o) * (1.0 + k_sat * e2));
    }
    c.INaK = P_NaK * (K_o / (K_o + K_mK)) * (Na_i / (Na_i + K_mNa))
             / (1.0 + 0.1245 * std::exp(-0.1 * v / RTF) + 0.0353 * std::exp(-v / RTF));
    c.IpCa = G_pCa * Ca_i / (K_pCa + Ca_i);
    c.IpK = G_pK * (v - E_K) / (1.0 + std::exp((25.0 - v) / 5.98));
    c.IbNa = G_bNa * (v - E_Na);
    c.IbCa = G_bCa * (v - E_Ca);
    c.iion = c.INa + c.ICaL + c.Ito + c.IKr + c.IKs + c.IK1 + c.INaCa + c.INaK + c.IpCa + c.IpK + c.IbNa + c.IbCa;
    {
        const double kcasr = max_sr - (max_sr - min_sr) / (1.0 + (EC / Ca_SR) * (EC / Ca_SR));
        const double k1 = k1p / kcasr;
        const double O = k1 * Ca_SS * Ca_SS * Rbar / (k3 + k1 * Ca_SS * Ca_SS);
        c.Irel = V_rel * O * (Ca_SR - Ca_SS);
        c.Ileak = V_leak * (Ca_SR - Ca_i);
        c.Iup = V_maxup / (1.0 + K_up * K_up / (Ca_i * Ca_i));
        c.Ixfer = V_xfer * (Ca_SS - Ca_i);
    }
}

// One explicit step of one cell, everything on the right-hand side at t^n (reading A13).
// dv_diff = D_c/(chi C_m) in mV/ms, istim = I_s/C_m in uA/uF. yn may not alias y.
void tp06_step(const double* y, int type, double dt, double istim, double dv_diff, double* yn) {
    Tp06Currents c;
    tp06_currents(y, type, c);
    double inf[13], tau[13];
    tp06_gates(y[0], type, y[16], y[15], inf, tau);
    for (int g = 0; g < 13; ++g)  // Rush-Larsen
        yn[1 + g] = inf[g] + (y[1 + g] - inf[g]) * std::exp(-dt / tau[g]);
    const double Ca_i = y[14], Ca_SR = y[15], Ca_SS = y[16];
    const double bi = 1.0 / (1.0 + Buf_c * K_bufc / ((Ca_i + K_bufc) * (Ca_i + K_bufc)));     // reading B3
    const double bsr = 1.0 / (1.0 + Buf_sr * K_bufsr / ((Ca_SR + K_bufsr) * (Ca_SR + K_bufsr)));
    const double bss = 1.0 / (1.0 + Buf_ss * K_bufss / ((Ca_SS + K_bufss) * (Ca_SS + K_bufss)));
    const double dCai = bi * ((c.Ileak - c.Iup) * V_sr / V_c + c.Ixfer
                              - (c.IbCa + c.IpCa - 2.0 * c.INaCa) * Cap / (2.0 * V_c * F_far));
    const double dCaSR = bsr * (c.Iup - c.Ileak - c.Irel);
    const double dCaSS = bss * (-c.ICaL * Cap / (2.0 * V_ss * F_far) + c.Irel * V_sr / V_ss - c.Ixfer * V_c / V_ss);
    const double dNai = -(c.INa + c.IbNa + 3.0 * c.INaK + 3.0 * c.INaCa) * Cap / (V_c * F_far);
    const double dKi = -(c.IK1 + c.Ito + c.IKr + c.IKs - 2.0 * c.INaK + c.IpK + istim) * Cap / (V_c * F_far);  // B8
    yn[14] = Ca_i + dt * dCai;
    yn[15] = Ca_SR + dt * dCaSR;
    yn[16] = Ca_SS + dt * dCaSS;
    yn[17] = y[17] + dt * dNai;
    yn[18] = y[18] + dt * dKi;
    yn[0] = y[0] + dt * (dv_diff - c.iion - istim);  // eq. (7), explicit increment :172
}


// ---------------------------------------------------------------------------------------------------------
// Courtemanche-Ramirez-Nattel 1998 human atrial cell model (ref [1] PAPER.md:352: 21 state
// variables, 15 of them gating variables advanced by Rush-Larsen).  Equations and constants restated from the
// published model (DESIGN.md Appendix B).  Units: mV, ms, mM; currents are per unit capacitance (pA/pF = uA/uF);
// where the published concentration equations use whole-cell currents in pA they are multiplied by C_m = 100 pF.
// State order: 0 V, 1 m, 2 h, 3 j, 4 oa, 5 oi, 6 ua, 7 ui, 8 xr, 9 xs, 10 d, 11 f, 12 fCa, 13 u, 14 v, 15 w,
//              16 Na_i, 17 K_i, 18 Ca_i, 19 Ca_up, 20 Ca_rel.
namespace crn {
const int S = 21;
const double R = 8.3143, T = 310.0, F = 96.4867;          // J/(K mol), K, C/mmol
const double RTF = R * T / F;                              // mV
const double Cm = 100.0;                                   // pF
const double Vi = 13668.0, Vup = 1109.52, Vrel = 96.48;    // um^3
const double Ko = 5.4, Nao = 140.0, Cao = 1.8;
const double gNa = 7.8, gK1 = 0.09, gto = 0.1652, gKr = 0.0294, gKs = 0.129, gCaL = 0.1238, gbCa = 0.00113, gbNa = 0.000674;
const double INaKmax = 0.60, INaCamax = 1600.0, IpCamax = 0.275, Iupmax = 0.005;
const double KQ10 = 3.0, gam = 0.35, KmNai = 10.0, KmKo = 1.5, KmNa = 87.5, KmCa = 1.38, ksat = 0.1;
const double krel = 30.0, Kup = 0.00092, Caupmax = 15.0, tau_tr = 180.0, tau_fCa = 2.0, tau_u = 8.0;
const double Cmdnmax = 0.05, Trpnmax = 0.07, Csqnmax = 10.0, KmCmdn = 0.00238, KmTrpn = 0.0005, KmCsqn = 0.8;
const double REST[S] = {-81.18, 2.91e-3, 0.965, 0.978, 0.0304, 0.999, 4.96e-3, 0.999, 3.29e-5, 0.0187, 1.37e-4, 0.999,
                        0.775, 0.0, 1.0, 0.999, 11.17, 139.0, 1.013e-4, 1.488, 1.488};

// phi(x) = x/(e^x - 1); reading B11: 1 - x/2 + x^2/12 for |x| < 1e-4 (removable singularities of the alpha/beta and
// tau expressions at V = -47.13, -14.1, 3.3328, 19.9, -10, 7.9 mV)
inline double phi(double x) {
    if (std::fabs(x) < 1e-4) return 1.0 - 0.5 * x + x * x / 12.0;
    return x / (std::exp(x) - 1.0);
}

struct Currents {
    double INa, IK1, Ito, IKur, IKr, IKs, ICaL, IpCa, INaK, INaCa, IbNa, IbCa, iion;
    double Irel, Itr, Iup, Iupleak, Fn;
};

void currents(const double* y, Currents& c) {
    const double V = y[0], m = y[1], h = y[2], j = y[3], oa = y[4], oi = y[5], ua = y[6], ui = y[7], xr = y[8], xs = y[9];
    const double d = y[10], f = y[11], fCa = y[12], u = y[13], v = y[14], w = y[15];
    const double Nai = y[16], Ki = y[17], Cai = y[18], Caup = y[19], Carel = y[20];
    const double ENa = RTF * std::log(Nao / Nai), EK = RTF * std::log(Ko / Ki), ECa = 0.5 * RTF * std::log(Cao / Cai);
    c.INa = gNa * m * m * m * h * j * (V - ENa);
    c.IK1 = gK1 * (V - EK) / (1.0 + std::exp(0.07 * (V + 80.0)));
    c.Ito = gto * oa * oa * oa * oi * (V - EK);
    const double gKur = 0.005 + 0.05 / (1.0 + std::exp(-(V - 15.0) / 13.0));
    c.IKur = gKur * ua * ua * ua * ui * (V - EK);
    c.IKr = gKr * xr * (V - EK) / (1.0 + std::exp((V + 15.0) / 22.4));
    c.IKs = gKs * xs * xs * (V - EK);
    c.ICaL = gCaL * d * f * fCa * (V - 65.0);
    const double sigma = (std::exp(Nao / 67.3) - 1.0) / 7.0;
    const double fNaK = 1.0 / (1.0 + 0.1245 * std::exp(-0.1 * V / RTF) + 0.0365 * sigma * std::exp(-V / RTF));
    c.INaK = INaKmax * fNaK / (1.0 + std::pow(KmNai / Nai, 1.5)) * Ko / (Ko + KmKo);
    {
        const double e1 = std::exp(gam * V / RTF), e2 = std::exp((gam - 1.0) * V / RTF);
        c.INaCa = INaCamax * (e1 * Nai * Nai * Nai * Cao - e2 * Nao * Nao * Nao * Cai)
                  / ((KmNa * KmNa * KmNa + Nao * Nao * Nao) * (KmCa + Cao) * (1.0 + ksat * e2));
    }
    c.IbCa = gbCa * (V - ECa);
    c.IbNa = gbNa * (V - ENa);
    c.IpCa = IpCamax * Cai / (0.0005 + Cai);
    c.iion = c.INa + c.IK1 + c.Ito + c.IKur + c.IKr + c.IKs + c.ICaL + c.IpCa + c.INaK + c.INaCa + c.IbNa + c.IbCa;
    c.Irel = krel * u * u * v * w * (Carel - Cai);
    c.Itr = (Caup - Carel) / tau_tr;
    c.Iup = Iupmax / (1.0 + Kup / Cai);
    c.Iupleak = Caup / Caupmax * Iupmax;
    // flux signal driving the u and v gates; whole-cell currents in pA = C_m * (pA/pF)
    c.Fn = 1e-12 * Vrel * c.Irel - (5e-13 / F) * (0.5 * Cm * c.ICaL - 0.2 * Cm * c.INaCa);
}

// steady states and time constants of the 15 gates, index g = state index - 1
void gates(double V, double Cai, double Fn, double* inf, double* tau) {
    {   // m
        const double am = 3.2 * phi(-0.1 * (V + 47.13));     // 0.32 (V+47.13)/(1 - exp(-0.1 (V+47.13)))
        const double bm = 0.08 * std::exp(-V / 11.0);
        inf[0] = am / (am + bm); tau[0] = 1.0 / (am + bm);
    }
    {   // h, j: V >= -40 takes the high-voltage branch (reading B7)
        double ah, bh, aj, bj;
        if (V >= -40.0) {
            ah = 0.0; bh = 1.0 / (0.13 * (1.0 + std::exp(-(V + 10.66) / 11.1)));
            aj = 0.0; bj = 0.3 * std::exp(-2.535e-7 * V) / (1.0 + std::exp(-0.1 * (V + 32.0)));
        } else {
            ah = 0.135 * std::exp(-(V + 80.0) / 6.8);
            bh = 3.56 * std::exp(0.079 * V) + 3.1e5 * std::exp(0.35 * V);
            aj = (-127140.0 * std::exp(0.2444 * V) - 3.474e-5 * std::exp(-0.04391 * V)) * (V + 37.78)
                 / (1.0 + std::exp(0.311 * (V + 79.23)));
            bj = 0.1212 * std::exp(-0.01052 * V) / (1.0 + std::exp(-0.1378 * (V + 40.14)));
        }
        inf[1] = ah / (ah + bh); tau[1] = 1.0 / (ah + bh);
        inf[2] = aj / (aj + bj); tau[2] = 1.0 / (aj + bj);
    }
    {   // oa, ua share alpha and beta
        const double a = 0.65 / (std::exp(-(V + 10.0) / 8.5) + std::exp(-(V - 30.0) / 59.0));
        const double b = 0.65 / (2.5 + std::exp((V + 82.0) / 17.0));
        inf[3] = 1.0 / (1.0 + std::exp(-(V + 20.47) / 17.54)); tau[3] = 1.0 / (a + b) / KQ10;
        inf[5] = 1.0 / (1.0 + std::exp(-(V + 30.3) / 9.6));     tau[5] = 1.0 / (a + b) / KQ10;
    }
    {   // oi
        const double a = 1.0 / (18.53 + std::exp((V + 113.7) / 10.95));
        const double b = 1.0 / (35.56 + std::exp(-(V + 1.26) / 7.44));
        inf[4] = 1.0 / (1.0 + std::exp((V + 43.1) / 5.3)); tau[4] = 1.0 / (a + b) / KQ10;
    }
    {   // ui
        const double a = 1.0 / (21.0 + std::exp(-(V - 185.0) / 28.0));
        const double b = std::exp((V - 158.0) / 16.0);
        inf[6] = 1.0 / (1.0 + std::exp((V - 99.45) / 27.48)); tau[6] = 1.0 / (a + b) / KQ10;
    }
    {   // xr
        const double a = 0.0015 * phi(-(V + 14.1) / 5.0);                    // 0.0003 (V+14.1)/(1 - exp(-(V+14.1)/5))
        const double b = 7.3898e-5 * 5.1237 * phi((V - 3.3328) / 5.1237);    // 7.3898e-5 (V-3.3328)/(exp((V-3.3328)/5.1237) - 1)
        inf[7] = 1.0 / (1.0 + std::exp(-(V + 14.1) / 6.5)); tau[7] = 1.0 / (a + b);
    }
    {   // xs
        const double a = 4e-5 * 17.0 * phi(-(V - 19.9) / 17.0);              // 4e-5 (V-19.9)/(1 - exp(-(V-19.9)/17))
        const double b = 3.5e-5 * 9.0 * phi((V - 19.9) / 9.0);               // 3.5e-5 (V-19.9)/(exp((V-19.9)/9) - 1)
        inf[8] = 1.0 / std::sqrt(1.0 + std::exp(-(V - 19.9) / 12.7)); tau[8] = 0.5 / (a + b);
    }
    {   // d: tau = (1 - e^x)/(0.035 (V+10)(1 + e^x)), x = -(V+10)/6.24
        const double x = -(V + 10.0) / 6.24;
        inf[9] = 1.0 / (1.0 + std::exp(-(V + 10.0) / 8.0));
        tau[9] = 1.0 / (0.035 * 6.24 * phi(x) * (1.0 + std::exp(x)));
    }
    {   // f
        inf[10] = 1.0 / (1.0 + std::exp((V + 28.0) / 6.9));
        tau[10] = 9.0 / (0.0197 * std::exp(-0.0337 * 0.0337 * (V + 10.0) * (V + 10.0)) + 0.02);
    }
    inf[11] = 1.0 / (1.0 + Cai / 0.00035); tau[11] = tau_fCa;   // fCa
    {   // u, v driven by Fn
        const double e1 = std::exp(-(Fn - 3.4175e-13) / 13.67e-16);
        inf[12] = 1.0 / (1.0 + e1); tau[12] = tau_u;
        inf[13] = 1.0 - 1.0 / (1.0 + std::exp(-(Fn - 6.835e-14) / 13.67e-16));
        tau[13] = 1.91 + 2.09 / (1.0 + e1);
    }
    {   // w: tau = 6 (1 - e^x)/((1 + 0.3 e^x)(V-7.9)), x = -(V-7.9)/5
        const double x = -(V - 7.9) / 5.0;
        inf[14] = 1.0 - 1.0 / (1.0 + std::exp(-(V - 40.0) / 17.0));
        tau[14] = 6.0 / (5.0 * phi(x) * (1.0 + 0.3 * std::exp(x)));
    }
}

// One explicit step of one cell: gates by Rush-Larsen, the rest by forward Euler, all from t^n.
void step(const double* y, double dt, double istim, double dv_diff, double* yn) {
    Currents c;
    currents(y, c);
    double inf[15], tau[15];
    gates(y[0], y[18], c.Fn, inf, tau);
    for (int g = 0; g < 15; ++g) yn[1 + g] = inf[g] + (y[1 + g] - inf[g]) * std::exp(-dt / tau[g]);
    const double Cai = y[18], Caup = y[19], Carel = y[20];
    const double FVi = F * Vi;
    // whole-cell currents in pA = C_m * per-capacitance currents (reading B10: the stimulus is not counted in dK_i/dt)
    const double dNai = Cm * (-3.0 * c.INaK - 3.0 * c.INaCa - c.IbNa - c.INa) / FVi;
    const double dKi = Cm * (2.0 * c.INaK - c.IK1 - c.Ito - c.IKur - c.IKr - c.IKs) / FVi;
    const double B1 = Cm * (2.0 * c.INaCa - c.IpCa - c.ICaL - c.IbCa) / (2.0 * FVi)
                      + (Vup * (c.Iupleak - c.Iup) + c.Irel * Vrel) / Vi;
    const double B2 = 1.0 + Trpnmax * KmTrpn / ((Cai + KmTrpn) * (Cai + KmTrpn))
                      + Cmdnmax * KmCmdn / ((Cai + KmCmdn) * (Cai + KmCmdn));
    const double dCaup = c.Iup - c.Iupleak - c.Itr * Vrel / Vup;
    const double dCarel = (c.Itr - c.Irel) / (1.0 + Csqnmax * KmCsqn / ((Carel + KmCsqn) * (Carel + KmCsqn)));
    yn[16] = y[16] + dt * dNai;
    yn[17] = y[17] + dt * dKi;
    yn[18] = Cai + dt * (B1 / B2);
    yn[19] = Caup + dt * dCaup;
    yn[20] = Carel + dt * dCarel;
    yn[0] = y[0] + dt * (dv_diff - c.iion - istim);
}
}  // namespace crn

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// Finite-volume mesh and the literal Fig. 8 pipeline.
namespace {

struct Vec3 { double x, y, z; };
inline Vec3 operator+(Vec3 a, Vec3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline Vec3 operator-(Vec3 a, Vec3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline Vec3 operator*(double s, Vec3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(Vec3 a, Vec3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline Vec3 cross(Vec3 a, Vec3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(Vec3 a) { return std::sqrt(dot(a, a)); }

struct Sym3 { double xx, xy, xz, yy, yz, zz; };
inline Vec3 mul(const Sym3& m, Vec3 a) {
    return {m.xx * a.x + m.xy * a.y + m.xz * a.z, m.xy * a.x + m.yy * a.y + m.yz * a.z,
            m.xz * a.x + m.yz * a.y + m.zz * a.z};
}

struct Face {            // interior face, c1 = lower cell id, normal outward of c1 (DESIGN.md 8(c) step 4)
    int64_t c1, c2;
    Vec3 s;              // area vector A_f n_f, outward of c1 (reading A5)
    double a1, a2;       // alpha_c1, alpha_c2 (reading A6)
    Vec3 e;              // unit vector from c2 to c1 (reading A7)
    double d;            // |x_c1 - x_c2|
    Sym3 Mf;             // alpha-weighted arithmetic mean (reading A8)
};

struct Stim { std::vector<char> mask; double amp, t0, dur; bool set; };
// triggered stimulus = communication-node coupling inside one mesh: first crossing of 0 mV by a
// monitored cell arms slot `slot` to start `delay` later
struct Trigger { std::vector<int64_t> cells; int slot = 0; double delay = 0.0; bool armed = false; int64_t n_fire1 = -1; };

struct Sim {
    int64_t nn = 0, nc = 0;
    std::vector<Vec3> x;               // nodes
    std::vector<int32_t> tet;          // [nc*4]
    std::vector<Vec3> xc;              // centroids (reading A1)
    std::vector<double> vol;
    std::vector<Vec3> sf;              // [nc*4] outward area vector of face j (opposite vertex j)
    std::vector<Sym3> Mc;
    std::vector<Face> faces;
    std::vector<int64_t> cell_face;    // [nc*4] interior face id or -1 (boundary, reading A11)
    std::vector<int64_t> star_ptr, star_cell;   // node -> cells, ascending cell id
    std::vector<double> star_invd;     // 1/d_k (reading A2)
    double chi = 0, Cm = 0;
    int model = -1, S = 0;
    std::vector<uint8_t> ctype;
    std::vector<double> y, yn;         // SoA [S][nc], two copies (Jacobi style, never in place)
    std::vector<double> tact;
    Stim stim[8];
    Trigger trig[4];
    int64_t step = 0;
    double dt = 0;
    // scratch
    std::vector<double> vn, D, flux;
    std::vector<Vec3> grad;
    // bidomain (eq. (1) / (6)): extra right-hand-side term div(M_int grad v_ext)/(chi C_m) per cell,
    // in mV/ms, supplied by the caller (oracle/ep_oracle_bidomain.py); empty = monodomain
    std::vector<double> dv_src;
};

const int FACE_NODES[4][3] = {{1, 2, 3}, {0, 2, 3}, {0, 1, 3}, {0, 1, 2}};  // face j is opposite vertex j

struct FaceKey { int32_t a, b, c; int64_t cell; int j; };
inline bool key_less(const FaceKey& p, const FaceKey& q) {
    if (p.a != q.a) return p.a < q.a;
    if (p.b != q.b) return p.b < q.b;
    if (p.c != q.c) return p.c < q.c;
    return p.cell < q.cell;
}

int build(Sim& s, const double* fibre, const double* scale, double sl, double st) {
    const int64_t nc = s.nc, nn = s.nn;
    s.xc.resize(nc); s.vol.resize(nc); s.sf.resize(nc * 4); s.Mc.resize(nc);
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t* t = &s.tet[c * 4];
        for (int k = 0; k < 4; ++k) if (t[k] < 0 || t[k] >= nn) return -2;
        const Vec3 p0 = s.x[t[0]], p1 = s.x[t[1]], p2 = s.x[t[2]], p3 = s.x[t[3]];
        s.xc[c] = 0.25 * (p0 + p1 + p2 + p3);
        s.vol[c] = std::fabs(dot(cross(p1 - p0, p2 - p0), p3 - p0)) / 6.0;
        if (!(s.vol[c] > 0.0)) return -2;
        for (int j = 0; j < 4; ++j) {
            const Vec3 a = s.x[t[FACE_NODES[j][0]]], b = s.x[t[FACE_NODES[j][1]]], cc = s.x[t[FACE_NODES[j][2]]];
            Vec3 sv = 0.5 * cross(b - a, cc - a);
            const Vec3 xf = (1.0 / 3.0) * (a + b + cc);
            if (dot(sv, xf - s.xc[c]) < 0.0) sv = -1.0 * sv;   // outward of c
            s.sf[c * 4 + j] = sv;
        }
        // M_c = scale * [sigma_t I + (sigma_l - sigma_t) f f^T]   (eq. (2)-(3), reading A9)
        double fx = 0, fy = 0, fz = 0, sc = scale ? scale[c] : 1.0;
        double slc = sl, stc = st;
        if (fibre) {
            fx = fibre[c * 3]; fy = fibre[c * 3 + 1]; fz = fibre[c * 3 + 2];
            const double n = std::sqrt(fx * fx + fy * fy + fz * fz);
            if (!(n > 0.0)) return -2;
            fx /= n; fy /= n; fz /= n;
        } else { stc = sl; }   // isotropic sigma_l
        const double dl = slc - stc;
        s.Mc[c] = {sc * (stc + dl * fx * fx), sc * (dl * fx * fy), sc * (dl * fx * fz),
                   sc * (stc + dl * fy * fy), sc * (dl * fy * fz), sc * (stc + dl * fz * fz)};
    }
    // faces matched by sorted node triple
    std::vector<FaceKey> keys(nc * 4);
    for (int64_t c = 0; c < nc; ++c)
        for (int j = 0; j < 4; ++j) {
            int32_t n3[3] = {s.tet[c * 4 + FACE_NODES[j][0]], s.tet[c * 4 + FACE_NODES[j][1]], s.tet[c * 4 + FACE_NODES[j][2]]};
            std::sort(n3, n3 + 3);
            keys[c * 4 + j] = {n3[0], n3[1], n3[2], c, j};
        }
    std::sort(keys.begin(), keys.end(), key_less);
    s.cell_face.assign(nc * 4, -1);
    s.faces.clear();
    for (size_t i = 0; i < keys.size();) {
        size_t k = i + 1;
        while (k < keys.size() && keys[k].a == keys[i].a && keys[k].b == keys[i].b && keys[k].c == keys[i].c) ++k;
        if (k - i > 2) return -2;
        if (k - i == 2) {
            const FaceKey& p = keys[i]; const FaceKey& q = keys[i + 1];   // p.cell < q.cell by the sort
            Face f;
            f.c1 = p.cell; f.c2 = q.cell;
            f.s = s.sf[p.cell * 4 + p.j];
            const int32_t* t = &s.tet[p.cell * 4];
            const Vec3 xf = (1.0 / 3.0) * (s.x[t[FACE_NODES[p.j][0]]] + s.x[t[FACE_NODES[p.j][1]]] + s.x[t[FACE_NODES[p.j][2]]]);
            const double d1 = norm(xf - s.xc[f.c1]), d2 = norm(xf - s.xc[f.c2]);
            f.a1 = d2 / (d1 + d2); f.a2 = 1.0 - f.a1;
            const Vec3 dc = s.xc[f.c1] - s.xc[f.c2];
            f.d = norm(dc); f.e = (1.0 / f.d) * dc;
            const Sym3& A = s.Mc[f.c1]; const Sym3& B = s.Mc[f.c2];
            f.Mf = {f.a1 * A.xx + f.a2 * B.xx, f.a1 * A.xy + f.a2 * B.xy, f.a1 * A.xz + f.a2 * B.xz,
                    f.a1 * A.yy + f.a2 * B.yy, f.a1 * A.yz + f.a2 * B.yz, f.a1 * A.zz + f.a2 * B.zz};
            const int64_t id = (int64_t)s.faces.size();
            s.faces.push_back(f);
            s.cell_face[p.cell * 4 + p.j] = id;
            s.cell_face[q.cell * 4 + q.j] = id;
        }
        i = k;
    }
    // node stars, ascending cell id (counting sort over cells in order)
    s.star_ptr.assign(nn + 1, 0);
    for (int64_t c = 0; c < nc; ++c) for (int k = 0; k < 4; ++k) s.star_ptr[s.tet[c * 4 + k] + 1]++;
    for (int64_t n = 0; n < nn; ++n) s.star_ptr[n + 1] += s.star_ptr[n];
    s.star_cell.resize(nc * 4); s.star_invd.resize(nc * 4);
    std::vector<int64_t> fill(s.star_ptr.begin(), s.star_ptr.end() - 1);
    for (int64_t c = 0; c < nc; ++c)
        for (int k = 0; k < 4; ++k) {
            const int32_t n = s.tet[c * 4 + k];
            const int64_t p = fill[n]++;
            s.star_cell[p] = c;
            s.star_invd[p] = 1.0 / norm(s.x[n] - s.xc[c]);
        }
    s.vn.resize(nn); s.D.resize(nc); s.grad.resize(nc); s.flux.resize(s.faces.size());
    return 0;
}

// (a)->(b): v_n = sum_k v_k/d_k / sum_k 1/d_k (boundary nodes one-sided, reading A3)
void node_values(const Sim& s, const double* v, double* vn) {
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < s.nn; ++n) {
        double num = 0.0, den = 0.0;
        for (int64_t p = s.star_ptr[n]; p < s.star_ptr[n + 1]; ++p) {
            num += v[s.star_cell[p]] * s.star_invd[p];
            den += s.star_invd[p];
        }
        vn[n] = (s.star_ptr[n + 1] > s.star_ptr[n]) ? num / den : 0.0;
    }
}

// (b)->(c)->(d): v_f = mean of 3 nodes; grad v_c = (1/V_c) sum_j v_fj S_fj n_fj (reading A4)
void cell_gradients(const Sim& s, const double* vn, Vec3* grad) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < s.nc; ++c) {
        const int32_t* t = &s.tet[c * 4];
        Vec3 g = {0, 0, 0};
        for (int j = 0; j < 4; ++j) {
            const double vf = (vn[t[FACE_NODES[j][0]]] + vn[t[FACE_NODES[j][1]]] + vn[t[FACE_NODES[j][2]]]) / 3.0;
            g = g + vf * s.sf[c * 4 + j];
        }
        grad[c] = (1.0 / s.vol[c]) * g;
    }
}

// (e) + eq. (8) + flux (eq. (7) :160). use_corr=0 drops the eq. (8) correction (test hook only).
void face_fluxes(const Sim& s, const double* v, const Vec3* grad, double* flux, int use_corr) {
    const int64_t nf = (int64_t)s.faces.size();
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nf; ++i) {
        const Face& f = s.faces[i];
        const Vec3 gbar = f.a1 * grad[f.c1] + f.a2 * grad[f.c2];
        Vec3 g = gbar;
        if (use_corr) g = gbar + ((v[f.c1] - v[f.c2]) / f.d - dot(gbar, f.e)) * f.e;
        flux[i] = dot(mul(f.Mf, g), f.s);
    }
}

// D_c = (1/V_c) sum_j F_fj in uA/cm^3 (lengths in mm, sigma in mS/cm: factor 100 per 1/mm^2; reading A14)
void divergence(const Sim& s, const double* flux, double* D) {
#pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < s.nc; ++c) {
        double acc = 0.0;
        for (int j = 0; j < 4; ++j) {
            const int64_t id = s.cell_face[c * 4 + j];
            if (id < 0) continue;                                  // no-flux boundary
            acc += (s.faces[id].c1 == c) ? flux[id] : -flux[id];
        }
        D[c] = 100.0 * acc / s.vol[c];
    }
}

void apply_diffusion(Sim& s, const double* v, double* D, int use_corr) {
    node_values(s, v, s.vn.data());
    cell_gradients(s, s.vn.data(), s.grad.data());
    face_fluxes(s, v, s.grad.data(), s.flux.data(), use_corr);
    divergence(s, s.flux.data(), D);
}

inline int64_t step_index(double t, double dt) { return (int64_t)std::ceil(t / dt - 1e-9); }   // reading A16

}  // namespace

// ---------------------------------------------------------------------------------------------------------
// C interface used by oracle/ep_oracle.py (ctypes). All pointers are host pointers.
extern "C" {

void* orc_create(int64_t n_nodes, const double* xyz, int64_t n_tets, const int32_t* tets, const double* fibre,
                 const double* sigma_scale, double sigma_l, double sigma_t, double chi, double Cm) {
    Sim* s = new Sim();
    s->nn = n_nodes; s->nc = n_tets; s->chi = chi; s->Cm = Cm;
    s->x.resize(n_nodes);
    for (int64_t n = 0; n < n_nodes; ++n) s->x[n] = {xyz[3 * n], xyz[3 * n + 1], xyz[3 * n + 2]};
    s->tet.assign(tets, tets + 4 * n_tets);
    for (int k = 0; k < 8; ++k) s->stim[k].set = false;
    if (build(*s, fibre, sigma_scale, sigma_l, sigma_t) != 0) { delete s; return nullptr; }
    return s;
}

void orc_destroy(void* h) { delete (Sim*)h; }

void orc_set_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n > 0 ? n : 1);
#else
    (void)n;
#endif
}

int orc_get_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int64_t orc_n_faces(void* h) { return (int64_t)((Sim*)h)->faces.size(); }

void orc_geometry(void* h, double* vol, double* centroids) {
    Sim& s = *(Sim*)h;
    for (int64_t c = 0; c < s.nc; ++c) {
        if (vol) vol[c] = s.vol[c];
        if (centroids) { centroids[3 * c] = s.xc[c].x; centroids[3 * c + 1] = s.xc[c].y; centroids[3 * c + 2] = s.xc[c].z; }
    }
}

// Pieces of the Fig. 8 pipeline, exposed so that tests can pin each one separately.
void orc_node_values(void* h, const double* v, double* vn) { node_values(*(Sim*)h, v, vn); }

void orc_cell_gradients(void* h, const double* v, double* grad /*[nc*3]*/) {
    Sim& s = *(Sim*)h;
    node_values(s, v, s.vn.data());
    cell_gradients(s, s.vn.data(), s.grad.data());
    for (int64_t c = 0; c < s.nc; ++c) { grad[3 * c] = s.grad[c].x; grad[3 * c + 1] = s.grad[c].y; grad[3 * c + 2] = s.grad[c].z; }
}

// D = div(M grad v) in uA/cm^3 for a cell field v [mV]; use_corr=0 drops eq. (8) (test hook).
void orc_apply_diffusion(void* h, const double* v, double* D, int use_corr) { apply_diffusion(*(Sim*)h, v, D, use_corr); }

int orc_state_init(void* h, int model, const uint8_t* cell_type, const double* y0) {
    Sim& s = *(Sim*)h;
    if (model != 0 && model != 1) return -3;
    s.model = model; s.S = (model == 0) ? TP06_S : crn::S;
    const double* rest = (model == 0) ? TP06_REST : crn::REST;
    s.ctype.assign(s.nc, 0);
    if (cell_type) s.ctype.assign(cell_type, cell_type + s.nc);
    s.y.resize((size_t)s.S * s.nc); s.yn.resize((size_t)s.S * s.nc);
    for (int64_t c = 0; c < s.nc; ++c) {
        const double* src = y0 ? y0 + (size_t)s.ctype[c] * s.S : rest;
        for (int k = 0; k < s.S; ++k) s.y[(size_t)k * s.nc + c] = src[k];
    }
    s.tact.assign(s.nc, -1.0);
    for (int t = 0; t < 4; ++t) s.trig[t].n_fire1 = -1;
    s.step = 0; s.dt = 0;
    return 0;
}

int orc_stimulus_set(void* h, int slot, int64_t n, const int64_t* ids, double amp, double t0, double dur) {
    Sim& s = *(Sim*)h;
    if (slot < 0 || slot >= 8) return -1;
    Stim& st = s.stim[slot];
    st.mask.assign(s.nc, 0);
    for (int64_t i = 0; i < n; ++i) { if (ids[i] < 0 || ids[i] >= s.nc) return -1; st.mask[ids[i]] = 1; }
    st.amp = amp; st.t0 = t0; st.dur = dur; st.set = (n > 0);
    return 0;
}

int orc_trigger_set(void* h, int trig, int64_t n, const int64_t* ids, int slot, double delay) {
    Sim& s = *(Sim*)h;
    if (trig < 0 || trig >= 4 || slot < 0 || slot >= 8) return -1;
    Trigger& g = s.trig[trig];
    g.cells.assign(ids, ids + n);
    for (int64_t c : g.cells) if (c < 0 || c >= s.nc) return -1;
    g.slot = slot; g.delay = delay; g.armed = n > 0; g.n_fire1 = -1;
    return 0;
}

double orc_trigger_time(void* h, int trig) {
    Sim& s = *(Sim*)h;
    return s.trig[trig].n_fire1 < 0 ? -1.0 : (double)s.trig[trig].n_fire1 * s.dt;
}

int orc_step(void* h, int64_t n_steps, double dt) {
    Sim& s = *(Sim*)h;
    if (s.model < 0 || !(dt > 0)) return -3;
    s.dt = dt;
    const int64_t nc = s.nc;
    const double inv_chiCm = 1.0 / (s.chi * s.Cm);
    for (int64_t it = 0; it < n_steps; ++it) {
        const int64_t n = s.step;
        apply_diffusion(s, s.y.data(), s.D.data(), 1);   // state 0 is v
        bool on[8];
        for (int k = 0; k < 8; ++k) {
            on[k] = false;
            if (!s.stim[k].set) continue;
            const int64_t n_on = step_index(s.stim[k].t0, dt), n_off = step_index(s.stim[k].t0 + s.stim[k].dur, dt);
            on[k] = (n_on <= n && n < n_off);
        }
        for (int t = 0; t < 4; ++t) {   // a slot driven by a trigger ignores its own window
            const Trigger& g = s.trig[t];
            if (!g.armed) continue;
            const int64_t nd = step_index(g.delay, dt), ndur = step_index(s.stim[g.slot].dur, dt);
            on[g.slot] = s.stim[g.slot].set && g.n_fire1 >= 0 && n >= g.n_fire1 + nd && n < g.n_fire1 + nd + ndur;
        }
#pragma omp parallel for schedule(static)
        for (int64_t c = 0; c < nc; ++c) {
            double y[32], yn[32];
            for (int k = 0; k < s.S; ++k) y[k] = s.y[(size_t)k * nc + c];
            double Is = 0.0;   // uA/cm^2, eq. (4)
            for (int k = 0; k < 8; ++k) if (on[k] && s.stim[k].mask[c]) Is += s.stim[k].amp;
            const double dvd = s.D[c] * inv_chiCm + (s.dv_src.empty() ? 0.0 : s.dv_src[c]);
            if (s.model == 0) tp06_step(y, s.ctype[c], dt, Is / s.Cm, dvd, yn);
            else crn::step(y, dt, Is / s.Cm, dvd, yn);
            for (int k = 0; k < s.S; ++k) s.yn[(size_t)k * nc + c] = yn[k];
            if (s.tact[c] < 0.0 && y[0] <= 0.0 && yn[0] > 0.0) s.tact[c] = (double)(n + 1) * dt;   // A18
        }
        for (int t = 0; t < 4; ++t) {   // a monitored cell exceeding 0 mV fires the trigger, once
            Trigger& g = s.trig[t];
            if (!g.armed || g.n_fire1 >= 0) continue;
            for (int64_t c : g.cells)
                if (s.y[c] <= 0.0 && s.yn[c] > 0.0) { g.n_fire1 = n + 1; break; }
        }
        s.y.swap(s.yn);
        s.step = n + 1;
    }
    return 0;
}

// bidomain coupling term for the following steps: src [nc] in mV/ms, or NULL to remove it
void orc_set_source(void* h, const double* src) {
    Sim& s = *(Sim*)h;
    if (src) s.dv_src.assign(src, src + s.nc); else s.dv_src.clear();
}

int orc_n_states(void* h) { return ((Sim*)h)->S; }
int64_t orc_step_count(void* h) { return ((Sim*)h)->step; }
void orc_get_state(void* h, int var, double* out) { Sim& s = *(Sim*)h; std::memcpy(out, &s.y[(size_t)var * s.nc], sizeof(double) * s.nc); }
void orc_set_state(void* h, int var, const double* in) { Sim& s = *(Sim*)h; std::memcpy(&s.y[(size_t)var * s.nc], in, sizeof(double) * s.nc); }
void orc_activation_times(void* h, double* out) { Sim& s = *(Sim*)h; std::memcpy(out, s.tact.data(), sizeof(double) * s.nc); }

// volume-averaged potential: sum_c V_c v_c / sum_c V_c, cells in ascending order
double orc_mean_vm(void* h) {
    Sim& s = *(Sim*)h;
    double num = 0.0, den = 0.0;
    for (int64_t c = 0; c < s.nc; ++c) { num += s.vol[c] * s.y[c]; den += s.vol[c]; }
    return num / den;
}

// ---- single-cell entry points (pins P8-P10)
void orc_tp06_rest(double* y) { std::memcpy(y, TP06_REST, sizeof(TP06_REST)); }
void orc_tp06_gates(double v, int type, double Ca_SS, double Ca_SR, double* inf, double* tau) { tp06_gates(v, type, Ca_SS, Ca_SR, inf, tau); }
void orc_tp06_currents(const double* y, int type, double* out17) {
    Tp06Currents c; tp06_currents(y, type, c);
    const double a[17] = {c.INa, c.ICaL, c.Ito, c.IKr, c.IKs, c.IK1, c.INaCa, c.INaK, c.IpCa, c.IpK, c.IbNa, c.IbCa,
                          c.iion, c.Irel, c.Ileak, c.Iup, c.Ixfer};
    std::memcpy(out17, a, sizeof(a));
}
// n_steps single-cell steps; stimulus istim (uA/uF) while n_on <= n < n_off; optional v trace [n_steps+1].
// freeze_v != 0 holds v at its initial value (used by the RL closed-form pin).
void orc_tp06_run(double* y, int type, double dt, int64_t n_steps, double istim, int64_t n_on, int64_t n_off,
                  double* vtrace, int freeze_v) {
    double yn[TP06_S];
    if (vtrace) vtrace[0] = y[0];
    for (int64_t n = 0; n < n_steps; ++n) {
        const double is = (n_on <= n && n < n_off) ? istim : 0.0;
        tp06_step(y, type, dt, is, 0.0, yn);
        if (freeze_v) yn[0] = y[0];
        std::memcpy(y, yn, sizeof(yn));
        if (vtrace) vtrace[n + 1] = y[0];
    }
}

// ---- Courtemanche single-cell entry points (pins P8, P12)
void orc_crn_rest(double* y) { std::memcpy(y, crn::REST, sizeof(crn::REST)); }
void orc_crn_gates(double V, double Cai, double Fn, double* inf, double* tau) { crn::gates(V, Cai, Fn, inf, tau); }
void orc_crn_currents(const double* y, double* out18) {
    crn::Currents c; crn::currents(y, c);
    const double a[18] = {c.INa, c.IK1, c.Ito, c.IKur, c.IKr, c.IKs, c.ICaL, c.IpCa, c.INaK, c.INaCa, c.IbNa, c.IbCa, c.iion,
                          c.Irel, c.Itr, c.Iup, c.Iupleak, c.Fn};
    std::memcpy(out18, a, sizeof(a));
}
void orc_crn_run(double* y, double dt, int64_t n_steps, double istim, int64_t n_on, int64_t n_off, double* vtrace,
                 int freeze_v) {
    double yn[crn::S];
    if (vtrace) vtrace[0] = y[0];
    for (int64_t n = 0; n < n_steps; ++n) {
        const double is = (n_on <= n && n < n_off) ? istim : 0.0;
        crn::step(y, dt, is, 0.0, yn);
        if (freeze_v) yn[0] = y[0];
        std::memcpy(y, yn, sizeof(yn));
        if (vtrace) vtrace[n + 1] = y[0];
    }
}

}  // extern "C"
