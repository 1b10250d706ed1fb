// ep_tp06.cuh -- ten Tusscher-Panfilov 2006 ventricular cell model, one explicit step of one cell (device code).
//
// PAPER.md:126, :174, :256 name the model (ref [3]: 19 states, 13 of them advanced by Rush-Larsen);
// the equations and constants are restated from the published model in DESIGN.md Appendix A.  Readings B1..B9 of
// DESIGN.md section 3 apply (13 RL variables = 12 gates + Rbar; buffer factors + forward Euler for the three calcium
// pools; v >= -40 mV takes the high-voltage h/j branch; removable singularity of I_CaL handled by a series).
// Everything on the right-hand side is taken at t^n: the function reads y[], returns the new values
// in y[] only after all right-hand sides have been formed.
//
// Units: mV, ms, mM, currents uA/uF, conductances nS/pF.
#pragma once
#include "ep_math.cuh"

namespace epk {

enum { TP06_S = 19 };
// state order at the ABI (ep_read_state var): v m h j xr1 xr2 xs r s d f f2 fCass Rbar Ca_i Ca_SR Ca_SS Na_i K_i
enum { Y_V = 0, Y_M, Y_H, Y_J, Y_XR1, Y_XR2, Y_XS, Y_R, Y_S, Y_D, Y_F, Y_F2, Y_FCASS, Y_RBAR, Y_CAI, Y_CASR, Y_CASS,
       Y_NAI, Y_KI };

__device__ __constant__ const double TP06_REST_STATE[TP06_S] = {
    -86.2, 0.0, 0.75, 0.75, 0.0, 1.0, 0.0, 0.0, 1.0, 0.0, 1.0, 1.0, 1.0, 1.0, 7e-5, 1.3, 7e-5, 7.67, 138.3};

namespace tp06 {
// physical constants
constexpr double R = 8314.472, T = 310.0, F = 96485.3415;
constexpr double RTF = R * T / F;          // mV
constexpr double FRT = F / (R * T);        // 1/mV
constexpr double Ko = 5.4, Cao = 2.0, Nao = 140.0;
constexpr double Vc = 0.016404, Vsr = 0.001094, Vss = 0.00005468, Cap = 0.185;
constexpr double GNa = 14.838, GK1 = 5.405, GKr = 0.153, GCaL = 3.980e-5, GbNa = 2.9e-4, GbCa = 5.92e-4;
constexpr double GpCa = 0.1238, KpCa = 5e-4, GpK = 0.0146, pKNa = 0.03;
constexpr double PNaK = 2.724, KmK = 1.0, KmNa = 40.0;
constexpr double kNaCa = 1000.0, KmNai = 87.5, KmCa = 1.38, ksat = 0.1, gam = 0.35, alpha = 2.5;
constexpr double Vmaxup = 0.006375, Kup = 2.5e-4, Vrel = 0.102, k1p = 0.15, k2p = 0.045, k3 = 0.060, k4 = 0.005;
constexpr double EC = 1.5, maxsr = 2.5, minsr = 1.0, Vleak = 3.6e-4, Vxfer = 0.0038;
constexpr double Bufc = 0.2, Kbufc = 0.001, Bufsr = 10.0, Kbufsr = 0.3, Bufss = 0.4, Kbufss = 2.5e-4;
}  // namespace tp06

// Rush-Larsen update y <- yinf + (y - yinf) exp(-dt/tau).  rate = 1/tau.
__device__ __forceinline__ double rl(double y, double yinf, double rate, double dt) {
    return fma(y - yinf, ep_exp(-dt * rate), yinf);
}

// sigma(z) = 1/(1+e^z)
__device__ __forceinline__ double sg(double z) { return ep_rcp(1.0 + ep_exp(z)); }

// One step. type: 0 endo, 1 mid, 2 epi.  istim = I_s/C_m [uA/uF], dv_diff = D_c/(chi C_m) [mV/ms].
__device__ __forceinline__ void tp06_step(double (&y)[TP06_S], int type, double dt, double istim, double dv_diff) {
    using namespace tp06;
    const double v = y[Y_V];
    const double Cai = y[Y_CAI], CaSR = y[Y_CASR], CaSS = y[Y_CASS], Nai = y[Y_NAI], Ki = y[Y_KI];

    // ---- reversal potentials
    const double EK = RTF * ep_log(ep_div(Ko, Ki));
    const double ENa = RTF * ep_log(ep_div(Nao, Nai));
    const double EKs = RTF * ep_log(ep_div(Ko + pKNa * Nao, Ki + pKNa * Nai));
    const double ECa = 0.5 * RTF * ep_log(ep_div(Cao, Cai));

    // ---- membrane currents
    const double m = y[Y_M];
    const double INa = GNa * m * m * m * y[Y_H] * y[Y_J] * (v - ENa);
    double ICaL;
    {
        const double x = 2.0 * (v - 15.0) * FRT;
        const double ex = ep_exp(x);
        // x/(e^x - 1), with the series 1 - x/2 inside |x| < 1e-7 (reading B6)
        const double xo = (fabs(x) < 1e-7) ? fma(-0.5, x, 1.0) : ep_div(x, ex - 1.0);
        ICaL = GCaL * y[Y_D] * y[Y_F] * y[Y_F2] * y[Y_FCASS] * 2.0 * F * xo * (0.25 * CaSS * ex - Cao);
    }
    const double Gto = (type == 0) ? 0.073 : 0.294;
    const double GKs = (type == 1) ? 0.098 : 0.392;
    const double Ito = Gto * y[Y_R] * y[Y_S] * (v - EK);
    const double IKr = GKr * ep_sqrt(Ko / 5.4) * y[Y_XR1] * y[Y_XR2] * (v - EK);
    const double IKs = GKs * y[Y_XS] * y[Y_XS] * (v - EKs);
    double IK1;
    {
        const double u = v - EK;
        const double aK1 = ep_div(0.1, 1.0 + ep_exp(0.06 * (u - 200.0)));
        const double bK1 = ep_div(3.0 * ep_exp(0.0002 * (u + 100.0)) + ep_exp(0.1 * (u - 10.0)), 1.0 + ep_exp(-0.5 * u));
        IK1 = GK1 * ep_div(aK1, aK1 + bK1) * u;
    }
    double INaCa;
    {
        const double e1 = ep_exp(gam * v * FRT), e2 = ep_exp((gam - 1.0) * v * FRT);
        const double num = e1 * Nai * Nai * Nai * Cao - e2 * Nao * Nao * Nao * Cai * alpha;
        const double den = (KmNai * KmNai * KmNai + Nao * Nao * Nao) * (KmCa + Cao) * (1.0 + ksat * e2);
        INaCa = kNaCa * ep_div(num, den);
    }
    const double INaK = PNaK * (Ko / (Ko + KmK)) * ep_div(Nai, Nai + KmNa)
                        * ep_rcp(1.0 + 0.1245 * ep_exp(-0.1 * v * FRT) + 0.0353 * ep_exp(-v * FRT));
    const double IpCa = GpCa * ep_div(Cai, KpCa + Cai);
    const double IpK = GpK * (v - EK) * sg((25.0 - v) / 5.98);
    const double IbNa = GbNa * (v - ENa);
    const double IbCa = GbCa * (v - ECa);
    const double iion = INa + ICaL + Ito + IKr + IKs + IK1 + INaCa + INaK + IpCa + IpK + IbNa + IbCa;

    // ---- sarcoplasmic-reticulum fluxes
    const double ecs = ep_div(EC, CaSR);
    const double kcasr = maxsr - ep_div(maxsr - minsr, 1.0 + ecs * ecs);
    const double k1 = ep_div(k1p, kcasr), k2 = k2p * kcasr;
    const double css2 = CaSS * CaSS;
    const double O = ep_div(k1 * css2 * y[Y_RBAR], k3 + k1 * css2);
    const double Irel = Vrel * O * (CaSR - CaSS);
    const double Ileak = Vleak * (CaSR - Cai);
    const double Iup = ep_div(Vmaxup, 1.0 + ep_div(Kup * Kup, Cai * Cai));
    const double Ixfer = Vxfer * (CaSS - Cai);

    // ---- concentrations: buffer factors (reading B3) and forward Euler
    const double bi = ep_rcp(1.0 + ep_div(Bufc * Kbufc, (Cai + Kbufc) * (Cai + Kbufc)));
    const double bsr = ep_rcp(1.0 + ep_div(Bufsr * Kbufsr, (CaSR + Kbufsr) * (CaSR + Kbufsr)));
    const double bss = ep_rcp(1.0 + ep_div(Bufss * Kbufss, (CaSS + Kbufss) * (CaSS + Kbufss)));
    const double dCai = bi * ((Ileak - Iup) * (Vsr / Vc) + Ixfer - (IbCa + IpCa - 2.0 * INaCa) * (Cap / (2.0 * Vc * F)));
    const double dCaSR = bsr * (Iup - Ileak - Irel);
    const double dCaSS = bss * (-ICaL * (Cap / (2.0 * Vss * F)) + Irel * (Vsr / Vss) - Ixfer * (Vc / Vss));
    const double dNai = -(INa + IbNa + 3.0 * INaK + 3.0 * INaCa) * (Cap / (Vc * F));
    const double dKi = -(IK1 + Ito + IKr + IKs - 2.0 * INaK + IpK + istim) * (Cap / (Vc * F));   // reading B8

    // ---- gates: steady states and rates (1/tau), Rush-Larsen
    {   // m
        const double s = sg((-56.86 - v) / 9.03);
        const double tau = sg((-60.0 - v) / 5.0) * (0.1 * sg((v + 35.0) / 5.0) + 0.1 * sg((v - 50.0) / 200.0));
        y[Y_M] = rl(y[Y_M], s * s, ep_rcp(tau), dt);
    }
    {   // h, j share the steady state; rates alpha+beta are used directly (tau = 1/(alpha+beta))
        const double s = sg((v + 71.55) / 7.43);
        const double hinf = s * s;
        double rh, rj;
        if (v >= -40.0) {   // reading B7
            rh = ep_div(0.77, 0.13 * (1.0 + ep_exp(-(v + 10.66) / 11.1)));
            rj = ep_div(0.6 * ep_exp(0.057 * v), 1.0 + ep_exp(-0.1 * (v + 32.0)));
        } else {
            rh = 0.057 * ep_exp(-(v + 80.0) / 6.8) + 2.7 * ep_exp(0.079 * v) + 3.1e5 * ep_exp(0.3485 * v);
            const double aj = ep_div((-2.5428e4 * ep_exp(0.2444 * v) - 6.948e-6 * ep_exp(-0.04391 * v)) * (v + 37.78),
                                     1.0 + ep_exp(0.311 * (v + 79.23)));
            const double bj = ep_div(0.02424 * ep_exp(-0.01052 * v), 1.0 + ep_exp(-0.1378 * (v + 40.14)));
            rj = aj + bj;
        }
        y[Y_H] = rl(y[Y_H], hinf, rh, dt);
        y[Y_J] = rl(y[Y_J], hinf, rj, dt);
    }
    {   // xr1, xr2, xs
        const double t1 = 450.0 * sg((-45.0 - v) / 10.0) * 6.0 * sg((v + 30.0) / 11.5);
        y[Y_XR1] = rl(y[Y_XR1], sg((-26.0 - v) / 7.0), ep_rcp(t1), dt);
        const double t2 = 3.0 * sg((-60.0 - v) / 20.0) * 1.12 * sg((v - 60.0) / 20.0);
        y[Y_XR2] = rl(y[Y_XR2], sg((v + 88.0) / 24.0), ep_rcp(t2), dt);
        const double t3 = ep_div(1400.0, ep_sqrt(1.0 + ep_exp((5.0 - v) / 6.0))) * sg((v - 35.0) / 15.0) + 80.0;
        y[Y_XS] = rl(y[Y_XS], sg((-5.0 - v) / 14.0), ep_rcp(t3), dt);
    }
    {   // r, s (reading B5: endo has its own s curves)
        const double tr = 9.5 * ep_exp(-(v + 40.0) * (v + 40.0) / 1800.0) + 0.8;
        y[Y_R] = rl(y[Y_R], sg((20.0 - v) / 6.0), ep_rcp(tr), dt);
        double sinf, ts;
        if (type == 0) {
            sinf = sg((v + 28.0) / 5.0);
            ts = 1000.0 * ep_exp(-(v + 67.0) * (v + 67.0) / 1000.0) + 8.0;
        } else {
            sinf = sg((v + 20.0) / 5.0);
            ts = 85.0 * ep_exp(-(v + 45.0) * (v + 45.0) / 320.0) + 5.0 * sg((v - 20.0) / 5.0) + 3.0;
        }
        y[Y_S] = rl(y[Y_S], sinf, ep_rcp(ts), dt);
    }
    {   // d, f, f2
        const double td = (1.4 * sg((-35.0 - v) / 13.0) + 0.25) * (1.4 * sg((v + 5.0) / 5.0)) + sg((50.0 - v) / 20.0);
        y[Y_D] = rl(y[Y_D], sg((-8.0 - v) / 7.5), ep_rcp(td), dt);
        const double g27 = (v + 27.0) * (v + 27.0);
        const double tf = 1102.5 * ep_exp(-g27 / 225.0) + 200.0 * sg((13.0 - v) / 10.0) + 180.0 * sg((v + 30.0) / 10.0) + 20.0;
        y[Y_F] = rl(y[Y_F], sg((v + 20.0) / 7.0), ep_rcp(tf), dt);
        const double tf2 = 562.0 * ep_exp(-g27 / 240.0) + 31.0 * sg((25.0 - v) / 10.0) + 80.0 * sg((v + 30.0) / 10.0);
        y[Y_F2] = rl(y[Y_F2], 0.67 * sg((v + 35.0) / 7.0) + 0.33, ep_rcp(tf2), dt);
    }
    {   // fCass
        const double q = ep_rcp(1.0 + (CaSS / 0.05) * (CaSS / 0.05));
        y[Y_FCASS] = rl(y[Y_FCASS], 0.6 * q + 0.4, ep_rcp(80.0 * q + 2.0), dt);
    }
    {   // Rbar: dR/dt = k4 (1 - R) - k2 CaSS R, linear in R at frozen Ca (reading B1)
        const double rate = k2 * CaSS + k4;
        y[Y_RBAR] = rl(y[Y_RBAR], ep_div(k4, rate), rate, dt);
    }
    y[Y_CAI] = fma(dt, dCai, Cai);
    y[Y_CASR] = fma(dt, dCaSR, CaSR);
    y[Y_CASS] = fma(dt, dCaSS, CaSS);
    y[Y_NAI] = fma(dt, dNai, Nai);
    y[Y_KI] = fma(dt, dKi, Ki);
    y[Y_V] = fma(dt, dv_diff - iion - istim, v);   // eq. (7); explicit increment PAPER.md:172
}

}  // namespace epk
