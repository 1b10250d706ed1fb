"""Hand-computed values of every TP06 time constant, conductance and flux constant (DESIGN.md Appendix A = SURVEY.md
Appendix A, the published model, PAPER.md:354 ref [3]).

Each expected value is written out for ONE argument chosen so that most of the expression collapses (a sigmoid at its
centre is 1/2, a Gaussian at its centre is 1, a Nernst potential with equal concentrations is 0, a saturating flux at
its half-saturation concentration is half its maximum) and only one or two literal exponentials remain; the number in
the comment is that expression evaluated by hand.  None of them calls or re-types the oracle's general formula, and a
change of any single constant of the model moves at least one of them (tests/test_oracle_mutations.py checks exactly
that).  Gate index g = state index - 1: 0 m, 1 h, 2 j, 3 xr1, 4 xr2, 5 xs, 6 r, 7 s, 8 d, 9 f, 10 f2, 11 fCass, 12 Rbar.
"""
import math

import numpy as np
import pytest

E = math.exp
RTF = 8314.472 * 310.0 / 96485.3415          # 26.7138 mV
IDX = dict(v=0, m=1, h=2, j=3, xr1=4, xr2=5, xs=6, r=7, s=8, d=9, f=10, f2=11, fcass=12, R=13, Cai=14, CaSR=15, CaSS=16,
           Nai=17, Ki=18)


def _tau(oracle, v, g, typ=0, **kw):
    return oracle.tp06_gates(v, typ, **kw)[1][g]


def _inf(oracle, v, g, typ=0, **kw):
    return oracle.tp06_gates(v, typ, **kw)[0][g]


def test_rtf_value():
    assert RTF == pytest.approx(26.713760659695648, rel=1e-15)


def test_tau_m_special_voltages(oracle):
    """tau_m = s(-60-v;5) [0.1 s(v+35;5) + 0.1 s(v-50;200)], s(z;k) = 1/(1+e^{z/k}).
    v=-60: first factor 1/2, then 0.1/(1+e^-5) + 0.1/(1+e^-0.55)           -> 0.08137213700432580
    v=-35: 1/(1+e^-5) * [0.05 + 0.1/(1+e^-0.425)]                          -> 0.10972856322808432
    v=+50: 1/(1+e^-22) * [0.1/(1+e^17) + 0.05]                             -> 0.05000000412599021"""
    assert _tau(oracle, -60.0, 0) == pytest.approx(0.5 * (0.1 / (1 + E(-5.0)) + 0.1 / (1 + E(-0.55))), rel=1e-14)
    assert _tau(oracle, -60.0, 0) == pytest.approx(0.0813721370043258, rel=1e-13)
    assert _tau(oracle, -35.0, 0) == pytest.approx(0.10972856322808432, rel=1e-13)
    assert _tau(oracle, 50.0, 0) == pytest.approx(0.050000004125990205, rel=1e-13)


def test_tau_h_tau_j_special_voltages(oracle):
    """Low branch (v < -40): alpha_h = 0.057 e^{-(v+80)/6.8}, beta_h = 2.7 e^{0.079 v} + 3.1e5 e^{0.3485 v}.
    v=-80: alpha_h = 0.057 exactly, beta_h = 2.7 e^-6.32 + 3.1e5 e^-27.88  -> tau_h = 16.165511784327766
    alpha_j = (-2.5428e4 e^{0.2444 v} - 6.948e-6 e^{-0.04391 v})(v+37.78)/(1+e^{0.311(v+79.23)}),
    beta_j = 0.02424 e^{-0.01052 v}/(1+e^{-0.1378(v+40.14)}).
    v=-79.23: the alpha_j denominator is exactly 2                          -> tau_j = 143.35402707629598
    v=-100:                                                                 -> tau_j = 28.654847385414854
    High branch (v >= -40): tau_h = 0.13 (1+e^{-(v+10.66)/11.1})/0.77; v=-10.66 -> 0.26/0.77
    tau_j = (1+e^{-0.1(v+32)})/(0.6 e^{0.057 v}); v=-32 -> 2/(0.6 e^-1.824) = 20.655317748165764; v=0 -> (1+e^-3.2)/0.6"""
    assert _tau(oracle, -80.0, 1) == pytest.approx(1.0 / (0.057 + 2.7 * E(-6.32) + 3.1e5 * E(-27.88)), rel=1e-14)
    assert _tau(oracle, -80.0, 1) == pytest.approx(16.165511784327766, rel=1e-13)
    aj = (-2.5428e4 * E(0.2444 * -79.23) - 6.948e-6 * E(0.04391 * 79.23)) * (-79.23 + 37.78) / 2.0
    bj = 0.02424 * E(0.01052 * 79.23) / (1 + E(-0.1378 * (-79.23 + 40.14)))
    assert _tau(oracle, -79.23, 2) == pytest.approx(1.0 / (aj + bj), rel=1e-13)
    assert _tau(oracle, -79.23, 2) == pytest.approx(143.35402707629598, rel=1e-12)
    assert _tau(oracle, -100.0, 2) == pytest.approx(28.654847385414854, rel=1e-12)
    assert _tau(oracle, -10.66, 1) == pytest.approx(0.26 / 0.77, rel=1e-14)
    assert _tau(oracle, -32.0, 2) == pytest.approx(2.0 / (0.6 * E(-1.824)), rel=1e-14)
    assert _tau(oracle, -32.0, 2) == pytest.approx(20.655317748165764, rel=1e-13)
    assert _tau(oracle, 0.0, 2) == pytest.approx((1 + E(-3.2)) / 0.6, rel=1e-14)


def test_tau_xr1_xr2_xs_special_voltages(oracle):
    """tau_xr1 = 450 s(-45-v;10) * 6 s(v+30;11.5): v=-45 -> 225 * 6/(1+e^{-15/11.5}) = 1061.863837646841;
                                                   v=-30 -> 450/(1+e^{-1.5}) * 3   = 1103.725542861419
    tau_xr2 = 3 s(-60-v;20) * 1.12 s(v-60;20):     v=-60 -> 1.5 * 1.12/(1+e^-6)    = 1.675845993096854 (= value at +60);
                                                   v=0   -> 3.36/((1+e^-3)^2)      = 3.048855489427512
    tau_xs = 1400/sqrt(1+e^{(5-v)/6}) * s(v-35;15) + 80: v=5 -> 1400/sqrt2/(1+e^-2) + 80 = 951.9446213624395;
                                                   v=35  -> 700/sqrt(1+e^-5) + 80  = 777.6535695078901"""
    assert _tau(oracle, -45.0, 3) == pytest.approx(225.0 * 6.0 / (1 + E(-15.0 / 11.5)), rel=1e-14)
    assert _tau(oracle, -45.0, 3) == pytest.approx(1061.863837646841, rel=1e-13)
    assert _tau(oracle, -30.0, 3) == pytest.approx(450.0 / (1 + E(-1.5)) * 3.0, rel=1e-14)
    assert _tau(oracle, -30.0, 3) == pytest.approx(1103.725542861419, rel=1e-13)
    assert _tau(oracle, -60.0, 4) == pytest.approx(1.5 * 1.12 / (1 + E(-6.0)), rel=1e-14)
    assert _tau(oracle, 60.0, 4) == pytest.approx(1.675845993096854, rel=1e-13)
    assert _tau(oracle, 0.0, 4) == pytest.approx(3.36 / (1 + E(-3.0)) ** 2, rel=1e-14)
    assert _tau(oracle, 5.0, 5) == pytest.approx(1400.0 / math.sqrt(2.0) / (1 + E(-2.0)) + 80.0, rel=1e-14)
    assert _tau(oracle, 5.0, 5) == pytest.approx(951.9446213624395, rel=1e-13)
    assert _tau(oracle, 35.0, 5) == pytest.approx(700.0 / math.sqrt(1 + E(-5.0)) + 80.0, rel=1e-14)
    assert _tau(oracle, 35.0, 5) == pytest.approx(777.6535695078901, rel=1e-13)


def test_tau_d_special_voltages(oracle):
    """tau_d = [1.4 s(-35-v;13) + 0.25][1.4 s(v+5;5)] + s(50-v;20).
    v=-35: (0.7+0.25) * 1.4/(1+e^-6) + 1/(1+e^4.25)                        -> 1.3407750382449213
    v=-5 : [1.4/(1+e^{-30/13}) + 0.25] * 0.7 + 1/(1+e^2.75)                 -> 1.1264085199429343
    v=50 : [1.4/(1+e^{-85/13}) + 0.25] * 1.4/(1+e^-11) + 1/2                -> 0.5000385329950581"""
    assert _tau(oracle, -35.0, 8) == pytest.approx(0.95 * 1.4 / (1 + E(-6.0)) + 1.0 / (1 + E(4.25)), rel=1e-14)
    assert _tau(oracle, -35.0, 8) == pytest.approx(1.3407750382449213, rel=1e-13)
    assert _tau(oracle, -5.0, 8) == pytest.approx((1.4 / (1 + E(-30.0 / 13.0)) + 0.25) * 0.7 + 1.0 / (1 + E(2.75)), rel=1e-14)
    assert _tau(oracle, -5.0, 8) == pytest.approx(1.1264085199429343, rel=1e-13)
    assert _tau(oracle, 50.0, 8) == pytest.approx(0.5000385329950581, rel=1e-13)


def test_tau_r_s_f_f2_away_from_the_gaussian_peak(oracle):
    """The Gaussian widths (1800, 1000, 320, 225, 240) are invisible at the peak; one point off the peak fixes each.
    tau_r(v=-10)  = 9.5 e^{-900/1800} + 0.8 = 9.5 e^-0.5 + 0.8
    tau_s endo(v=-37) = 1000 e^{-900/1000} + 8;  tau_s epi(v=-5) = 85 e^{-1600/320} + 5/(1+e^{-5}) + 3
    tau_f(v=-12)  = 1102.5 e^{-1} + 200/(1+e^{2.5}) + 180/(1+e^{1.8}) + 20     (225 = 15^2)
    tau_f2(v=-27+sqrt(240)) has its Gaussian at e^-1: checked at v=-12 instead: 562 e^{-225/240} + 31/(1+e^{3.7}) + 80/(1+e^{1.8})"""
    assert _tau(oracle, -10.0, 6) == pytest.approx(9.5 * E(-0.5) + 0.8, rel=1e-14)
    assert _tau(oracle, -37.0, 7, 0) == pytest.approx(1000.0 * E(-0.9) + 8.0, rel=1e-14)
    assert _tau(oracle, -5.0, 7, 2) == pytest.approx(85.0 * E(-5.0) + 5.0 / (1 + E(-5.0)) + 3.0, rel=1e-14)
    assert _tau(oracle, -5.0, 7, 1) == _tau(oracle, -5.0, 7, 2)
    assert _tau(oracle, -12.0, 9) == pytest.approx(1102.5 * E(-1.0) + 200.0 / (1 + E(2.5)) + 180.0 / (1 + E(1.8)) + 20.0,
                                                  rel=1e-14)
    assert _tau(oracle, -12.0, 10) == pytest.approx(562.0 * E(-225.0 / 240.0) + 31.0 / (1 + E(3.7)) + 80.0 / (1 + E(1.8)),
                                                   rel=1e-14)


def test_steady_state_slopes(oracle):
    """Half points are pinned in test_oracle_tp06.py; one e-fold away each sigmoid is 1/(1+e) or 1/(1+1/e), which fixes the
    slope factors 9.03, 7.43, 7, 24, 14, 6, 5, 7.5, 7, 7 and their signs."""
    lo, hi = 1.0 / (1.0 + math.e), 1.0 / (1.0 + 1.0 / math.e)     # 0.2689..., 0.7310...
    assert _inf(oracle, -56.86 + 9.03, 0) == pytest.approx(hi * hi, rel=1e-13)       # m: rises
    assert _inf(oracle, -71.55 + 7.43, 1) == pytest.approx(lo * lo, rel=1e-13)       # h: falls
    assert _inf(oracle, -71.55 - 7.43, 2) == pytest.approx(hi * hi, rel=1e-13)       # j = h
    assert _inf(oracle, -26.0 + 7.0, 3) == pytest.approx(hi, rel=1e-13)              # xr1 rises
    assert _inf(oracle, -88.0 + 24.0, 4) == pytest.approx(lo, rel=1e-13)             # xr2 falls
    assert _inf(oracle, -5.0 + 14.0, 5) == pytest.approx(hi, rel=1e-13)              # xs rises
    assert _inf(oracle, 20.0 + 6.0, 6) == pytest.approx(hi, rel=1e-13)               # r rises
    assert _inf(oracle, -28.0 + 5.0, 7, 0) == pytest.approx(lo, rel=1e-13)           # s endo falls
    assert _inf(oracle, -20.0 + 5.0, 7, 2) == pytest.approx(lo, rel=1e-13)           # s epi falls
    assert _inf(oracle, -8.0 + 7.5, 8) == pytest.approx(hi, rel=1e-13)               # d rises
    assert _inf(oracle, -20.0 + 7.0, 9) == pytest.approx(lo, rel=1e-13)              # f falls
    assert _inf(oracle, -35.0 + 7.0, 10) == pytest.approx(0.67 * lo + 0.33, rel=1e-13)   # f2 falls to 0.33


def test_fcass_and_rbar(oracle):
    """fCass: q = 1 + (Ca_SS/0.05)^2; Ca_SS = 0.1 -> q = 5: inf = 0.6/5 + 0.4 = 0.52, tau = 80/5 + 2 = 18.
    Rbar (reading B1): k_casr = max_sr - (max_sr-min_sr)/(1+(EC/Ca_SR)^2); Ca_SR = 3 (= 2 EC) -> 2.5 - 1.5/1.25 = 1.3;
    k2 = 0.045*1.3 = 0.0585; Ca_SS = 0.1 -> rate = 0.00585 + 0.005 = 0.01085: tau = 92.16589861751152, inf = 0.4608294930875576."""
    inf, tau = oracle.tp06_gates(-80.0, 0, Ca_SS=0.1, Ca_SR=3.0)
    assert inf[11] == pytest.approx(0.52, rel=1e-14) and tau[11] == pytest.approx(18.0, rel=1e-14)
    assert tau[12] == pytest.approx(1.0 / 0.01085, rel=1e-13) and inf[12] == pytest.approx(0.005 / 0.01085, rel=1e-13)


def _state(**kw):
    """All gates open (1), concentrations equal to the extracellular ones (every Nernst potential 0), v = 10 mV."""
    y = np.ones(19)
    y[IDX["v"]] = 10.0
    y[IDX["Ki"]] = 5.4
    y[IDX["Nai"]] = 140.0
    y[IDX["Cai"]] = 2.0
    y[IDX["CaSS"]] = 2.0
    y[IDX["CaSR"]] = 1.5
    for k, val in kw.items():
        y[IDX[k]] = val
    return y


def test_conductances_with_zero_reversal_potentials(oracle):
    """With K_i = K_o, Na_i = Na_o, Ca_i = Ca_o all Nernst potentials vanish (E_Ks too: both sums are equal), so at v = 10 mV
    with every gate equal to 1 each ohmic current is 10 G:  I_Na 148.38, I_to 0.73 (endo) / 2.94 (mid, epi), I_Kr 1.53
    (sqrt(K_o/5.4) = 1), I_Ks 3.92 (endo, epi) / 0.98 (mid), I_bNa 0.0029, I_bCa 0.00592; I_pK = 10 G_pK/(1+e^{15/5.98}),
    and at v = 25 mV exactly G_pK (25)/2 = 0.1825; I_pCa = G_pCa Ca_i/(K_pCa + Ca_i): Ca_i = K_pCa = 5e-4 -> 0.0619."""
    c = oracle.tp06_currents(_state(), 0)
    assert c["INa"] == pytest.approx(148.38, rel=1e-13)
    assert c["Ito"] == pytest.approx(0.73, rel=1e-13)
    assert c["IKr"] == pytest.approx(1.53, rel=1e-13)
    assert c["IKs"] == pytest.approx(3.92, rel=1e-13)
    assert c["IbNa"] == pytest.approx(0.0029, rel=1e-13)
    assert c["IbCa"] == pytest.approx(0.00592, rel=1e-13)
    assert c["IpK"] == pytest.approx(0.146 / (1 + E(15.0 / 5.98)), rel=1e-13)
    c1, c2 = oracle.tp06_currents(_state(), 1), oracle.tp06_currents(_state(), 2)
    assert c1["Ito"] == pytest.approx(2.94, rel=1e-13) and c2["Ito"] == pytest.approx(2.94, rel=1e-13)
    assert c1["IKs"] == pytest.approx(0.98, rel=1e-13) and c2["IKs"] == pytest.approx(3.92, rel=1e-13)
    assert oracle.tp06_currents(_state(v=25.0), 0)["IpK"] == pytest.approx(0.1825, rel=1e-13)
    assert oracle.tp06_currents(_state(Cai=5e-4), 0)["IpCa"] == pytest.approx(0.0619, rel=1e-13)
    # gate exponents: m^3 h j, xs^2, r s, xr1 xr2, d f f2 fCass
    c = oracle.tp06_currents(_state(m=0.5, h=0.25, j=0.5, xs=0.5, r=0.5, s=0.25, xr1=0.5, xr2=0.25), 0)
    assert c["INa"] == pytest.approx(148.38 / 64.0, rel=1e-13)
    assert c["IKs"] == pytest.approx(3.92 / 4.0, rel=1e-13)
    assert c["Ito"] == pytest.approx(0.73 / 8.0, rel=1e-13) and c["IKr"] == pytest.approx(1.53 / 8.0, rel=1e-13)


def test_ik1_rectifier_special_arguments(oracle):
    """I_K1 = G_K1 a/(a+b) u, u = v - E_K (E_K = 0 here), a = 0.1/(1+e^{0.06(u-200)}),
    b = [3 e^{0.0002(u+100)} + e^{0.1(u-10)}]/(1+e^{-0.5u}).
    u=200 : a = 0.05,              b = [3 e^0.06 + e^19]/(1+e^-100)
    u=-100: a = 0.1/(1+e^-18),     b = [3 + e^-11]/(1+e^50)
    u=10  : a = 0.1/(1+e^-11.4),   b = [3 e^0.022 + 1]/(1+e^-5)               -> I_K1 = 1.305694782...
    u=0   : the current vanishes."""
    def ik1(u):
        return oracle.tp06_currents(_state(v=u), 0)["IK1"]

    a, b = 0.05, (3 * E(0.06) + E(19.0)) / (1 + E(-100.0))
    assert ik1(200.0) == pytest.approx(5.405 * a / (a + b) * 200.0, rel=1e-13)
    a, b = 0.1 / (1 + E(-18.0)), (3.0 + E(-11.0)) / (1 + E(50.0))
    assert ik1(-100.0) == pytest.approx(5.405 * a / (a + b) * -100.0, rel=1e-13)
    assert ik1(-100.0) == pytest.approx(-540.5, rel=1e-6)        # b ~ 6e-22: fully open inward rectifier, G_K1 u
    a, b = 0.1 / (1 + E(-11.4)), (3 * E(0.022) + 1.0) / (1 + E(-5.0))
    assert ik1(10.0) == pytest.approx(5.405 * a / (a + b) * 10.0, rel=1e-13)
    assert ik1(10.0) == pytest.approx(1.305694782, rel=1e-9)
    assert ik1(0.0) == 0.0


def test_exchanger_and_pump_at_zero_voltage(oracle):
    """At v = 0 every voltage factor is 1.
    I_NaCa = k_NaCa (Na_i^3 Ca_o - Na_o^3 Ca_i alpha)/((K_mNai^3 + Na_o^3)(K_mCa + Ca_o)(1 + k_sat)), Na_i = 10, Ca_i = 1e-4:
             1000 (2000 - 686) / ((669921.875 + 2744000)(3.38)(1.1))                      = 0.10352193984...
    I_NaK  = P_NaK K_o/(K_o+K_mK) Na_i/(Na_i+K_mNa)/(1 + 0.1245 + 0.0353), Na_i = 40 (= K_mNa): 2.724 (5.4/6.4)/2/1.1598
    and the voltage dependence: v = RTF ln 2 / 0.35 makes e^{gamma v/RTF} = 2, e^{(gamma-1) v/RTF} = 2^{-13/7}."""
    y = _state(v=0.0, Nai=10.0, Cai=1e-4)
    c = oracle.tp06_currents(y, 0)
    assert c["INaCa"] == pytest.approx(1000.0 * (2000.0 - 686.0) / ((87.5 ** 3 + 140.0 ** 3) * 3.38 * 1.1), rel=1e-13)
    assert c["INaCa"] == pytest.approx(0.10352193984, rel=1e-9)
    c = oracle.tp06_currents(_state(v=0.0, Nai=40.0), 0)
    assert c["INaK"] == pytest.approx(2.724 * (5.4 / 6.4) * 0.5 / 1.1598, rel=1e-13)
    v2 = RTF * math.log(2.0) / 0.35
    e2 = 2.0 ** (-13.0 / 7.0)
    c = oracle.tp06_currents(_state(v=v2, Nai=10.0, Cai=1e-4), 0)
    assert c["INaCa"] == pytest.approx(1000.0 * (2.0 * 2000.0 - e2 * 686.0)
                                       / ((87.5 ** 3 + 140.0 ** 3) * 3.38 * (1.0 + 0.1 * e2)), rel=1e-12)
    c = oracle.tp06_currents(_state(v=10.0 * RTF, Nai=40.0), 0)      # e^{-0.1 v/RTF} = e^-1, e^{-v/RTF} = e^-10
    assert c["INaK"] == pytest.approx(2.724 * (5.4 / 6.4) * 0.5 / (1 + 0.1245 * E(-1.0) + 0.0353 * E(-10.0)), rel=1e-13)


def test_ical_magnitude(oracle):
    """I_CaL = G_CaL d f f2 fCass 4 (v-15) F/RTF (0.25 Ca_SS e^x - Ca_o)/(e^x - 1), x = 2 (v-15)/RTF.
    v = 15 + RTF/2 (x = 1), Ca_SS = 0.4, gates 1:  3.98e-5 * 2 F * (0.1 e - 2)/(e - 1) = -7.7244386..."""
    y = _state(v=15.0 + 0.5 * RTF, CaSS=0.4)
    c = oracle.tp06_currents(y, 0)
    assert c["ICaL"] == pytest.approx(3.980e-5 * 2.0 * 96485.3415 * (0.1 * math.e - 2.0) / (math.e - 1.0), rel=1e-12)
    assert c["ICaL"] == pytest.approx(-7.7244386, rel=1e-7)


def test_sr_fluxes_at_half_saturation(oracle):
    """I_up = V_maxup/(1 + K_up^2/Ca_i^2): Ca_i = K_up = 2.5e-4 -> 0.0031875.
    I_leak = V_leak (Ca_SR - Ca_i), I_xfer = V_xfer (Ca_SS - Ca_i): Ca_SR = 1.5, Ca_SS = 0.002, Ca_i = 2.5e-4.
    I_rel = V_rel O (Ca_SR - Ca_SS), O = k1 Ca_SS^2 Rbar/(k3 + k1 Ca_SS^2), k1 = k1'/k_casr: at Ca_SR = EC = 1.5 k_casr = 1.75;
    choose Ca_SS^2 = k3 k_casr / k1' = 0.06*1.75/0.15 = 0.7 so that O = Rbar/2 = 0.4 with Rbar = 0.8."""
    css = math.sqrt(0.7)
    y = _state(Cai=2.5e-4, CaSR=1.5, CaSS=0.002)
    c = oracle.tp06_currents(y, 0)
    assert c["Iup"] == pytest.approx(0.0031875, rel=1e-13)
    assert c["Ileak"] == pytest.approx(3.6e-4 * (1.5 - 2.5e-4), rel=1e-13)
    assert c["Ixfer"] == pytest.approx(0.0038 * (0.002 - 2.5e-4), rel=1e-13)
    c = oracle.tp06_currents(_state(CaSR=1.5, CaSS=css, R=0.8), 0)
    assert c["Irel"] == pytest.approx(0.102 * 0.4 * (1.5 - css), rel=1e-13)


def test_buffer_factors_and_volume_ratios_in_one_euler_step(oracle):
    """Reading B3: beta = 1/(1 + Buf K/(Ca+K)^2): at Ca = K the factor is 1/(1 + Buf/(4K)):
    beta_i(Ca_i=0.001) = 1/51, beta_sr(Ca_SR=0.3) = 1/(1+10/1.2) = 3/28, beta_ss(Ca_SS=2.5e-4) = 1/401.
    With every gate 0 (no membrane Ca current except the background and pump, no release since Rbar = 0):
      dCa_SR/dt = beta_sr (I_up - I_leak);  dCa_i/dt = beta_i [(I_leak - I_up) V_sr/V_c + I_xfer - (I_bCa + I_pCa - 2 I_NaCa) C/(2 V_c F)]
      dCa_SS/dt = beta_ss (- I_xfer V_c/V_ss)."""
    y = np.zeros(19)
    y[IDX["v"]] = -80.0
    y[IDX["Ki"]] = 138.3; y[IDX["Nai"]] = 7.67
    y[IDX["Cai"]] = 0.001; y[IDX["CaSR"]] = 0.3; y[IDX["CaSS"]] = 2.5e-4
    dt = 0.25
    c = oracle.tp06_currents(y, 0)
    yn, _ = oracle.tp06_run(y, 0, dt, 1)
    Vc, Vsr, Vss, Cap, F = 0.016404, 0.001094, 0.00005468, 0.185, 96485.3415
    iup = 0.006375 / (1 + (2.5e-4 / 0.001) ** 2)          # = 0.006
    ileak = 3.6e-4 * (0.3 - 0.001)
    ixfer = 0.0038 * (2.5e-4 - 0.001)
    assert c["Iup"] == pytest.approx(0.006, rel=1e-13) and c["Irel"] == 0.0 and c["ICaL"] == 0.0
    assert (yn[IDX["CaSR"]] - 0.3) / dt == pytest.approx((3.0 / 28.0) * (iup - ileak), rel=1e-10)
    assert (yn[IDX["CaSS"]] - 2.5e-4) / dt == pytest.approx((1.0 / 401.0) * (-ixfer * Vc / Vss), rel=1e-10)
    memb = (c["IbCa"] + c["IpCa"] - 2.0 * c["INaCa"]) * Cap / (2.0 * Vc * F)
    assert (yn[IDX["Cai"]] - 0.001) / dt == pytest.approx((1.0 / 51.0) * ((ileak - iup) * Vsr / Vc + ixfer - memb), rel=1e-10)


def test_reversal_potential_values(oracle):
    """E_K = RTF ln(5.4/138.3) = -86.6334..., E_Na = RTF ln(140/7.67) = 77.58..., E_Ca = (RTF/2) ln(2/7e-5) = 137.04...,
    E_Ks = RTF ln((5.4 + 0.03*140)/(138.3 + 0.03*7.67)) read off the zero crossings of I_Kr, I_bNa, I_bCa, I_Ks."""
    y = oracle.tp06_rest()
    y[1:14] = 1.0

    def root(name, lo, hi):
        f = lambda v: oracle.tp06_currents(np.r_[v, y[1:]], 0)[name]
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if (f(lo) < 0) == (f(mid) < 0):
                lo = mid
            else:
                hi = mid
        return 0.5 * (lo + hi)

    assert root("IKr", -120.0, 0.0) == pytest.approx(-86.6334280, abs=1e-5)
    assert root("IbNa", 0.0, 150.0) == pytest.approx(77.58546, abs=1e-4)
    assert root("IbCa", 0.0, 250.0) == pytest.approx(137.04376, abs=1e-4)
    assert root("IKs", -120.0, 0.0) == pytest.approx(RTF * math.log(9.6 / (138.3 + 0.2301)), abs=1e-6)
    assert root("IKs", -120.0, 0.0) == pytest.approx(-71.307697, abs=1e-5)
