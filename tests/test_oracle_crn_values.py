"""Hand-computed values of the Courtemanche model's conductances, rate constants and fluxes (DESIGN.md Appendix B, the
published model, PAPER.md:352 ref [1]) at arguments where the expressions collapse: a sigmoid at its centre is 1/2, an
exponential with zero argument is 1, a Nernst potential with equal concentrations is 0, phi(0) = 1.  Companion of
tests/test_oracle_tp06_values.py; tests/test_oracle_mutations.py checks that single-constant edits fail these.
Gate order: m h j oa oi ua ui xr xs d f fCa u v w."""
import math

import numpy as np
import pytest

E = math.exp
F = 96.4867
RTF = 8.3143 * 310.0 / F
N = ["m", "h", "j", "oa", "oi", "ua", "ui", "xr", "xs", "d", "f", "fCa", "u", "v", "w"]


def _g(oracle, V, **k):
    inf, tau = oracle.crn_gates(V, **k)
    return dict(zip(N, inf)), dict(zip(N, tau))


def _state(V=10.0, **kw):
    """every gate 1, intracellular = extracellular concentrations (all Nernst potentials 0)"""
    y = np.ones(21)
    y[0] = V
    y[16], y[17], y[18], y[19], y[20] = 140.0, 5.4, 1.8, 1.5, 1.5
    names = dict(m=1, h=2, j=3, oa=4, oi=5, ua=6, ui=7, xr=8, xs=9, d=10, f=11, fCa=12, u=13, v=14, w=15, Nai=16, Ki=17,
                 Cai=18, Caup=19, Carel=20)
    for k, val in kw.items():
        y[names[k]] = val
    return y


def test_conductances_with_zero_reversal_potentials(oracle):
    """V = 10 mV, E_K = E_Na = E_Ca = 0, gates 1: I_Na = 78, I_to = 1.652, I_Ks = 1.29, I_bNa = 0.00674, I_bCa = 0.0113,
    I_CaL = g_CaL (10 - 65) = -6.809; I_K1(V=-80) = g_K1 (-80)/2 = -3.6; I_Kr(V=-15) = g_Kr (-15)/2 = -0.2205;
    g_Kur(V=15) = 0.005 + 0.05/2 = 0.03 -> I_Kur = 0.45; I_pCa(Ca_i = 0.0005) = 0.1375; gate powers m^3 h j, oa^3 oi, ua^3 ui, xs^2."""
    c = oracle.crn_currents(_state())
    assert c["INa"] == pytest.approx(78.0, rel=1e-13) and c["Ito"] == pytest.approx(1.652, rel=1e-13)
    assert c["IKs"] == pytest.approx(1.29, rel=1e-13) and c["IbNa"] == pytest.approx(0.00674, rel=1e-13)
    assert c["IbCa"] == pytest.approx(0.0113, rel=1e-13) and c["ICaL"] == pytest.approx(-6.809, rel=1e-13)
    assert oracle.crn_currents(_state(-80.0))["IK1"] == pytest.approx(-3.6, rel=1e-13)
    assert oracle.crn_currents(_state(-15.0))["IKr"] == pytest.approx(-0.2205, rel=1e-13)
    assert oracle.crn_currents(_state(15.0))["IKur"] == pytest.approx(0.45, rel=1e-13)
    assert oracle.crn_currents(_state(Cai=0.0005))["IpCa"] == pytest.approx(0.1375, rel=1e-13)
    c = oracle.crn_currents(_state(m=0.5, h=0.5, j=0.25, oa=0.5, oi=0.5, ua=0.5, ui=0.25, xs=0.5, xr=0.5))
    assert c["INa"] == pytest.approx(78.0 / 64, rel=1e-13) and c["Ito"] == pytest.approx(1.652 / 16, rel=1e-13)
    assert c["IKs"] == pytest.approx(1.29 / 4, rel=1e-13)
    gkur10 = 0.005 + 0.05 / (1 + E(5.0 / 13.0))
    assert c["IKur"] == pytest.approx(gkur10 * 10.0 / 32, rel=1e-13)
    assert c["IKr"] == pytest.approx(0.0294 * 0.5 * 10.0 / (1 + E(25.0 / 22.4)), rel=1e-13)
    # slopes of the two rectifier sigmoids one e-fold from their centres: 1/0.07 and 22.4 mV
    assert oracle.crn_currents(_state(-80.0 + 1 / 0.07))["IK1"] == pytest.approx(0.09 * (-80 + 1 / 0.07) / (1 + math.e), rel=1e-13)
    assert oracle.crn_currents(_state(-15.0 + 22.4))["IKr"] == pytest.approx(0.0294 * 7.4 / (1 + math.e), rel=1e-13)


def test_exchanger_pump_and_sr_fluxes(oracle):
    """V = 0: I_NaCa = 1600 (Na_i^3 Ca_o - Na_o^3 Ca_i)/((87.5^3 + 140^3)(1.38 + 1.8)(1.1)) with Na_i = 10, Ca_i = 1e-4:
    1600 (1800 - 274.4)/(3413921.875 * 3.18 * 1.1) = 0.20440...;
    I_up(Ca_i = K_up) = 0.0025; I_up,leak = Ca_up/15 * 0.005 (Ca_up = 3 -> 0.001); I_tr = (Ca_up - Ca_rel)/180;
    I_rel = 30 u^2 v w (Ca_rel - Ca_i);  Fn (u = 0 so I_rel = 0) = -(5e-13/F) C_m (0.5 I_CaL - 0.2 I_NaCa)."""
    y = _state(0.0, Nai=10.0, Cai=1e-4)
    c = oracle.crn_currents(y)
    inaca = 1600.0 * (1000.0 * 1.8 - 140.0 ** 3 * 1e-4) / ((87.5 ** 3 + 140.0 ** 3) * 3.18 * 1.1)
    assert c["INaCa"] == pytest.approx(inaca, rel=1e-13) and inaca == pytest.approx(0.2044, rel=2e-4)
    assert oracle.crn_currents(_state(Cai=0.00092))["Iup"] == pytest.approx(0.0025, rel=1e-13)
    c = oracle.crn_currents(_state(Caup=3.0, Carel=1.2, Cai=2e-4, u=0.5, v=0.5, w=0.8))
    assert c["Iupleak"] == pytest.approx(0.001, rel=1e-13) and c["Itr"] == pytest.approx(0.01, rel=1e-13)
    assert c["Irel"] == pytest.approx(30.0 * 0.25 * 0.5 * 0.8 * (1.2 - 2e-4), rel=1e-13)
    y = _state(0.0, Nai=10.0, Cai=1e-4, u=0.0)
    c = oracle.crn_currents(y)
    assert c["Irel"] == 0.0
    assert c["Fn"] == pytest.approx(-(5e-13 / F) * 100.0 * (0.5 * 0.1238 * (-65.0) - 0.2 * inaca), rel=1e-12, abs=0.0)
    y[13] = 1.0                                   # and the release term: 1e-12 V_rel I_rel
    c2 = oracle.crn_currents(y)
    assert c2["Fn"] - c["Fn"] == pytest.approx(1e-12 * 96.48 * 30.0 * (1.5 - 1e-4), rel=1e-9, abs=0.0)


def test_sodium_gate_rates(oracle):
    """V = -80: alpha_h = 0.135, beta_h = 3.56 e^-6.32 + 3.1e5 e^-28; V = -47.13: alpha_m = 3.2, beta_m = 0.08 e^{47.13/11};
    V = 0: beta_m = 0.08, alpha_m = 0.32*47.13/(1 - e^-4.713); V = -32 (high branch): beta_j = 0.3 e^{2.535e-7*32}/2;
    V = -10.66: beta_h = 1/(0.13*2); V = -79.23 (low branch): the alpha_j denominator is 2."""
    inf, tau = _g(oracle, -80.0)
    bh = 3.56 * E(-6.32) + 3.1e5 * E(-28.0)
    assert tau["h"] == pytest.approx(1 / (0.135 + bh), rel=1e-13) and inf["h"] == pytest.approx(0.135 / (0.135 + bh), rel=1e-13)
    inf, tau = _g(oracle, 0.0)
    am = 0.32 * 47.13 / (1 - E(-4.713))
    assert tau["m"] == pytest.approx(1 / (am + 0.08), rel=1e-13) and inf["m"] == pytest.approx(am / (am + 0.08), rel=1e-13)
    assert _g(oracle, -32.0)[1]["j"] == pytest.approx(2.0 / (0.3 * E(2.535e-7 * 32.0)), rel=1e-13)
    assert _g(oracle, -10.66)[1]["h"] == pytest.approx(0.26, rel=1e-13)
    aj = (-127140.0 * E(-0.2444 * 79.23) - 3.474e-5 * E(0.04391 * 79.23)) * (-79.23 + 37.78) / 2.0
    bj = 0.1212 * E(0.01052 * 79.23) / (1 + E(-0.1378 * (-79.23 + 40.14)))
    inf, tau = _g(oracle, -79.23)
    assert tau["j"] == pytest.approx(1 / (aj + bj), rel=1e-12) and inf["j"] == pytest.approx(aj / (aj + bj), rel=1e-12)


def test_potassium_gate_rates(oracle):
    """oa/ua: V = -10: alpha = 0.65/(1 + e^{40/59}); V = -82: beta = 0.65/3.5; tau = 1/(alpha+beta)/3 (K_Q10 = 3).
    oi: V = -113.7: alpha = 1/19.53; V = -1.26: beta = 1/36.56.  ui: V = 185: alpha = 1/22; V = 158: beta = 1.
    xr: V = 3.3328: beta = 7.3898e-5*5.1237, alpha = 0.0003*17.4328/(1 - e^{-17.4328/5}).  Slopes one e-fold from the centres."""
    for V in (-10.0, -82.0):
        a = 0.65 / (E(-(V + 10) / 8.5) + E(-(V - 30) / 59.0)) if V != -10.0 else 0.65 / (1 + E(40.0 / 59.0))
        b = 0.65 / (2.5 + E((V + 82) / 17.0)) if V != -82.0 else 0.65 / 3.5
        assert _g(oracle, V)[1]["oa"] == pytest.approx(1 / (a + b) / 3.0, rel=1e-13)
        assert _g(oracle, V)[1]["ua"] == pytest.approx(1 / (a + b) / 3.0, rel=1e-13)
    a, b = 1 / 19.53, 1 / (35.56 + E(112.44 / 7.44))
    assert _g(oracle, -113.7)[1]["oi"] == pytest.approx(1 / (a + b) / 3.0, rel=1e-13)
    a, b = 1 / (18.53 + E(112.44 / 10.95)), 1 / 36.56
    assert _g(oracle, -1.26)[1]["oi"] == pytest.approx(1 / (a + b) / 3.0, rel=1e-13)
    assert _g(oracle, 185.0)[1]["ui"] == pytest.approx(1 / (1 / 22.0 + E(27.0 / 16.0)) / 3.0, rel=1e-13)
    assert _g(oracle, 158.0)[1]["ui"] == pytest.approx(1 / (1 / (21.0 + E(27.0 / 28.0)) + 1.0) / 3.0, rel=1e-13)
    a = 0.0003 * 17.4328 / (1 - E(-17.4328 / 5.0))
    assert _g(oracle, 3.3328)[1]["xr"] == pytest.approx(1 / (a + 7.3898e-5 * 5.1237), rel=1e-12)
    hi, lo = 1 / (1 + 1 / math.e), 1 / (1 + math.e)
    assert _g(oracle, -20.47 + 17.54)[0]["oa"] == pytest.approx(hi, rel=1e-13)
    assert _g(oracle, -43.1 + 5.3)[0]["oi"] == pytest.approx(lo, rel=1e-13)
    assert _g(oracle, -30.3 + 9.6)[0]["ua"] == pytest.approx(hi, rel=1e-13)
    assert _g(oracle, 99.45 + 27.48)[0]["ui"] == pytest.approx(lo, rel=1e-13)
    assert _g(oracle, -14.1 + 6.5)[0]["xr"] == pytest.approx(hi, rel=1e-13)
    assert _g(oracle, 19.9 + 12.7)[0]["xs"] == pytest.approx(math.sqrt(hi), rel=1e-13)


def test_calcium_gate_rates(oracle):
    """d: V = -10 + 8 -> d_inf = 1/(1+1/e); f: V = -10 -> tau = 9/(0.0197 + 0.02), V = -28 + 6.9 -> f_inf = 1/(1+e);
    tau_f one Gaussian e-fold away: V = -10 + 1/0.0337 -> 9/(0.0197/e + 0.02); w_inf slope 17; tau_fCa = 2, tau_u = 8;
    tau_v = 1.91 + 2.09 u_inf."""
    hi, lo = 1 / (1 + 1 / math.e), 1 / (1 + math.e)
    assert _g(oracle, -2.0)[0]["d"] == pytest.approx(hi, rel=1e-13)
    assert _g(oracle, -10.0)[1]["f"] == pytest.approx(9.0 / 0.0397, rel=1e-13)
    assert _g(oracle, -10.0 + 1 / 0.0337)[1]["f"] == pytest.approx(9.0 / (0.0197 / math.e + 0.02), rel=1e-12)
    assert _g(oracle, -28.0 + 6.9)[0]["f"] == pytest.approx(lo, rel=1e-13)
    assert _g(oracle, 40.0 + 17.0)[0]["w"] == pytest.approx(lo, rel=1e-13)      # w_inf = 1 - s(-(V-40)/17) falls with V
    inf, tau = _g(oracle, 0.0, Fn=3.4175e-13)
    assert tau["v"] == pytest.approx(1.91 + 2.09 / 2, rel=1e-12) and tau["u"] == 8.0 and tau["fCa"] == 2.0
    inf, tau = _g(oracle, 0.0, Fn=3.4175e-13 + 13.67e-16)
    assert inf["u"] == pytest.approx(hi, rel=1e-9)
    assert _g(oracle, 0.0, Fn=6.835e-14 + 13.67e-16)[0]["v"] == pytest.approx(lo, rel=1e-9)
    assert _g(oracle, 0.0, Cai=0.0007)[0]["fCa"] == pytest.approx(1.0 / 3.0, rel=1e-13)
