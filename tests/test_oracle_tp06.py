"""Pins for the oracle's TP06 cell model and its Rush-Larsen / forward-Euler step.

The model's equations are not printed in PAPER.md (ref [3]); DESIGN.md Appendix A states them. These tests pin the
oracle against things fixed outside its own code: the paper's stated rest / plateau figures (tests/golden), the
half-activation points and special-argument values of the sigmoids (where every exponential equals one), Nernst /
detailed-balance reversal potentials, ion-conservation identities linking fluxes and concentration derivatives, the
Rush-Larsen closed form, and the first-order-in-time trend.
"""
import json
import math
import os

import numpy as np
import pytest

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))

RTF = 8314.472 * 310.0 / 96485.3415
F = 96485.3415
IDX = dict(v=0, m=1, h=2, j=3, xr1=4, xr2=5, xs=6, r=7, s=8, d=9, f=10, f2=11, fcass=12, R=13, Cai=14, CaSR=15, CaSS=16,
           Nai=17, Ki=18)


def test_state_and_gate_counts(oracle):
    """TP06 has 19 states of which 13 are integrated by Rush-Larsen (reading B1: 12 HH gates + Rbar)."""
    assert oracle.tp06_rest().size == GOLD["tp06_states"]["value"]
    inf, tau = oracle.tp06_gates(-80.0)
    assert inf.size == GOLD["tp06_gating_variables"]["value"] and tau.size == 13


def test_gate_half_points_and_special_values(oracle):
    """Each steady-state sigmoid equals 1/2 (or 1/4 when squared) at its half-activation voltage, and the time constants
    reduce to hand-computable numbers where a Gaussian argument vanishes. Catches wrong offsets, slopes' signs, swapped
    gates and the endo/epi s-gate switch (reading B5)."""
    g = oracle.tp06_gates
    assert g(-56.86)[0][0] == pytest.approx(0.25, abs=1e-15)          # m_inf = sigma^2
    assert g(-71.55)[0][1] == pytest.approx(0.25, abs=1e-15)          # h_inf
    assert g(-71.55)[0][2] == pytest.approx(0.25, abs=1e-15)          # j_inf = h_inf
    assert g(-26.0)[0][3] == pytest.approx(0.5, abs=1e-15)            # xr1
    assert g(-88.0)[0][4] == pytest.approx(0.5, abs=1e-15)            # xr2
    assert g(-5.0)[0][5] == pytest.approx(0.5, abs=1e-15)             # xs
    assert g(20.0)[0][6] == pytest.approx(0.5, abs=1e-15)             # r
    assert g(-28.0, 0)[0][7] == pytest.approx(0.5, abs=1e-15)         # s endo
    assert g(-20.0, 1)[0][7] == pytest.approx(0.5, abs=1e-15)         # s mid
    assert g(-20.0, 2)[0][7] == pytest.approx(0.5, abs=1e-15)         # s epi
    assert g(-8.0)[0][8] == pytest.approx(0.5, abs=1e-15)             # d
    assert g(-20.0)[0][9] == pytest.approx(0.5, abs=1e-15)            # f
    assert g(-35.0)[0][10] == pytest.approx(0.67 * 0.5 + 0.33, abs=1e-15)   # f2
    inf, tau = g(-80.0, 0, Ca_SS=0.05)
    assert inf[11] == pytest.approx(0.7, abs=1e-15) and tau[11] == pytest.approx(42.0, abs=1e-13)   # fCass at Ca_SS=0.05
    # directions: activation gates rise with v, inactivation gates fall
    lo, hi = g(-90.0)[0], g(40.0)[0]
    for k in (0, 3, 5, 6, 8):
        assert lo[k] < 0.05 and hi[k] > 0.5, k
    for k in (1, 2, 7, 9, 10):
        assert lo[k] > 0.8 and hi[k] < 0.45, k
    assert lo[4] > 0.5 > 0.01 > hi[4]                                 # xr2: shallow slope (24 mV), half point -88 mV
    # Gaussian peaks
    assert g(-40.0)[1][6] == pytest.approx(9.5 + 0.8, abs=1e-13)                          # tau_r
    assert g(-67.0, 0)[1][7] == pytest.approx(1008.0, abs=1e-10)                          # tau_s endo
    assert g(-45.0, 2)[1][7] == pytest.approx(85.0 + 5.0 / (1 + math.exp(-13.0)) + 3.0, abs=1e-12)   # tau_s epi
    assert g(-27.0)[1][9] == pytest.approx(1102.5 + 200.0 / (1 + math.exp(4.0)) + 180.0 / (1 + math.exp(0.3)) + 20.0,
                                           rel=1e-14)                                     # tau_f
    assert g(-27.0)[1][10] == pytest.approx(562.0 + 31.0 / (1 + math.exp(5.2)) + 80.0 / (1 + math.exp(0.3)), rel=1e-14)
    # tau_m is tiny (sub-ms) everywhere, tau_h / tau_j are ms-scale near rest and shrink when depolarised
    for v in np.linspace(-100, 60, 33):
        inf, tau = g(float(v))
        assert 0 < tau[0] < 0.2
        assert np.all(tau > 0) and np.all(inf >= 0) and np.all(inf <= 1)
    # reading B7: the h/j rate branch switches at v = -40 with v >= -40 on the high-voltage branch
    t_hi = g(-40.0)[1][1]
    assert t_hi == pytest.approx(0.13 * (1 + math.exp(-(-40 + 10.66) / 11.1)) / 0.77, rel=1e-14)
    assert abs(g(-40.0 - 1e-9)[1][1] / t_hi - 1) < 0.05     # ~1% jump only
    assert g(-40.0 - 1e-9)[1][1] != t_hi


def test_rbar_linear_ode(oracle):
    """Reading B1: dR/dt = k4(1-R) - k2 Ca_SS R is linear in R => R_inf = k4/(k2 CaSS + k4), tau = 1/(k2 CaSS + k4);
    at Ca_SR = EC = 1.5 the SR factor k_casr = max_sr - (max_sr-min_sr)/2 = 1.75."""
    inf, tau = oracle.tp06_gates(-80.0, 0, Ca_SS=1e-3, Ca_SR=1.5)
    k2 = 0.045 * 1.75
    assert tau[12] == pytest.approx(1.0 / (k2 * 1e-3 + 0.005), rel=1e-14)
    assert inf[12] == pytest.approx(0.005 / (k2 * 1e-3 + 0.005), rel=1e-14)


def test_reversal_potentials_and_current_signs(oracle):
    """Nernst potentials: every K current vanishes at v = E_K, I_Na and I_bNa at E_Na, I_bCa at E_Ca, I_Ks at E_Ks; the
    exchanger vanishes at its detailed-balance potential v = RTF ln(alpha Na_o^3 Ca_i / (Na_i^3 Ca_o))."""
    y = oracle.tp06_rest()
    y[IDX["m"]] = 0.3; y[IDX["xr1"]] = 0.4; y[IDX["xs"]] = 0.5; y[IDX["r"]] = 0.6; y[IDX["d"]] = 0.2
    Ki, Nai, Cai = y[IDX["Ki"]], y[IDX["Nai"]], y[IDX["Cai"]]
    EK = RTF * math.log(5.4 / Ki)
    ENa = RTF * math.log(140.0 / Nai)
    ECa = 0.5 * RTF * math.log(2.0 / Cai)
    EKs = RTF * math.log((5.4 + 0.03 * 140.0) / (Ki + 0.03 * Nai))
    assert EK == pytest.approx(-86.6, abs=0.3) and ENa == pytest.approx(77.6, abs=0.5)   # textbook magnitudes

    def at(v):
        z = y.copy(); z[0] = v
        return oracle.tp06_currents(z, 2)

    c = at(EK)
    for k in ("IK1", "Ito", "IKr", "IpK"):
        assert abs(c[k]) < 1e-12, k
    assert abs(at(ENa)["INa"]) < 1e-10 and abs(at(ENa)["IbNa"]) < 1e-14
    assert abs(at(ECa)["IbCa"]) < 1e-14
    assert abs(at(EKs)["IKs"]) < 1e-13
    vrev = RTF * math.log(2.5 * 140.0 ** 3 * Cai / (Nai ** 3 * 2.0))
    assert abs(at(vrev)["INaCa"]) < 1e-12
    assert at(vrev + 20)["INaCa"] > 0 > at(vrev - 20)["INaCa"]      # outward (3 Na+ out... net +1 charge) above reversal
    # signs at a depolarised potential: Na and Ca currents inward, K currents outward, pump outward
    c = at(0.0)
    assert c["INa"] < 0 and c["ICaL"] < 0 and c["IbNa"] < 0 and c["IbCa"] < 0
    assert c["IK1"] >= 0 and c["Ito"] > 0 and c["IKr"] > 0 and c["IKs"] > 0 and c["IpK"] > 0 and c["INaK"] > 0
    assert c["IpCa"] > 0
    # i_ion is the sum of the twelve membrane currents
    s12 = sum(c[k] for k in ("INa", "ICaL", "Ito", "IKr", "IKs", "IK1", "INaCa", "INaK", "IpCa", "IpK", "IbNa", "IbCa"))
    assert c["iion"] == pytest.approx(s12, rel=1e-15)
    # pump saturation: I_NaK -> P_NaK * Ko/(Ko+KmK) * Nai/(Nai+KmNa) as v -> +inf
    assert at(20000.0)["INaK"] == pytest.approx(2.724 * 5.4 / 6.4 * Nai / (Nai + 40.0), rel=1e-12)
    # cell-type conductances (reading B5)
    assert at(0.0)["IKs"] / oracle.tp06_currents(np.r_[0.0, y[1:]], 1)["IKs"] == pytest.approx(0.392 / 0.098, rel=1e-14)
    assert oracle.tp06_currents(np.r_[0.0, y[1:]], 0)["Ito"] / at(0.0)["Ito"] == pytest.approx(0.073 / 0.294, rel=1e-14)


def test_ical_removable_singularity(oracle):
    """Reading B6: I_CaL at v = 15 mV is the analytic limit G d f f2 fCass 2F (Ca_SS/4 - Ca_o) and is continuous there."""
    y = oracle.tp06_rest()
    y[IDX["d"]] = 0.5
    y[IDX["CaSS"]] = 0.01

    def ical(v):
        z = y.copy(); z[0] = v
        return oracle.tp06_currents(z, 0)["ICaL"]

    lim = 3.980e-5 * 0.5 * 1 * 1 * 1 * 2 * F * (0.25 * 0.01 - 2.0)
    assert ical(15.0) == pytest.approx(lim, rel=1e-14)
    for dv in (1e-9, 1e-7, 1e-5, 1e-3):
        # |d ln I / dv| ~ 0.04/mV here, so the values differ from the limit by ~0.04 dv; round-off stays below 1e-8
        assert abs(ical(15.0 + dv) / lim - 1) < 0.05 * dv + 1e-8
        assert abs(ical(15.0 - dv) / lim - 1) < 0.05 * dv + 1e-8


def test_ion_conservation_identities(oracle):
    """One forward-Euler step must move each concentration by dt * (its flux balance). Internal Ca fluxes
    (release, leak, uptake, transfer) cancel in the volume-weighted sum of the unbuffered Ca derivatives, leaving only the
    sarcolemmal Ca currents; Na and K follow from the membrane currents with charge 1. Pins volumes, capacitance, valence,
    the stoichiometry 3:1 / 3:2 and reading B8 (the stimulus enters K_i)."""
    y = oracle.tp06_rest()
    y[0] = -20.0
    y[IDX["m"]] = 0.2; y[IDX["d"]] = 0.3; y[IDX["xr1"]] = 0.3; y[IDX["xs"]] = 0.2; y[IDX["r"]] = 0.5
    y[IDX["CaSS"]] = 2e-3; y[IDX["Cai"]] = 2e-4; y[IDX["R"]] = 0.9
    typ, dt, istim = 2, 0.5, -7.0    # forward Euler is linear in dt; a large dt keeps the difference quotients clean
    c = oracle.tp06_currents(y, typ)
    yn, _ = oracle.tp06_run(y, typ, dt, 1, istim, 0, 1)
    Vc, Vsr, Vss, Cap = 0.016404, 0.001094, 0.00005468, 0.185
    dNa = (yn[IDX["Nai"]] - y[IDX["Nai"]]) / dt
    dK = (yn[IDX["Ki"]] - y[IDX["Ki"]]) / dt
    assert dNa == pytest.approx(-(c["INa"] + c["IbNa"] + 3 * c["INaK"] + 3 * c["INaCa"]) * Cap / (Vc * F), rel=1e-9)
    assert dK == pytest.approx(-(c["IK1"] + c["Ito"] + c["IKr"] + c["IKs"] - 2 * c["INaK"] + c["IpK"] + istim) * Cap
                               / (Vc * F), rel=1e-9)
    bi = 1 / (1 + 0.2 * 0.001 / (y[IDX["Cai"]] + 0.001) ** 2)
    bsr = 1 / (1 + 10.0 * 0.3 / (y[IDX["CaSR"]] + 0.3) ** 2)
    bss = 1 / (1 + 0.4 * 2.5e-4 / (y[IDX["CaSS"]] + 2.5e-4) ** 2)
    dCai = (yn[IDX["Cai"]] - y[IDX["Cai"]]) / dt / bi
    dCaSR = (yn[IDX["CaSR"]] - y[IDX["CaSR"]]) / dt / bsr
    dCaSS = (yn[IDX["CaSS"]] - y[IDX["CaSS"]]) / dt / bss
    total = Vc * dCai + Vsr * dCaSR + Vss * dCaSS
    memb = -(c["IbCa"] + c["IpCa"] - 2 * c["INaCa"] + c["ICaL"]) * Cap / (2 * F)
    assert total == pytest.approx(memb, rel=1e-7)
    # SR balance alone: dCaSR = Iup - Ileak - Irel
    assert dCaSR == pytest.approx(c["Iup"] - c["Ileak"] - c["Irel"], rel=1e-9)
    # v: dv/dt = -(i_ion + i_stim) with no diffusion (eq. (1) with the sign printed at PAPER.md:107, reading A15)
    assert (yn[0] - y[0]) / dt == pytest.approx(-(c["iion"] + istim), rel=1e-10)


def test_rush_larsen_closed_form(oracle):
    """P8 / PAPER.md:174: with v (and Ca) frozen the quasi-linear gate ODE has the exact solution
    y(t) = y_inf + (y0 - y_inf) exp(-t/tau), which Rush-Larsen reproduces for ANY dt; gates stay in [0,1]."""
    y0 = oracle.tp06_rest()
    y0[0] = -30.0
    inf, tau = oracle.tp06_gates(-30.0, 2, y0[IDX["CaSS"]], y0[IDX["CaSR"]])
    for dt, n in ((0.02, 500), (0.5, 20), (5.0, 2)):
        y, _ = oracle.tp06_run(y0, 2, dt, n, freeze_v=True)
        T = dt * n
        for g in range(11):     # the 11 voltage-only gates (fCass and Rbar see Ca_SS / Ca_SR, which keep moving)
            exact = inf[g] + (y0[1 + g] - inf[g]) * math.exp(-T / tau[g])
            assert y[1 + g] == pytest.approx(exact, abs=1e-12), (dt, g)
        assert np.all(y[1:14] >= 0) and np.all(y[1:14] <= 1)


def _apd90(tr, dt):
    rest, peak = tr[0], tr.max()
    v90 = rest + 0.1 * (peak - rest)
    up = int(np.argmax(np.diff(tr)))
    below = np.nonzero(tr[up:] < v90)[0]
    return below[0] * dt


def test_single_cell_rest_and_action_potential(oracle):
    """P9 / PAPER.md:256: 'resting potential of about -85 mV ... plateau of about 300 ms'. Unstimulated the built-in rest
    set holds within 0.1 mV of -86.1 for 1 s (north_star: 'hold rest near -86 mV'); paced with -52 uA/uF for 1 ms it shows
    a full upstroke (overshoot > +30 mV, max dv/dt in the hundreds of mV/ms) and repolarises; mid cells (G_Ks / 4) have
    the longest action potential."""
    y0 = oracle.tp06_rest()
    dt = 0.02
    apd = {}
    for typ in (0, 1, 2):
        y, tr = oracle.tp06_run(y0, typ, dt, 50000, trace=True)
        assert abs(tr[-1] - GOLD["tp06_rest_mV"]["value"]) < GOLD["tp06_rest_mV"]["tol"]
        assert np.abs(tr + 86.1).max() < 0.15
        y, tr = oracle.tp06_run(y0, typ, dt, 30000, -52.0, 0, 50, trace=True)
        assert 30.0 < tr.max() < 50.0
        dvdt = np.diff(tr).max() / dt
        assert 250.0 < dvdt < 500.0
        assert tr[-1] < -85.0                      # repolarised after 600 ms
        apd[typ] = _apd90(tr, dt)
    assert abs(apd[0] - GOLD["tp06_plateau_ms"]["value"]) < GOLD["tp06_plateau_ms"]["tol"]
    assert abs(apd[2] - GOLD["tp06_plateau_ms"]["value"]) < GOLD["tp06_plateau_ms"]["tol"]
    assert apd[1] > apd[0] + 60 and apd[1] > apd[2] + 60


def test_first_order_in_time_and_large_dt_stability(oracle):
    """P10 / PAPER.md:232 ('first-order accuracy in time') and :174 (RL allows time steps 'more than one order of
    magnitude' larger than plain explicit)."""
    y0 = oracle.tp06_rest()
    T = 20.0
    ref, _ = oracle.tp06_run(y0, 0, 0.00125, int(T / 0.00125), -52.0, 0, int(1 / 0.00125))
    errs = []
    for dt in (0.04, 0.02, 0.01):
        y, _ = oracle.tp06_run(y0, 0, dt, int(round(T / dt)), -52.0, 0, int(round(1 / dt)))
        errs.append(abs(y[0] - ref[0]))
    assert 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.6, errs
    y, tr = oracle.tp06_run(y0, 0, 0.1, 6000, -52.0, 0, 10, trace=True)     # dt = 0.1 ms: still a normal AP
    assert np.isfinite(tr).all() and tr.max() > 25 and tr[-1] < -85
