"""Pins of the Stewart 2009 Purkinje cell model in oracle/ep_oracle2d.cpp (Table 2 :271).

What fixes the transcription from outside the oracle: the paper's counts (20 states, 13 Rush-Larsen gates) and facts
("high peak of depolarization followed by a stable plateau phase of about 250 ms"; "3.95 mS/mm
corresponding to a velocity 4.0 m/s", Table 2), numbers computed by hand at voltages where the exponentials are 1 or
e^+-1 (typed below as numbers, not as the oracle's expressions), zero crossings of the currents, ion-conservation
identities, the Rush-Larsen closed form, and -- for the equations the model inherits unchanged from ten Tusscher-Panfilov
2006 -- the separately transcribed and separately pinned TP06 functions of oracle/ep_oracle.cpp.
"""
import numpy as np
import pytest

from oracle import ep_oracle as O3
from oracle import ep_oracle2d as O2

RTF = 8314.472 * 310.0 / 96485.3415          # 26.713760659695648 mV
F = 96485.3415
IDX = {n: i for i, n in enumerate(O2.STW_STATES)}
G = {n: i for i, n in enumerate(O2.STW_GATES)}


def _state(**kw):
    y = O2.stw_init()
    for k, v in kw.items():
        y[IDX[k]] = v
    return y


def test_counts_match_the_paper():
    """'the Stewart model with 13 gating variables out of 20 state variables'."""
    assert len(O2.STW_STATES) == 20 and len(O2.STW_GATES) == 13
    assert O2.stw_init().shape == (20,)
    inf, tau = O2.stw_gates(-70.0)
    assert inf.shape == (13,) and (tau > 0).all() and ((inf >= 0) & (inf <= 1)).all()


def test_purkinje_specific_gates_by_hand():
    # y (I_f): half-point -80.6 mV, slope 6.8; tau_y = 4000/(e^{-2.9-0.04v} + e^{3.6+0.11v})
    inf, tau = O2.stw_gates(-80.6)
    assert inf[G["y"]] == pytest.approx(0.5, abs=1e-15)
    inf, tau = O2.stw_gates(-73.8)                     # (v+80.6)/6.8 = 1
    assert inf[G["y"]] == pytest.approx(0.2689414213699951, rel=1e-14)
    assert O2.stw_gates(0.0)[1][G["y"]] == pytest.approx(109.13081823986671, rel=1e-13)
    assert O2.stw_gates(-72.5)[1][G["y"]] == pytest.approx(3950.2733965872562, rel=1e-13)   # first exponent is 0
    assert O2.stw_gates(-100.0)[1][G["y"]] == pytest.approx(1331.2134749577635, rel=1e-13)
    # r, s of the Purkinje transient outward current
    inf, tau = O2.stw_gates(20.0)
    assert inf[G["r"]] == pytest.approx(0.5, abs=1e-15)
    assert O2.stw_gates(7.0)[0][G["r"]] == pytest.approx(0.2689414213699951, rel=1e-14)      # (20-7)/13 = 1
    assert O2.stw_gates(-40.0)[1][G["r"]] == pytest.approx(17.75, rel=1e-15)                 # Gaussian at its peak
    assert O2.stw_gates(-40.0 + np.sqrt(1800.0))[1][G["r"]] == pytest.approx(11.144340160241573, rel=1e-13)
    inf, tau = O2.stw_gates(-27.0)
    assert inf[G["s"]] == pytest.approx(0.5, abs=1e-15)
    assert O2.stw_gates(-14.0)[0][G["s"]] == pytest.approx(0.2689414213699951, rel=1e-14)    # (-14+27)/13 = 1
    assert O2.stw_gates(-25.0)[1][G["s"]] == pytest.approx(131.9999886983785, rel=1e-13)
    assert O2.stw_gates(40.0)[1][G["s"]] == pytest.approx(44.500156810303125, rel=1e-13)


def test_inherited_gates_equal_the_tp06_transcription():
    """xr1 xr2 xs m h j d f f2 fCass are ten Tusscher-Panfilov 2006's (reading B13); oracle/ep_oracle.cpp states them
    separately and tests/test_oracle_tp06_values.py pins every constant of them by hand."""
    tp = {"m": 0, "h": 1, "j": 2, "xr1": 3, "xr2": 4, "xs": 5, "d": 8, "f": 9, "f2": 10, "fCass": 11}
    for v in (-95.0, -86.2, -60.0, -40.0, -39.999, -20.0, 0.0, 15.0, 30.0, 55.0):
        for cass in (1e-4, 4e-4, 0.02, 0.3):
            i2, t2 = O2.stw_gates(v, cass)
            i3, t3 = O3.tp06_gates(v, 0, cass, 3.1)
            for n, k in tp.items():
                assert i2[G[n]] == pytest.approx(i3[k], rel=1e-14, abs=1e-300), (n, v)
                assert t2[G[n]] == pytest.approx(t3[k], rel=1e-14), (n, v)


def test_currents_zero_crossings_conductances_and_hand_values():
    y = O2.stw_init()
    EK = RTF * np.log(5.4 / y[IDX["K_i"]])
    ENa = RTF * np.log(140.0 / y[IDX["Na_i"]])
    assert EK == pytest.approx(-86.33857232561857, rel=1e-13) and ENa == pytest.approx(73.90130055961373, rel=1e-13)
    # I_f: sodium part reverses at E_Na, potassium part at E_K, conductances 0.0145654 / 0.0234346 per unit y
    assert abs(O2.stw_currents(_state(V=ENa))["IfNa"]) < 1e-15
    assert abs(O2.stw_currents(_state(V=EK))["IfK"]) < 1e-15
    c = O2.stw_currents(_state(V=-60.0, y=1.0))
    assert c["IfNa"] == pytest.approx(0.0145654 * (-60.0 - ENa), rel=1e-13)
    assert c["IfK"] == pytest.approx(0.0234346 * (-60.0 - EK), rel=1e-13)
    assert O2.stw_currents(_state(V=-60.0, y=0.25))["IfK"] == pytest.approx(0.25 * c["IfK"], rel=1e-13)
    # I_K1 = 0.065 / (1 + e^{0.1 (v + 75.44)}) (v - 8 - E_K): zero at E_K + 8, hand values where the exponent is 0 and 1
    assert abs(O2.stw_currents(_state(V=EK + 8.0))["IK1"]) < 1e-15
    assert O2.stw_currents(_state(V=-75.44))["IK1"] == pytest.approx(0.09420360058260364, rel=1e-12)
    assert O2.stw_currents(_state(V=-65.44))["IK1"] == pytest.approx(0.22548242436821028, rel=1e-12)
    # I_sus = 0.0227 / (1 + e^{(5 - v)/17}) (v - E_K)
    assert O2.stw_currents(_state(V=5.0))["Isus"] == pytest.approx(1.0366927958957708, rel=1e-12)
    assert O2.stw_currents(_state(V=22.0))["Isus"] == pytest.approx(1.797881829180375, rel=1e-12)
    # conductances of the gated currents with every gate open
    v = -20.0
    c = O2.stw_currents(_state(V=v, m=1.0, h=1.0, j=1.0, r=1.0, s=1.0, xr1=1.0, xr2=1.0, xs=1.0))
    EKs = RTF * np.log((5.4 + 0.03 * 140.0) / (y[IDX["K_i"]] + 0.03 * y[IDX["Na_i"]]))
    assert c["INa"] == pytest.approx(130.5744 * (v - ENa), rel=1e-13)
    assert c["Ito"] == pytest.approx(0.08184 * (v - EK), rel=1e-13)
    assert c["IKr"] == pytest.approx(0.0918 * (v - EK), rel=1e-13)
    assert c["IKs"] == pytest.approx(0.2352 * (v - EKs), rel=1e-13)
    # gate exponents: m^3 h j, r s, xr1 xr2, xs^2
    c2 = O2.stw_currents(_state(V=v, m=0.5, h=0.5, j=0.25, r=0.5, s=0.25, xr1=0.5, xr2=0.25, xs=0.5))
    assert c2["INa"] == pytest.approx(c["INa"] / 64.0, rel=1e-13) and c2["Ito"] == pytest.approx(c["Ito"] / 8.0, rel=1e-13)
    assert c2["IKr"] == pytest.approx(c["IKr"] / 8.0, rel=1e-13) and c2["IKs"] == pytest.approx(c["IKs"] / 4.0, rel=1e-13)
    # the sum
    names = ["IfNa", "IfK", "IK1", "Ito", "Isus", "IKr", "IKs", "ICaL", "INaK", "INa", "IbNa", "INaCa", "IbCa", "IpK", "IpCa"]
    assert c2["iion"] == pytest.approx(sum(c2[n] for n in names), rel=1e-13)


def test_inherited_currents_equal_the_tp06_transcription():
    """I_CaL, I_NaK, I_NaCa, I_pCa, I_pK, I_bNa, I_bCa and the SR fluxes are TP06's with TP06's constants."""
    rng = np.random.default_rng(5)
    for _ in range(20):
        y2 = O2.stw_init()
        y2[0] = rng.uniform(-90, 40)
        y2[1:14] = rng.uniform(0.01, 0.99, 13)
        y2[IDX["Ca_i"]] *= rng.uniform(0.5, 5); y2[IDX["Ca_SS"]] *= rng.uniform(0.5, 20)
        y2[IDX["Ca_SR"]] *= rng.uniform(0.5, 1.2); y2[IDX["Na_i"]] *= rng.uniform(0.8, 1.2)
        y3 = O3.tp06_rest()
        y3[0] = y2[0]
        for n3, n2 in ((9, "d"), (10, "f"), (11, "f2"), (12, "fCass"), (13, "Rprime"), (14, "Ca_i"), (15, "Ca_SR"),
                       (16, "Ca_SS"), (17, "Na_i"), (18, "K_i")):
            y3[n3] = y2[IDX[n2]]
        c2, c3 = O2.stw_currents(y2), O3.tp06_currents(y3, 0)
        for n in ("ICaL", "INaK", "INaCa", "IpCa", "IpK", "IbNa", "IbCa", "Irel", "Ileak", "Iup", "Ixfer"):
            assert c2[n] == pytest.approx(c3[n], rel=1e-13, abs=1e-300), n


def test_step_rush_larsen_forward_euler_and_ion_balances():
    """One step: gates by the Rush-Larsen closed form, R' and the five concentrations by forward Euler (reading B12), and
    the ion balances dNa_i = -(I_Na + I_bNa + I_fNa + 3 I_NaK + 3 I_NaCa) Cap/(V_c F),
    dK_i = -(I_K1 + I_to + I_fK + I_sus + I_Kr + I_Ks + I_pK + I_stim - 2 I_NaK) Cap/(V_c F)."""
    rng = np.random.default_rng(9)
    Cap, Vc = 0.185, 0.016404
    for _ in range(10):
        y = O2.stw_init()
        y[0] = rng.uniform(-85, 30)
        y[1:14] = rng.uniform(0.05, 0.95, 13)
        dt, istim, dvd = 0.01, -7.0, 3.0
        yn = O2.stw_step(y, dt, istim, dvd)
        inf, tau = O2.stw_gates(y[0], y[IDX["Ca_SS"]])
        assert np.allclose(yn[1:14], inf + (y[1:14] - inf) * np.exp(-dt / tau), rtol=1e-14, atol=0)
        c = O2.stw_currents(y)
        assert yn[0] == pytest.approx(y[0] + dt * (dvd - c["iion"] - istim), rel=1e-14)
        assert yn[IDX["Rprime"]] == pytest.approx(y[IDX["Rprime"]] + dt * c["dR"], rel=1e-15)
        dNa = -(c["INa"] + c["IbNa"] + c["IfNa"] + 3 * c["INaK"] + 3 * c["INaCa"]) * Cap / (Vc * F)
        dK = -(c["IK1"] + c["Ito"] + c["IfK"] + c["Isus"] + c["IKr"] + c["IKs"] + c["IpK"] + istim - 2 * c["INaK"]) * Cap / (Vc * F)
        assert yn[IDX["Na_i"]] - y[IDX["Na_i"]] == pytest.approx(dt * dNa, rel=1e-9)
        assert yn[IDX["K_i"]] - y[IDX["K_i"]] == pytest.approx(dt * dK, rel=1e-9)
    # ryanodine-receptor variable: dR'/dt = -k2 Ca_SS R' + k4 (1 - R'), k2 = 0.045 kcasr, k4 = 0.005; at Ca_SR = EC = 1.5
    # kcasr = 2.5 - 1.5/2 = 1.75
    y = _state(Ca_SR=1.5, Ca_SS=0.001, Rprime=0.5)
    assert O2.stw_currents(y)["dR"] == pytest.approx(-0.045 * 1.75 * 0.001 * 0.5 + 0.005 * 0.5, rel=1e-13)


def test_rush_larsen_closed_form_with_frozen_potential():
    """with v held constant N Rush-Larsen steps reproduce y_inf + (y0 - y_inf) e^{-N dt/tau} for any dt."""
    y0 = O2.stw_init()
    y0[0] = -30.0
    inf, tau = O2.stw_gates(-30.0, y0[IDX["Ca_SS"]])
    for dt, n in ((0.01, 500), (0.5, 10)):
        y, _ = O2.stw_run(y0, dt, n, freeze_v=True)
        for g in range(13):
            if O2.STW_GATES[g] == "fCass":
                continue                                   # its steady state follows Ca_SS, which moves
            want = inf[g] + (y0[1 + g] - inf[g]) * np.exp(-n * dt / tau[g])
            assert y[1 + g] == pytest.approx(want, rel=1e-10, abs=1e-13), O2.STW_GATES[g]


def test_automaticity_and_the_papers_plateau():
    """The Purkinje cell is auto-rhythmic (I_f): unstimulated it fires, again and again, about once a second, from a maximum
    diastolic potential near -75 mV.  PAPER.md:256: 'high peak of depolarization followed by a stable plateau phase of about
    250 ms'."""
    dt = 0.01
    y, tr = O2.stw_run(O2.stw_init(), dt, 300000, trace=True)           # 3 s, no stimulus
    up = np.nonzero((tr[:-1] <= 0) & (tr[1:] > 0))[0] * dt
    assert len(up) == 3, up
    assert 1000.0 < up[1] - up[0] < 1500.0 and abs((up[2] - up[1]) - (up[1] - up[0])) < 20.0
    assert -80.0 < tr.min() < -70.0 and 20.0 < tr.max() < 50.0
    # paced beat from the published initial state: peak, upstroke, plateau length (time above -40 mV)
    y, tr = O2.stw_run(O2.stw_init(), dt, 60000, istim=-52.0, n_on=0, n_off=100, trace=True)
    assert 35.0 < tr.max() < 55.0                                        # "high peak"
    assert np.diff(tr).max() / dt > 250.0                                # fast sodium upstroke, mV/ms
    plateau = (tr > -40.0).sum() * dt
    assert 220.0 < plateau < 300.0, plateau                              # "about 250 ms"
    # first order in time
    ref, _ = O2.stw_run(O2.stw_init(), 0.0025, 40000, istim=-52.0, n_on=0, n_off=400)
    e = []
    for dt2 in (0.02, 0.01):
        n = int(round(100.0 / dt2))
        yy, _ = O2.stw_run(O2.stw_init(), dt2, n, istim=-52.0, n_on=0, n_off=int(round(1.0 / dt2)))
        e.append(abs(yy[0] - ref[0]))
    assert 1.6 < e[0] / e[1] < 2.6, e


def test_published_initial_state_recurs_after_one_spontaneous_cycle():
    """The 20 published initial values are a point of the model's own limit cycle (they were taken from a converged
    spontaneous rhythm): integrating the equations as transcribed, unstimulated, the trajectory comes back through
    V = -69.137 mV (rising, in diastole) one cycle later with EVERY state variable within 0.1 % of its published initial
    value (gates near 0 within 1e-5 absolute).  A wrong constant anywhere moves the cycle away from the published point, so
    this ties the equations (DESIGN.md Appendix C, recalled from the published model) to 20 numbers of the publication."""
    y0 = O2.stw_init()
    dt = 0.01
    _, tr = O2.stw_run(y0, dt, 140000, trace=True)
    hits = np.nonzero((tr[:-1] <= y0[0]) & (tr[1:] > y0[0]))[0]
    hits = hits[hits > 50000]                               # the return after one cycle, not the start
    assert len(hits) == 1 and 1150.0 < hits[0] * dt < 1300.0, hits * dt
    y, _ = O2.stw_run(y0, dt, int(hits[0]) + 1)
    assert np.allclose(y, y0, rtol=1e-3, atol=1e-5), np.abs(y / y0 - 1).max()
    assert abs((tr[hits[0] + 1] - tr[hits[0]]) / dt - 0.01526) < 2e-4     # diastolic slope, mV/ms: the same point of the cycle
