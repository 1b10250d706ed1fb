"""Pins for the oracle's Courtemanche-Ramirez-Nattel atrial cell model (config 5).

The equations are not in PAPER.md (ref [1]); what fixes them here: the counts the paper prints (21 states,
15 Rush-Larsen gates), its stated facts (rest about -80 mV, repolarisation of about 200 ms),
half-activation points and limits that can be read off the published formulas, the removable singularities' limits,
reversal potentials, ion-conservation identities that tie every current to its concentration equation (a wrong volume,
valence or sign fails them), the Rush-Larsen closed form, and first-order convergence in dt.
"""
import numpy as np
import pytest

F, Vi, Vup, Vrel, Cm = 96.4867, 13668.0, 1109.52, 96.48, 100.0
RTF = 8.3143 * 310.0 / F
NAMES = ["m", "h", "j", "oa", "oi", "ua", "ui", "xr", "xs", "d", "f", "fCa", "u", "v", "w"]


def test_counts_and_rest_state(oracle):
    y = oracle.crn_rest()
    assert y.size == 21 and len(NAMES) == 15
    assert abs(y[0] + 80.0) < 2.0                                 # "-80 mV"
    yf, tr = oracle.crn_run(y, 0.01, 100000, trace=True)          # 1 s unstimulated
    assert np.abs(tr + 81.2).max() < 0.1
    assert np.all(yf[1:16] >= 0) and np.all(yf[1:16] <= 1)


def test_half_points_limits_and_constants(oracle):
    g = lambda V, **k: dict(zip(NAMES, oracle.crn_gates(V, **k)[0]))
    t = lambda V, **k: dict(zip(NAMES, oracle.crn_gates(V, **k)[1]))
    assert abs(g(-20.47)["oa"] - 0.5) < 1e-14 and abs(g(-43.1)["oi"] - 0.5) < 1e-14
    assert abs(g(-30.3)["ua"] - 0.5) < 1e-14 and abs(g(99.45)["ui"] - 0.5) < 1e-14
    assert abs(g(-14.1)["xr"] - 0.5) < 1e-14 and abs(g(19.9)["xs"] - 2 ** -0.5) < 1e-14
    assert abs(g(-10.0)["d"] - 0.5) < 1e-14 and abs(g(-28.0)["f"] - 0.5) < 1e-14
    assert abs(g(40.0)["w"] - 0.5) < 1e-14
    assert abs(g(0.0, Cai=0.00035)["fCa"] - 0.5) < 1e-14
    assert abs(g(0.0, Fn=3.4175e-13)["u"] - 0.5) < 1e-12 and abs(g(0.0, Fn=6.835e-14)["v"] - 0.5) < 1e-12
    assert g(0.0, Fn=0.0)["u"] < 1e-100 and g(0.0, Fn=0.0)["v"] == 1.0       # closed release gate at rest
    assert g(0.0, Fn=1e-11)["u"] == 1.0 and g(0.0, Fn=1e-11)["v"] < 1e-100
    assert t(0.0)["u"] == 8.0 and t(0.0)["fCa"] == 2.0
    assert abs(t(0.0, Fn=0.0)["v"] - 1.91) < 1e-12 and abs(t(0.0, Fn=1e-11)["v"] - 4.0) < 1e-12
    # sodium inactivation: alpha = 0 above -40 mV, so h_inf = j_inf = 0 there; fully available at -120 mV
    assert g(-39.9)["h"] == 0.0 and g(10.0)["j"] == 0.0
    assert g(-120.0)["h"] > 0.999 and g(-120.0)["j"] > 0.999 and g(-120.0)["m"] < 1e-3 and g(30.0)["m"] > 0.99
    # oa and ua share their time constant; Q10 = 3 divides it
    assert t(-30.0)["oa"] == t(-30.0)["ua"]
    a = 0.65 / (np.exp(-(-30 + 10) / 8.5) + np.exp(-(-30 - 30) / 59.0)); b = 0.65 / (2.5 + np.exp((-30 + 82) / 17.0))
    assert abs(t(-30.0)["oa"] - 1 / (a + b) / 3.0) < 1e-13


def test_removable_singularities(oracle):
    """alpha_m(-47.13) = 3.2 and the other 0/0 points have their analytic limits; the functions are smooth across them."""
    t = lambda V: dict(zip(NAMES, oracle.crn_gates(V)[1]))
    g = lambda V: dict(zip(NAMES, oracle.crn_gates(V)[0]))
    bm = 0.08 * np.exp(47.13 / 11.0)
    assert abs(t(-47.13)["m"] - 1 / (3.2 + bm)) < 1e-15 and abs(g(-47.13)["m"] - 3.2 / (3.2 + bm)) < 1e-15
    axr, bxr = 0.0003 * 5.0, 7.3898e-5 * (-14.1 - 3.3328) / (np.exp((-14.1 - 3.3328) / 5.1237) - 1)
    assert abs(t(-14.1)["xr"] - 1 / (axr + bxr)) < 1e-12
    assert abs(t(19.9)["xs"] - 0.5 / (4e-5 * 17 + 3.5e-5 * 9)) < 1e-10
    assert abs(t(-10.0)["d"] - 1 / (0.035 * 6.24 * 2)) < 1e-13
    assert abs(t(7.9)["w"] - 6.0 / (5.0 * 1.3)) < 1e-13
    for V0, name in ((-47.13, "m"), (-14.1, "xr"), (3.3328, "xr"), (19.9, "xs"), (-10.0, "d"), (7.9, "w")):
        for eps in (3e-4, 1e-5, 1e-9):      # across the series threshold |x| = 1e-4
            lo, mid, hi = t(V0 - eps)[name], t(V0)[name], t(V0 + eps)[name]
            assert abs(lo + hi - 2 * mid) <= 1e-9 * abs(mid), (V0, name, eps)


def test_reversal_potentials_and_signs(oracle):
    y = oracle.crn_rest()
    EK, ENa = RTF * np.log(5.4 / y[17]), RTF * np.log(140.0 / y[16])
    ECa = 0.5 * RTF * np.log(1.8 / y[18])
    y[13] = 0.5                                   # open the release gate a little so that I_rel is exercised
    for V, keys in ((EK, ["IK1", "Ito", "IKur", "IKr", "IKs"]), (ENa, ["INa", "IbNa"]), (ECa, ["IbCa"]), (65.0, ["ICaL"])):
        yy = y.copy(); yy[0] = V
        c = oracle.crn_currents(yy)
        for k in keys:
            assert abs(c[k]) < 1e-12, (k, V)
    c = oracle.crn_currents(y)
    assert c["IK1"] > 0 and c["INaK"] > 0 and c["IbNa"] < 0 and c["IbCa"] < 0 and c["IpCa"] > 0 and c["ICaL"] < 0
    assert c["Irel"] > 0 and abs(sum(c[k] for k in oracle.CRN_CURRENTS[:12]) - c["iion"]) < 1e-15
    assert abs(c["Iup"] - c["Iupleak"]) < 2e-6   # SR uptake balances the leak at rest
    # sigma of the Na/K pump: (exp(Nao/67.3) - 1)/7
    yy = y.copy(); yy[0] = 0.0
    fnak = 1 / (1 + 0.1245 + 0.0365 * (np.exp(140 / 67.3) - 1) / 7)
    assert abs(oracle.crn_currents(yy)["INaK"] - 0.6 * fnak / (1 + (10.0 / yy[16]) ** 1.5) * 5.4 / 6.9) < 1e-15


def test_ion_conservation_identities(oracle):
    """One forward-Euler step: every concentration increment equals the currents that carry that ion; SR fluxes cancel."""
    rng_states = [oracle.crn_rest()]
    yb = oracle.crn_rest(); yb[0] = -10.0; yb[1:16] = 0.5; yb[18] = 8e-4; yb[19] = 1.8; yb[20] = 0.7
    rng_states.append(yb)
    dt = 1e-3
    for y in rng_states:
        c = oracle.crn_currents(y)
        yn, _ = oracle.crn_run(y, dt, 1)
        d = (yn - y) / dt
        assert abs(d[16] * F * Vi / Cm + (c["INa"] + c["IbNa"] + 3 * c["INaK"] + 3 * c["INaCa"])) < 1e-6   # (yn-y)/dt rounds at eps*y/dt
        assert abs(d[17] * F * Vi / Cm - (2 * c["INaK"] - c["IK1"] - c["Ito"] - c["IKur"] - c["IKr"] - c["IKs"])) < 1e-5
        Cai, Carel = y[18], y[20]
        B2 = 1 + 0.07 * 0.0005 / (Cai + 0.0005) ** 2 + 0.05 * 0.00238 / (Cai + 0.00238) ** 2
        Bsq = 1 + 10.0 * 0.8 / (Carel + 0.8) ** 2
        total = Vi * B2 * d[18] + Vup * d[19] + Vrel * Bsq * d[20]      # d/dt of total (free + buffered) calcium
        memb = Cm * (2 * c["INaCa"] - c["IpCa"] - c["ICaL"] - c["IbCa"]) / (2 * F)
        assert abs(total - memb) < 1e-6 * max(1.0, abs(memb))
        assert abs(d[0] + c["iion"]) < 1e-8                            # dV/dt = -i_ion without stimulus and diffusion


def test_rush_larsen_closed_form(oracle):
    y0 = oracle.crn_rest(); y0[0] = -25.0; y0[1:16] = np.linspace(0.05, 0.95, 15)
    inf, tau = oracle.crn_gates(y0[0], y0[18], oracle.crn_currents(y0)["Fn"])
    for dt, n in ((0.01, 100), (0.5, 2), (5.0, 1)):
        y = y0.copy()
        for _ in range(n):                       # V, Ca_i and the currents that set Fn frozen: only gates move
            yn, _ = oracle.crn_run(y, dt, 1, freeze_v=True)
            y[1:13] = yn[1:13]; y[15] = yn[15]
        idx = list(range(0, 11)) + [14]          # u, v (Fn moves with the gates) and fCa (Ca_i moves) are left out
        exact = inf + (y0[1:16] - inf) * np.exp(-n * dt / tau)
        assert np.abs(y[1:16][idx] - exact[idx]).max() < 1e-12
        assert np.all(y[1:16] >= 0) and np.all(y[1:16] <= 1)


def _apd(tr, dt, level):
    above = np.nonzero(tr > level)[0]
    return (above[-1] - above[0]) * dt


def test_action_potential_matches_paper_facts(oracle):
    """atrial rest of -80 mV and repolarisation after about 200 ms."""
    y = oracle.crn_rest()
    yf, tr = oracle.crn_run(y, 0.01, 50000, istim=-20.0, n_on=0, n_off=200, trace=True)
    assert 15.0 < tr.max() < 35.0                                   # overshoot
    assert 150.0 < np.diff(tr).max() / 0.01 < 300.0                 # upstroke velocity, mV/ms
    assert 150.0 < _apd(tr, 0.01, -40.0) < 260.0                    # "about 200 ms" to leave the plateau
    assert 280.0 < _apd(tr, 0.01, tr.max() - 0.9 * (tr.max() - tr[0])) < 330.0   # APD90
    assert abs(tr[-1] + 80.0) < 2.0                                 # back at rest
    # spike and dome: a notch after the spike, then a dome
    k_peak = tr.argmax()
    notch = tr[k_peak:k_peak + 3000].min()
    dome = tr[k_peak + 1500:k_peak + 8000].max()
    assert notch < dome - 1.0 and notch < tr.max() - 20.0


def test_first_order_in_time(oracle):
    y = oracle.crn_rest()
    ref, _ = oracle.crn_run(y, 0.00125, 16000, istim=-20.0, n_on=0, n_off=1600)
    errs = []
    for dt in (0.02, 0.01, 0.005):
        n = int(round(20.0 / dt))
        yf, _ = oracle.crn_run(y, dt, n, istim=-20.0, n_on=0, n_off=int(round(2.0 / dt)))
        errs.append(abs(yf[0] - ref[0]))
    assert 1.6 < errs[0] / errs[1] < 2.6 and 1.6 < errs[1] / errs[2] < 2.8     # first order


def test_tissue_step_uses_crn(oracle):
    """orc_state_init(model=1) + orc_step: an uncoupled single tet reproduces the single-cell run bit for bit."""
    from ep_inputs import meshes as M
    m = M.TetMesh(np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1.0]]), np.array([[0, 1, 2, 3]], np.int32))
    s = oracle.OracleSim(m.xyz, m.tets)
    s.state_init(1, None)
    assert s.n_states == 21
    s.stimulus_set(0, np.array([0]), -20.0, 0.0, 2.0)
    s.step(500, 0.01)
    yf, _ = oracle.crn_run(oracle.crn_rest(), 0.01, 500, istim=-20.0, n_on=0, n_off=200)
    got = np.array([s.read_state(k)[0] for k in range(21)])
    assert np.array_equal(got, yf)
