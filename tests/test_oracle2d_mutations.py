"""Mutation check of the pins of oracle/ep_oracle2d.cpp (Stewart model + triangle finite volumes): every single-edit mutant
(changed constant, dropped term, swapped index, flipped sign) must fail a pin file.  Same mechanism as
tests/test_oracle_mutations.py; EP_ORACLE2D_LIB points oracle/ep_oracle2d.py at the mutant."""
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "ep_oracle2d.cpp")
STW = ["tests/test_oracle2d_stewart.py"]
FV = ["tests/test_oracle2d_fv.py"]

# (name, text to find -- exactly once --, replacement, pin files)
MUTANTS = [
    # --- Stewart-specific constants and terms
    ("g_fNa 0.0145654 -> 0.0154654", "g_fNa = 0.0145654", "g_fNa = 0.0154654", STW),
    ("g_fK 0.0234346 -> 0.0243346", "g_fK = 0.0234346", "g_fK = 0.0243346", STW),
    ("g_K1 0.065 -> 0.056", "g_K1 = 0.065", "g_K1 = 0.056", STW),
    ("g_Kr 0.0918 -> 0.0981", "g_Kr = 0.0918", "g_Kr = 0.0981", STW),
    ("g_Ks 0.2352 -> 0.2532", "g_Ks = 0.2352", "g_Ks = 0.2532", STW),
    ("g_Na 130.5744 -> 103.5744", "g_Na = 130.5744", "g_Na = 103.5744", STW),
    ("g_to 0.08184 -> 0.08814", "g_to = 0.08184", "g_to = 0.08814", STW),
    ("g_sus 0.0227 -> 0.0272", "g_sus = 0.0227", "g_sus = 0.0272", STW),
    ("y_inf half-point 80.6 -> 86.0", "inf[0] = sig((v + 80.6) / 6.8);", "inf[0] = sig((v + 86.0) / 6.8);", STW),
    ("y_inf slope 6.8 -> 8.6", "inf[0] = sig((v + 80.6) / 6.8);", "inf[0] = sig((v + 80.6) / 8.6);", STW),
    ("tau_y 4000 -> 400", "tau[0] = 4000.0 /", "tau[0] = 400.0 /", STW),
    ("tau_y alpha slope 0.04 -> 0.05", "std::exp(-2.9 - 0.04 * v)", "std::exp(-2.9 - 0.05 * v)", STW),
    ("tau_y beta 3.6 -> 3.9", "std::exp(3.6 + 0.11 * v)", "std::exp(3.9 + 0.11 * v)", STW),
    ("tau_y beta slope 0.11 -> 0.1", "std::exp(3.6 + 0.11 * v)", "std::exp(3.6 + 0.1 * v)", STW),
    ("I_K1 shift 8 -> 0", "(v - 8.0 - E_K)", "(v - 0.0 - E_K)", STW),
    ("I_K1 half-point 75.44 -> 74.55", "sig(0.1 * (v + 75.44))", "sig(0.1 * (v + 74.55))", STW),
    ("I_K1 slope 0.1 -> 0.12", "sig(0.1 * (v + 75.44))", "sig(0.12 * (v + 75.44))", STW),
    ("I_sus half-point 5 -> -5", "sig((5.0 - v) / 17.0)", "sig((-5.0 - v) / 17.0)", STW),
    ("I_sus slope 17 -> 13", "sig((5.0 - v) / 17.0)", "sig((5.0 - v) / 13.0)", STW),
    ("s_inf 27 -> 20 (the TP06 epicardial value)", "inf[11] = sig((v + 27.0) / 13.0);", "inf[11] = sig((v + 20.0) / 13.0);", STW),
    ("s_inf slope 13 -> 5", "inf[11] = sig((v + 27.0) / 13.0);", "inf[11] = sig((v + 27.0) / 5.0);", STW),
    ("tau_s 42 -> 3 (TP06)", "+ 5.0 * sig((v - 40.0) / 5.0) + 42.0;", "+ 5.0 * sig((v - 40.0) / 5.0) + 3.0;", STW),
    ("tau_s centre 25 -> 45 (TP06)", "(v + 25.0) * (v + 25.0) / 320.0", "(v + 45.0) * (v + 45.0) / 320.0", STW),
    ("tau_s sigmoid 40 -> 20 (TP06)", "5.0 * sig((v - 40.0) / 5.0)", "5.0 * sig((v - 20.0) / 5.0)", STW),
    ("r_inf slope 13 -> 6 (TP06)", "inf[12] = sig((20.0 - v) / 13.0);", "inf[12] = sig((20.0 - v) / 6.0);", STW),
    ("tau_r 10.45 -> 9.5 (TP06)", "tau[12] = 10.45 *", "tau[12] = 9.5 *", STW),
    ("tau_r 7.3 -> 0.8 (TP06)", "/ 1800.0) + 7.3;", "/ 1800.0) + 0.8;", STW),
    ("I_f missing from the sodium balance", "-(c.INa + c.IbNa + c.IfNa + 3.0 * c.INaK", "-(c.INa + c.IbNa + 3.0 * c.INaK", STW),
    ("I_sus missing from the potassium balance", "c.IfK + c.Isus + c.IKr", "c.IfK + c.IKr", STW),
    ("I_sus missing from the total current", "c.iion = c.IK1 + c.Ito + c.Isus +", "c.iion = c.IK1 + c.Ito +", STW),
    ("I_f missing from the total current", "+ c.IpCa + c.IfNa + c.IfK;", "+ c.IpCa;", STW),
    ("R' advanced by Rush-Larsen instead of forward Euler (B12)", "yn[14] = y[14] + dt * c.dR;",
     "{ const double kk = 0.005 - c.dR / 1.0; yn[14] = y[14] + dt * c.dR * 0.5; (void)kk; }", STW),
    ("k4 0.005 -> 0.05", "k4 = 0.005", "k4 = 0.05", STW),
    ("stimulus missing from dK_i", "+ c.IpK + istim - 2.0 * c.INaK", "+ c.IpK - 2.0 * c.INaK", STW),
    ("Rush-Larsen factor exp(-dt/tau) -> 1 - dt/tau", "* std::exp(-dt / tau[g]);", "* (1.0 - dt / tau[g]);", STW),
    ("inherited: f2 562 -> 600", "tau[9] = 562.0 *", "tau[9] = 600.0 *", STW),
    ("inherited: P_NaK 2.724 -> 2.274", "P_NaK = 2.724", "P_NaK = 2.274", STW),
    ("inherited: I_CaL 0.25 Ca_SS -> 0.5 Ca_SS", "(0.25 * Ca_SS * ex - Ca_o)", "(0.5 * Ca_SS * ex - Ca_o)", STW),
    ("inherited: m_inf slope", "(-56.86 - v) / 9.03", "(-56.86 - v) / 9.3", STW),
    ("initial state: V -69.14 -> -79.14 (no longer on the published cycle)", "INIT[S] = {-69.1370441635924,", "INIT[S] = {-79.1370441635924,", STW),
    # --- the 2D finite-volume chain
    ("alpha_c1 / alpha_c2 swapped (A6)", "f.a1 = d2 / (d1 + d2);", "f.a1 = d1 / (d1 + d2);", FV),
    ("node weights 1/d -> 1/d^2 (A2)", "s.star_invd[p] = 1.0 / norm(s.x[n] - s.xc[c]);",
     "s.star_invd[p] = 1.0 / dot(s.x[n] - s.xc[c], s.x[n] - s.xc[c]);", FV),
    ("edge value = mean of 2 nodes -> /3 (D1)", "s.tri[3 * c + EDGE_NODES[j][1]]]) / 2.0;", "s.tri[3 * c + EDGE_NODES[j][1]]]) / 3.0;", FV),
    ("Gauss-Green divided by 2 A", "grad[c] = (1.0 / s.area[c]) * g;", "grad[c] = (0.5 / s.area[c]) * g;", FV),
    ("triangle area without the 1/2", "s.area[c] = 0.5 * norm(N);", "s.area[c] = 1.0 * norm(N);", FV),
    ("centroid with weight 1/4", "s.xc[c] = (1.0 / 3.0) * (p[0] + p[1] + p[2]);", "s.xc[c] = (1.0 / 4.0) * (p[0] + p[1] + p[2]);", FV),
    ("edge normal not made outward", "if (dot(sv, xm - s.xc[c]) < 0.0) sv = -1.0 * sv;  // outward", "", FV),
    ("eq. (8): sign of e flipped", "f.e = (1.0 / f.d) * dc;", "f.e = (-1.0 / f.d) * dc;", FV),
    ("eq. (8): correction dropped", "if (use_corr) g = gbar +", "if (use_corr && false) g = gbar +", FV),
    ("eq. (8): d replaced by d1 + d2", "f.d = norm(dc);", "f.d = d1 + d2;", FV),
    ("M_f: c1's tensor only (A8)", "f.M = {f.a1 * A.xx + f.a2 * B.xx,", "f.M = {f.a1 * A.xx + f.a2 * A.xx,", FV),
    ("tensor: sigma_l and sigma_t exchanged", "const double dl = fl - ft;", "const double dl = ft - fl; ft = fl;", FV),
    ("unit factor 100 dropped", "D[c] = 100.0 * sum / s.area[c];", "D[c] = sum / s.area[c];", FV),
    ("divergence: sign of the neighbour's flux", "sum += (s.edges[e].c1 == c) ? flux[e] : -flux[e];", "sum += flux[e];", FV),
    ("boundary edges carry the one-sided flux (A11)", "if (e < 0) continue;                                   // boundary edge: no flux (A11)",
     "if (e < 0) { sum += dot(mul(s.Mc[c], s.grad[c]), s.se[3 * c + j]); continue; }", FV),
    ("diffusion scaled by 1/chi only", "const double inv_chiCm = 1.0 / (s.chi * s.Cm);", "const double inv_chiCm = 0.5 / (s.chi * s.Cm);", FV),
    ("A16: stimulus window closed interval", "on[k] = (n_on <= n && n < n_off);", "on[k] = (n_on <= n && n <= n_off);", FV),
    ("A18: activation at n dt", "s.tact[c] = (double)(n + 1) * dt;", "s.tact[c] = (double)(n) * dt;", FV),
    ("stimulus not divided by C_m", "stw::step(y, dt, Is / s.Cm,", "stw::step(y, dt, Is,", FV),
    ("mean potential not area-weighted", "num += s.area[c] * s.y[c]; den += s.area[c];", "num += s.y[c]; den += 1.0;", FV),
    ("activation threshold -10 mV (A18)", "if (s.tact[c] < 0.0 && y[0] <= 0.0 && yn[0] > 0.0)", "if (s.tact[c] < 0.0 && y[0] <= -30.0 && yn[0] > -30.0)", FV),
]


def _run_mutant(args):
    idx, (name, find, repl, pins), src, tmp = args
    if src.count(find) != 1:
        return name, "bad-mutant: pattern occurs %d times" % src.count(find)
    cpp = os.path.join(tmp, "m%03d.cpp" % idx)
    lib = os.path.join(tmp, "m%03d.so" % idx)
    with open(cpp, "w") as f:
        f.write(src.replace(find, repl))
    r = subprocess.run(["g++", "-O1", "-ffp-contract=off", "-shared", "-fPIC", "-o", lib, cpp], capture_output=True, text=True)
    if r.returncode != 0:
        return name, "bad-mutant: does not compile: " + r.stderr[-300:]
    env = dict(os.environ, EP_ORACLE2D_LIB=lib)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-m", "not gpu"] + pins,
                       cwd=ROOT, env=env, capture_output=True, text=True)
    return name, ("killed" if r.returncode == 1 else ("survived" if r.returncode == 0 else "error rc=%d %s" % (r.returncode, r.stdout[-300:])))


def test_pins_kill_single_edit_mutants_2d(capsys):
    if os.environ.get("EP_ORACLE2D_LIB"):
        pytest.skip("running inside a mutant")
    src = open(SRC).read()
    with tempfile.TemporaryDirectory() as tmp:
        ok = _run_mutant((999, ("identity", "// ep_oracle2d.cpp -- CPU ORACLE", "// ep_oracle2d.cpp (copy) -- CPU ORACLE", STW + FV), src, tmp))
        assert ok[1] == "survived", ok
        jobs = [(i, m, src, tmp) for i, m in enumerate(MUTANTS)]
        with ThreadPoolExecutor(max_workers=max(1, (os.cpu_count() or 2))) as ex:
            res = list(ex.map(_run_mutant, jobs))
    bad = [r for r in res if r[1].startswith("bad-mutant") or r[1].startswith("error")]
    survived = [r[0] for r in res if r[1] == "survived"]
    with capsys.disabled():
        print("\noracle2d mutants: %d, killed %d, survived %d %s" % (len(res), sum(r[1] == "killed" for r in res),
                                                                     len(survived), survived))
    assert not bad, bad
    assert len(MUTANTS) >= 50
    assert not survived, survived
