"""Mutation check of the oracle's pins: does a plausible transcription mistake in oracle/ep_oracle.cpp fail a pin?

Each mutant is a copy of the oracle source with ONE edit (a changed constant, a swapped index, a dropped term, a flipped
sign), compiled to a temporary library; the oracle pin files are then run against it in a subprocess
(EP_ORACLE_LIB points oracle/ep_oracle.py at the mutant).  A mutant is "killed" if pytest fails.  The list holds the
seven mutants that survived the round-1 pins (tau_xr1 slope, alpha_j exponent, tau_d slope, the I_K1 0.06
factor, G_Kr, tau_xs 1400, V_maxup), the alpha_c1/alpha_c2 swap of reading A6, and one or more edits of every group of
constants of both cell models and of every stage of the Fig. 8 pipeline.  Required: every mutant killed by the fast pins
(no tissue run needed), i.e. by values fixed outside the oracle.
"""
import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "ep_oracle.cpp")

TP06_PINS = ["tests/test_oracle_tp06_values.py", "tests/test_oracle_tp06.py"]
CRN_PINS = ["tests/test_oracle_crn_values.py", "tests/test_oracle_crn.py"]
FV_PINS = ["tests/test_oracle_fv.py"]
STEP_PINS = ["tests/test_oracle_step.py"]

# (name, text to find -- must occur exactly once --, replacement, pin files)
MUTANTS = [
    # --- the seven round-1 survivors and the alpha swap
    ("tau_xr1 slope 11.5 -> 10.5", "sig((v + 30.0) / 11.5)", "sig((v + 30.0) / 10.5)", TP06_PINS),
    ("alpha_j exponent 0.2444 -> 0.2144", "aj = (-2.5428e4 * std::exp(0.2444 * v)", "aj = (-2.5428e4 * std::exp(0.2144 * v)", TP06_PINS),
    ("tau_d slope 13 -> 15", "sig((-35.0 - v) / 13.0)", "sig((-35.0 - v) / 15.0)", TP06_PINS),
    ("I_K1 0.06 -> 0.07", "std::exp(0.06 * (v - E_K - 200.0))", "std::exp(0.07 * (v - E_K - 200.0))", TP06_PINS),
    ("G_Kr +12 %", "G_Kr = 0.153,", "G_Kr = 0.171,", TP06_PINS),
    ("tau_xs 1400 -> 1100", "tau[5] = 1400.0 /", "tau[5] = 1100.0 /", TP06_PINS),
    ("V_maxup -16 %", "V_maxup = 0.006375", "V_maxup = 0.005355", TP06_PINS),
    ("alpha_c1 / alpha_c2 swapped (A6)", "f.a1 = d2 / (d1 + d2);", "f.a1 = d1 / (d1 + d2);", FV_PINS),
    # --- TP06 gates
    ("h beta exponent 0.3485 -> 0.3385", "3.1e5 * std::exp(0.3485 * v)", "3.1e5 * std::exp(0.3385 * v)", TP06_PINS),
    ("m_inf slope 9.03 -> 9.3", "(-56.86 - v) / 9.03", "(-56.86 - v) / 9.3", TP06_PINS),
    ("tau_m 35 -> 30", "0.1 * sig((v + 35.0) / 5.0)", "0.1 * sig((v + 30.0) / 5.0)", TP06_PINS),
    ("tau_m 200 -> 100", "sig((v - 50.0) / 200.0)", "sig((v - 50.0) / 100.0)", TP06_PINS),
    ("alpha_h 0.057 -> 0.075", "ah = 0.057 * std::exp", "ah = 0.075 * std::exp", TP06_PINS),
    ("beta_j high 0.6 -> 0.3", "bj = 0.6 * std::exp(0.057 * v)", "bj = 0.3 * std::exp(0.057 * v)", TP06_PINS),
    ("beta_j low 0.02424 -> 0.1212", "bj = 0.02424 * std::exp", "bj = 0.1212 * std::exp", TP06_PINS),
    ("alpha_j 37.78 -> 37.87", "* (v + 37.78)\n               / (1.0 + std::exp(0.311 * (v + 79.23)));\n          bj = 0.02424",
     "* (v + 37.87)\n               / (1.0 + std::exp(0.311 * (v + 79.23)));\n          bj = 0.02424", TP06_PINS),
    ("tau_xr1 450 -> 540", "tau[3] = 450.0 *", "tau[3] = 540.0 *", TP06_PINS),
    ("tau_xr2 1.12 -> 1.21", "* 1.12 * sig((v - 60.0) / 20.0)", "* 1.21 * sig((v - 60.0) / 20.0)", TP06_PINS),
    ("xr2_inf slope 24 -> 20", "inf[4] = sig((v + 88.0) / 24.0)", "inf[4] = sig((v + 88.0) / 20.0)", TP06_PINS),
    ("tau_xs sqrt slope 6 -> 5", "std::exp((5.0 - v) / 6.0)", "std::exp((5.0 - v) / 5.0)", TP06_PINS),
    ("tau_r width 1800 -> 1500", "(v + 40.0) / 1800.0", "(v + 40.0) / 1500.0", TP06_PINS),
    ("tau_s epi width 320 -> 230", "(v + 45.0) / 320.0", "(v + 45.0) / 230.0", TP06_PINS),
    ("tau_s endo 1000 width", "(v + 67.0) / 1000.0", "(v + 67.0) / 1100.0", TP06_PINS),
    ("tau_d 1.4 -> 1.2 (second factor)", "* (1.4 * sig((v + 5.0) / 5.0))", "* (1.2 * sig((v + 5.0) / 5.0))", TP06_PINS),
    ("tau_f 200 -> 100", "200.0 * sig((13.0 - v) / 10.0)", "100.0 * sig((13.0 - v) / 10.0)", TP06_PINS),
    ("tau_f width 225 -> 240", "(v + 27.0) / 225.0", "(v + 27.0) / 240.0", TP06_PINS),
    ("tau_f2 562 -> 600 (published text vs released constants, B2)", "tau[10] = 562.0 *", "tau[10] = 600.0 *", TP06_PINS),
    ("tau_f2 31 -> 13", "31.0 * sig((25.0 - v) / 10.0)", "13.0 * sig((25.0 - v) / 10.0)", TP06_PINS),
    ("f2_inf 0.67 -> 0.76", "inf[10] = 0.67 * sig((v + 35.0) / 7.0) + 0.33", "inf[10] = 0.76 * sig((v + 35.0) / 7.0) + 0.24", TP06_PINS),
    ("fCass tau 80 -> 60", "tau[11] = 80.0 / q + 2.0", "tau[11] = 60.0 / q + 2.0", TP06_PINS),
    ("Rbar: k2' 0.045 -> 0.054", "k2p = 0.045", "k2p = 0.054", TP06_PINS),
    ("Rbar: max_sr 2.5 -> 2.0", "max_sr = 2.5", "max_sr = 2.0", TP06_PINS),
    # --- TP06 currents and concentrations
    ("G_Na 14.838 -> 14.388", "G_Na = 14.838", "G_Na = 14.388", TP06_PINS),
    ("G_K1 5.405 -> 5.045", "G_K1 = 5.405", "G_K1 = 5.045", TP06_PINS),
    ("G_to endo 0.073 -> 0.037", "(type == 0) ? 0.073 : 0.294", "(type == 0) ? 0.037 : 0.294", TP06_PINS),
    ("G_Ks mid on the wrong type", "(type == 1) ? 0.098 : 0.392", "(type == 2) ? 0.098 : 0.392", TP06_PINS),
    ("G_pK 0.0146 -> 0.0164", "G_pK = 0.0146", "G_pK = 0.0164", TP06_PINS),
    ("I_pK slope 5.98 -> 5.89", "(25.0 - v) / 5.98", "(25.0 - v) / 5.89", TP06_PINS),
    ("G_pCa 0.1238 -> 0.1328", "G_pCa = 0.1238", "G_pCa = 0.1328", TP06_PINS),
    ("G_bNa 2.9e-4 -> 2.9e-3", "G_bNa = 2.9e-4", "G_bNa = 2.9e-3", TP06_PINS),
    ("G_bCa 5.92e-4 -> 5.29e-4", "G_bCa = 5.92e-4", "G_bCa = 5.29e-4", TP06_PINS),
    ("p_KNa 0.03 -> 0.3", "p_KNa = 0.03", "p_KNa = 0.3", TP06_PINS),
    ("P_NaK 2.724 -> 2.274", "P_NaK = 2.724", "P_NaK = 2.274", TP06_PINS),
    ("I_NaK 0.0353 -> 0.0365 (the Courtemanche value)", "0.0353 * std::exp(-v / RTF)", "0.0365 * std::exp(-v / RTF)", TP06_PINS),
    ("K_mNa 40 -> 10", "K_mNa = 40.0", "K_mNa = 10.0", TP06_PINS),
    ("k_sat 0.1 -> 0.2", "k_sat = 0.1, gam", "k_sat = 0.2, gam", TP06_PINS),
    ("gamma 0.35 -> 0.5", "gam = 0.35, alp", "gam = 0.5, alp", TP06_PINS),
    ("I_NaCa alpha 2.5 -> 2.0", "alp = 2.5", "alp = 2.0", TP06_PINS),
    ("K_mCa 1.38 -> 1.83", "K_mCa = 1.38, k_sat", "K_mCa = 1.83, k_sat", TP06_PINS),
    ("I_K1 0.0002 -> 0.002", "3.0 * std::exp(0.0002 *", "3.0 * std::exp(0.002 *", TP06_PINS),
    ("I_K1 0.1(u-10) -> 0.1(u+10)", "std::exp(0.1 * (v - E_K - 10.0))", "std::exp(0.1 * (v - E_K + 10.0))", TP06_PINS),
    ("I_CaL: Ca_SS/4 -> Ca_SS", "(0.25 * Ca_SS * ex - Ca_o)", "(1.0 * Ca_SS * ex - Ca_o)", TP06_PINS),
    ("V_rel 0.102 -> 0.12", "V_rel = 0.102", "V_rel = 0.12", TP06_PINS),
    ("V_leak 3.6e-4 -> 3.6e-3", "V_leak = 3.6e-4", "V_leak = 3.6e-3", TP06_PINS),
    ("V_xfer 0.0038 -> 0.0083", "V_xfer = 0.0038", "V_xfer = 0.0083", TP06_PINS),
    ("k3 0.06 -> 0.006", "k3 = 0.060", "k3 = 0.006", TP06_PINS),
    ("k1' 0.15 -> 0.51", "k1p = 0.15", "k1p = 0.51", TP06_PINS),
    ("K_up 2.5e-4 -> 5e-4", "K_up = 2.5e-4", "K_up = 5e-4", TP06_PINS),
    ("Buf_c 0.2 -> 0.15", "Buf_c = 0.2", "Buf_c = 0.15", TP06_PINS),
    ("K_bufsr 0.3 -> 0.03", "K_bufsr = 0.3", "K_bufsr = 0.03", TP06_PINS),
    ("Buf_ss 0.4 -> 0.04", "Buf_ss = 0.4", "Buf_ss = 0.04", TP06_PINS),
    ("V_ss 5.468e-5 -> 5.648e-5", "V_ss = 0.00005468", "V_ss = 0.00005648", TP06_PINS),
    ("V_sr 0.001094 -> 0.001904", "V_sr = 0.001094", "V_sr = 0.001904", TP06_PINS),
    ("stimulus dropped from dK_i/dt (B8)", "c.IpK + istim) * Cap", "c.IpK) * Cap", TP06_PINS),
    ("I_NaCa stoichiometry in dNa_i 3 -> 1", "3.0 * c.INaK + 3.0 * c.INaCa) * Cap", "3.0 * c.INaK + 1.0 * c.INaCa) * Cap", TP06_PINS),
    ("Rush-Larsen written as forward Euler", "for (int g = 0; g < 13; ++g)  // Rush-Larsen, PAPER.md:174\n        yn[1 + g] = inf[g] + (y[1 + g] - inf[g]) * std::exp(-dt / tau[g]);",
     "for (int g = 0; g < 13; ++g)\n        yn[1 + g] = y[1 + g] + dt * (inf[g] - y[1 + g]) / tau[g];", TP06_PINS),
    ("sign of the stimulus in dv/dt", "yn[0] = y[0] + dt * (dv_diff - c.iion - istim);  // eq. (7)", "yn[0] = y[0] + dt * (dv_diff - c.iion + istim);  // eq. (7)", TP06_PINS),
    # --- Courtemanche
    ("CRN g_Na 7.8 -> 8.7", "gNa = 7.8", "gNa = 8.7", CRN_PINS),
    ("CRN g_K1 0.09 -> 0.9", "gK1 = 0.09", "gK1 = 0.9", CRN_PINS),
    ("CRN g_to 0.1652 -> 0.1562", "gto = 0.1652", "gto = 0.1562", CRN_PINS),
    ("CRN g_Kr 0.0294 -> 0.0249", "gKr = 0.0294", "gKr = 0.0249", CRN_PINS),
    ("CRN g_Ks 0.129 -> 0.192", "gKs = 0.129", "gKs = 0.192", CRN_PINS),
    ("CRN g_CaL 0.1238 -> 0.1328", "gCaL = 0.1238", "gCaL = 0.1328", CRN_PINS),
    ("CRN g_Kur 0.05 -> 0.005", "0.005 + 0.05 / (1.0 + std::exp(-(V - 15.0) / 13.0))", "0.005 + 0.005 / (1.0 + std::exp(-(V - 15.0) / 13.0))", CRN_PINS),
    ("CRN I_K1 slope 0.07 -> 0.06", "std::exp(0.07 * (V + 80.0))", "std::exp(0.06 * (V + 80.0))", CRN_PINS),
    ("CRN I_Kr 22.4 -> 24.2", "(V + 15.0) / 22.4", "(V + 15.0) / 24.2", CRN_PINS),
    ("CRN I_NaCa,max 1600 -> 1000", "INaCamax = 1600.0", "INaCamax = 1000.0", CRN_PINS),
    ("CRN I_pCa,max 0.275 -> 0.257", "IpCamax = 0.275", "IpCamax = 0.257", CRN_PINS),
    ("CRN k_rel 30 -> 3", "krel = 30.0", "krel = 3.0", CRN_PINS),
    ("CRN K_up 0.00092 -> 0.0092", "Kup = 0.00092", "Kup = 0.0092", CRN_PINS),
    ("CRN tau_tr 180 -> 108", "tau_tr = 180.0", "tau_tr = 108.0", CRN_PINS),
    ("CRN K_Q10 3 -> 2", "KQ10 = 3.0", "KQ10 = 2.0", CRN_PINS),
    ("CRN beta_m 11 -> 10", "0.08 * std::exp(-V / 11.0)", "0.08 * std::exp(-V / 10.0)", CRN_PINS),
    ("CRN alpha_h 0.135 -> 0.153", "ah = 0.135 * std::exp", "ah = 0.153 * std::exp", CRN_PINS),
    ("CRN beta_h 3.56 -> 3.65", "bh = 3.56 * std::exp", "bh = 3.65 * std::exp", CRN_PINS),
    ("CRN beta_j high 0.3 -> 0.6 (the TP06 value)", "bj = 0.3 * std::exp(-2.535e-7 * V)", "bj = 0.6 * std::exp(-2.535e-7 * V)", CRN_PINS),
    ("CRN oa alpha 8.5 -> 5.8", "std::exp(-(V + 10.0) / 8.5)", "std::exp(-(V + 10.0) / 5.8)", CRN_PINS),
    ("CRN oi beta 35.56 -> 53.56", "1.0 / (35.56 + std::exp", "1.0 / (53.56 + std::exp", CRN_PINS),
    ("CRN ui alpha 21 -> 12", "1.0 / (21.0 + std::exp(-(V - 185.0) / 28.0))", "1.0 / (12.0 + std::exp(-(V - 185.0) / 28.0))", CRN_PINS),
    ("CRN xr beta 7.3898e-5 -> 7.3898e-4", "const double b = 7.3898e-5 * 5.1237", "const double b = 7.3898e-4 * 5.1237", CRN_PINS),
    ("CRN xs tau 0.5 -> 1", "tau[8] = 0.5 / (a + b)", "tau[8] = 1.0 / (a + b)", CRN_PINS),
    ("CRN xr_inf slope 6.5 -> 5.6", "std::exp(-(V + 14.1) / 6.5)", "std::exp(-(V + 14.1) / 5.6)", CRN_PINS),
    ("CRN tau_f 0.0197 -> 0.0179", "9.0 / (0.0197 * std::exp", "9.0 / (0.0179 * std::exp", CRN_PINS),
    ("CRN d_inf slope 8 -> 6.24", "inf[9] = 1.0 / (1.0 + std::exp(-(V + 10.0) / 8.0))", "inf[9] = 1.0 / (1.0 + std::exp(-(V + 10.0) / 6.24))", CRN_PINS),
    ("CRN tau_w 0.3 -> 0.03", "(1.0 + 0.3 * std::exp(x))", "(1.0 + 0.03 * std::exp(x))", CRN_PINS),
    ("CRN tau_v 2.09 -> 2.9", "1.91 + 2.09 / (1.0 + e1)", "1.91 + 2.9 / (1.0 + e1)", CRN_PINS),
    ("CRN Fn: 0.2 I_NaCa -> 0.5", "0.5 * Cm * c.ICaL - 0.2 * Cm * c.INaCa", "0.5 * Cm * c.ICaL - 0.5 * Cm * c.INaCa", CRN_PINS),
    ("CRN Trpn 0.07 -> 0.7", "Trpnmax = 0.07", "Trpnmax = 0.7", CRN_PINS),
    ("CRN V_up 1109.52 -> 1190.52", "Vup = 1109.52", "Vup = 1190.52", CRN_PINS),
    ("CRN Ca_up,max 15 -> 10", "Caupmax = 15.0", "Caupmax = 10.0", CRN_PINS),
    ("CRN K_m,Na(i) 10 -> 1", "KmNai = 10.0", "KmNai = 1.0", CRN_PINS),
    # --- finite-volume pipeline
    ("A8: harmonic instead of arithmetic M_f (xx only)", "f.Mf = {f.a1 * A.xx + f.a2 * B.xx,", "f.Mf = {1.0 / (f.a1 / A.xx + f.a2 / B.xx),", FV_PINS),
    ("A2: uniform node weights instead of 1/d", "s.star_invd[p] = 1.0 / norm(s.x[n] - s.xc[c]);", "s.star_invd[p] = 1.0;", FV_PINS),
    ("A2: 1/d^2 node weights", "s.star_invd[p] = 1.0 / norm(s.x[n] - s.xc[c]);", "s.star_invd[p] = 1.0 / dot(s.x[n] - s.xc[c], s.x[n] - s.xc[c]);", FV_PINS),
    ("face value = mean of 3 nodes -> /4", "vn[t[FACE_NODES[j][2]]]) / 3.0;", "vn[t[FACE_NODES[j][2]]]) / 4.0;", FV_PINS),
    ("eq. (8) correction with the wrong sign of e", "f.d = norm(dc); f.e = (1.0 / f.d) * dc;", "f.d = norm(dc); f.e = (-1.0 / f.d) * dc;", FV_PINS),
    ("eq. (8): d_c1c2 replaced by d1 + d2", "f.d = norm(dc); f.e = (1.0 / f.d) * dc;", "f.d = d1 + d2; f.e = (1.0 / norm(dc)) * dc;", FV_PINS),
    ("unit factor 100 dropped", "D[c] = 100.0 * acc / s.vol[c];", "D[c] = acc / s.vol[c];", FV_PINS),
    ("tensor: sigma_l and sigma_t exchanged", "const double dl = slc - stc;", "const double dl = stc - slc; stc = slc;", FV_PINS),
    ("face area vector without the 1/2", "Vec3 sv = 0.5 * cross(b - a, cc - a);", "Vec3 sv = 1.0 * cross(b - a, cc - a);", FV_PINS),
    ("boundary faces carry the one-sided flux", "if (id < 0) continue;                                  // no-flux boundary",
     "if (id < 0) { acc += dot(mul(s.Mc[c], s.grad[c]), s.sf[c * 4 + j]); continue; }", FV_PINS),
    # --- time stepping, stimulus windows, activation, trigger (readings A16-A18)
    ("A16: stimulus window closed interval", "on[k] = (n_on <= n && n < n_off);", "on[k] = (n_on <= n && n <= n_off);", STEP_PINS),
    ("A18: activation at n dt instead of (n+1) dt", "s.tact[c] = (double)(n + 1) * dt;", "s.tact[c] = (double)(n) * dt;", STEP_PINS),
    ("A18: threshold -10 mV", "if (s.tact[c] < 0.0 && y[0] <= 0.0 && yn[0] > 0.0)", "if (s.tact[c] < 0.0 && y[0] <= -10.0 && yn[0] > -10.0)", STEP_PINS),
    ("A13: diffusion scaled by 1/chi only", "const double inv_chiCm = 1.0 / (s.chi * s.Cm);", "const double inv_chiCm = 1.0 / (s.chi);", STEP_PINS),
    ("stimulus not divided by C_m", "tp06_step(y, s.ctype[c], dt, Is / s.Cm,", "tp06_step(y, s.ctype[c], dt, Is,", STEP_PINS),
    ("Jacobi update replaced by in-place use of new v (node values from yn)", "apply_diffusion(s, s.y.data(), s.D.data(), 1);   // state 0 is v",
     "apply_diffusion(s, it > 0 ? s.yn.data() : s.y.data(), s.D.data(), 1);", STEP_PINS),
    ("trigger delay ignored", "n >= g.n_fire1 + nd && n < g.n_fire1 + nd + ndur;", "n >= g.n_fire1 && n < g.n_fire1 + ndur;", STEP_PINS),
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
    env = dict(os.environ, EP_ORACLE_LIB=lib)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider", "-m", "not gpu and not slow_pin"]
                       + pins, cwd=ROOT, env=env, capture_output=True, text=True)
    return name, ("killed" if r.returncode == 1 else ("survived" if r.returncode == 0 else "error rc=%d %s" % (r.returncode, r.stdout[-300:])))


def test_pins_kill_single_edit_mutants(capsys):
    if os.environ.get("EP_ORACLE_LIB"):
        pytest.skip("running inside a mutant")
    src = open(SRC).read()
    with tempfile.TemporaryDirectory() as tmp:
        # the unmutated source must pass the same pin files through the same route
        ok = _run_mutant((999, ("identity", "// ep_oracle.cpp -- CPU ORACLE.", "// ep_oracle.cpp -- CPU ORACLE (copy).",
                                TP06_PINS + CRN_PINS + FV_PINS + STEP_PINS), src, tmp))
        assert ok[1] == "survived", ok
        jobs = [(i, m, src, tmp) for i, m in enumerate(MUTANTS)]
        with ThreadPoolExecutor(max_workers=max(1, (os.cpu_count() or 2))) as ex:
            res = list(ex.map(_run_mutant, jobs))
    bad = [r for r in res if r[1].startswith("bad-mutant") or r[1].startswith("error")]
    survived = [r[0] for r in res if r[1] == "survived"]
    with capsys.disabled():
        print("\noracle mutants: %d, killed %d, survived %d %s" % (len(res), sum(r[1] == "killed" for r in res),
                                                                   len(survived), survived))
    assert not bad, bad
    assert len(MUTANTS) >= 100
    assert not survived, survived
