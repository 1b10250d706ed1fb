"""Step-level pins of the oracle's tissue time step (orc_step): what is fixed outside its own code.

Stimulus windows on integer steps (reading A16), the activation rule (A18), the explicit update
v^{n+1} = v^n + dt [D_c/(chi C_m) - i_ion - I_s/C_m] (eq. (7)) with its unit factors, the Jacobi
(all-from-t^n) update of PAPER.md:176, and the communication-node trigger.  The expected values come
from hand-chosen integer step indices, the hand-worked two-tet flux of tests/golden/two_tet_flux.json and single-cell
runs driven with explicitly given step indices.
"""
import json
import os

import numpy as np
import pytest

TWO = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "two_tet_flux.json")))


def _two_tet(oracle, scale, chi=1400.0, Cm=1.0):
    g = TWO["case_A"]
    return oracle.OracleSim(np.array(TWO["nodes"], float), np.array(g["tets"], np.int32), None, np.asarray(scale, float),
                            g["sigma_l"], g["sigma_t"], chi, Cm)


def test_stimulus_window_is_half_open_on_integer_steps(oracle):
    """Reading A16: 1 ms at dt = 0.02 ms from t = 0.3 ms is exactly the 50 steps n = 15..64.  An uncoupled cell (sigma
    scale 0) must follow the single-cell run that is told those indices explicitly."""
    s = _two_tet(oracle, [0.0, 0.0])
    s.state_init(0, None)
    s.stimulus_set(0, np.array([1]), -52.0, 0.3, 1.0)
    s.step(200, 0.02)
    y_ref, _ = oracle.tp06_run(oracle.tp06_rest(), 0, 0.02, 200, istim=-52.0, n_on=15, n_off=65)
    assert np.array_equal(np.array([s.read_state(k)[1] for k in range(19)]), y_ref)
    y_rest, _ = oracle.tp06_run(oracle.tp06_rest(), 0, 0.02, 200)
    assert np.array_equal(np.array([s.read_state(k)[0] for k in range(19)]), y_rest)      # cell 0 is not in the slot


def test_explicit_update_units_and_hand_flux(oracle):
    """Eq. (7): the coupled step differs from the uncoupled one by exactly dt D_c/(chi C_m), with D_c the hand-worked
    -548.132... / +274.066... uA/cm^3 of the two-tet mesh (v = 1, 0 mV), chi = 1400 /cm, C_m = 2 uF/cm^2; and a stimulus
    of -52 uA/cm^2 moves an uncoupled cell by -dt I_s/C_m = +26 dt mV more than an unstimulated one."""
    dt, chi, Cm = 0.01, 1400.0, 2.0
    D = np.array(TWO["case_A"]["D"])
    out = {}
    for name, scale, stim in (("coupled", TWO["sigma_scale"], False), ("free", [0.0, 0.0], False), ("stim", [0.0, 0.0], True)):
        s = _two_tet(oracle, scale, chi, Cm)
        s.state_init(0, None)
        s.write_state(0, np.array(TWO["v"]))
        if stim:
            s.stimulus_set(0, np.array([0, 1]), -52.0, 0.0, 1.0)
        s.step(1, dt)
        out[name] = s.read_vm()
    assert out["coupled"] - out["free"] == pytest.approx(dt * D / (chi * Cm), rel=1e-9)
    assert out["stim"] - out["free"] == pytest.approx(np.full(2, dt * 26.0), rel=1e-9)


def test_every_right_hand_side_is_taken_at_the_old_time_level(oracle):
    """PAPER.md:176 (reading A13): n steps in one call equal n calls of one step, bit for bit, and the diffusion term of
    step 2 is built from the potentials after step 1, not before: with sigma switched off after the first step nothing
    of the first-step field may leak into the second."""
    a = _two_tet(oracle, TWO["sigma_scale"]); b = _two_tet(oracle, TWO["sigma_scale"])
    for s in (a, b):
        s.state_init(0, None)
        s.write_state(0, np.array([20.0, -60.0]))
    a.step(3, 0.02)
    for _ in range(3):
        b.step(1, 0.02)
    for k in range(19):
        assert np.array_equal(a.read_state(k), b.read_state(k)), k


def test_triggered_stimulus_timing(oracle):
    """Communication-node coupling in the oracle, pinned on two UNCOUPLED cells (sigma scale 0, so each
    tet is a single cell): cell 0 is paced and monitored; the trigger must fire at the step after its first crossing of
    0 mV (read off an independent single-cell trace), and cell 1 must then follow exactly the single-cell trace of a cell
    stimulated for the slot's duration starting `delay` after that instant."""
    xyz = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1.0]])
    tets = np.array([[0, 1, 2, 3], [1, 2, 3, 4]], np.int32)
    s = oracle.OracleSim(xyz, tets, None, np.zeros(2))
    s.state_init(0, None)
    dt, delay, dur = 0.02, 5.0, 0.5                          # PAPER.md:196 orthodromic delay, S_d = 0.5 ms
    s.stimulus_set(0, np.array([0]), -52.0, 0.0, 1.0)
    s.stimulus_set(1, np.array([1]), -80.0, 123.0, dur)      # its own t_start must be ignored once a trigger drives it
    s.trigger_set(0, np.array([0]), 1, delay)
    s.step(1500, dt)
    _, tr0 = oracle.tp06_run(oracle.tp06_rest(), 0, dt, 1500, istim=-52.0, n_on=0, n_off=50, trace=True)
    n_cross = int(np.argmax(tr0 > 0.0))                      # first index with v > 0 = (crossing step + 1)
    assert tr0[n_cross - 1] <= 0.0 < tr0[n_cross]
    assert s.trigger_time(0) == n_cross * dt
    assert s.activation_times()[0] == n_cross * dt
    n_on = n_cross + 250                                     # 5 ms / 0.02 ms
    y1, _ = oracle.tp06_run(oracle.tp06_rest(), 0, dt, 1500, istim=-80.0, n_on=n_on, n_off=n_on + 25)
    got = np.array([s.read_state(k)[1] for k in range(19)])
    assert np.array_equal(got, y1)
    # never fired -> the driven slot stays off even inside its own window
    s2 = oracle.OracleSim(xyz, tets, None, np.zeros(2))
    s2.state_init(0, None)
    s2.stimulus_set(1, np.array([1]), -80.0, 0.0, 1.0)
    s2.trigger_set(0, np.array([0]), 1, 0.0)
    s2.step(200, dt)
    assert s2.trigger_time(0) == -1.0 and abs(s2.read_vm()[1] + 86.2) < 0.5
