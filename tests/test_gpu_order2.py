"""GPU parity and measured order of the second-order time stepping (ep_set_time_order(2))
against oracle/ep_oracle_o2.  Tolerances: north_star's (one step 1e-11 relative per state variable, runs 1e-6 mV)."""
import numpy as np
import pytest

from ep_inputs import make, states
from ep_inputs import meshes as M

pytestmark = pytest.mark.gpu
ONE_STEP_TOL = 1e-11
RUN_TOL_MV = 1e-6


@pytest.fixture(scope="module")
def ep():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2112_12854_b200 as ep
    return ep


@pytest.fixture(scope="module")
def OO():
    from oracle import ep_oracle_o2
    ep_oracle_o2.set_threads(8)
    return ep_oracle_o2


def _err(g, o):
    e = []
    for k in range(19):
        a, b = g.read_state(k), o.read_state(k)
        e.append(np.abs(a - b).max() / np.abs(b).max())
    return np.array(e)


def test_first_steps_from_random_states(ep, OO):
    """Random physiological states, all three cell types, stimulus on part of the cells: step 1 (no history: first order),
    then steps 2 and 3 (Adams-Bashforth + extrapolated gate arguments) against the oracle, state by state."""
    prob = make(3, coarsen=3.0)
    n = prob.mesh.n_tets
    prob.stimuli[0].cell_ids = np.arange(0, n, 6, dtype=np.int64)
    g = ep.Sim.from_problem(prob)
    g.set_time_order(2)
    o = OO.OracleSimO2.from_problem(prob)
    y = states.random_states(0, 55, n)
    sv = states.special_voltages()
    y[0, : sv.size] = sv
    for k in range(19):
        g.write_state(k, y[k]); o.write_state(k, y[k])
    dt = 0.01
    for step, tol in ((1, ONE_STEP_TOL), (2, 3 * ONE_STEP_TOL), (3, 10 * ONE_STEP_TOL)):
        g.step(1, dt); o.step(1, dt)
        e = _err(g, o)
        assert e.max() <= tol, (step, e)
    g.close(); o.close()


def test_config1_run_second_order(ep, OO, capsys):
    """Config 1 (9,600 cells) for 2,000 steps of 0.01 ms (single first step + 62 graph replays + tail): fields, activation
    times and activated set against the oracle."""
    prob = make(1)
    g = ep.Sim.from_problem(prob)
    g.set_time_order(2)
    o = OO.OracleSimO2.from_problem(prob)
    dt = 0.01
    worst = 0.0
    for _ in range(4):
        g.step(500, dt); o.step(500, dt)
        worst = max(worst, np.abs(g.read_vm() - o.read_vm()).max())
    ta_g, ta_o = g.activation_times(), o.activation_times()
    with capsys.disabled():
        print("second-order scheme, config 1 x 2,000 steps: max|dVm| = %.3e mV, %d cells activated" % (worst, int((ta_g >= 0).sum())))
    assert worst <= RUN_TOL_MV and g.check_finite()
    assert np.array_equal(ta_g >= 0, ta_o >= 0) and (ta_g >= 0).all() and np.abs(ta_g - ta_o).max() <= dt + 1e-12
    # order 1 on the same handle again: back to the paper's scheme, bit-identical to a fresh first-order run
    g.set_time_order(1)
    g.state_init(ep.EP_MODEL_TP06, prob.mesh.cell_type)
    g.step(200, 0.02)
    g1 = ep.Sim.from_problem(prob)
    g1.step(200, 0.02)
    assert np.array_equal(g.read_vm(), g1.read_vm())
    g.close(); g1.close(); o.close()


def test_measured_temporal_order_on_the_slab(ep, capsys):
    """Fig. 14b's experiment with both schemes on the GPU path: the paper's slab at dx = 0.25 mm, v_bar at
    t = 20 ms for dt = 0.02 / 0.01 / 0.005 / 0.0025 ms.  Successive differences shrink by ~2 per halving with the paper's
    first-order scheme and by ~4 with the second-order one; at dt = 0.01 ms the second-order result is already closer to the
    dt -> 0 limit than the first-order result at dt = 0.0025 ms."""
    from ep_inputs.configs import paper_slab
    prob = paper_slab(0.25)
    vb = {1: [], 2: []}
    for order in (1, 2):
        for dt in (0.02, 0.01, 0.005, 0.0025):
            g = ep.Sim.from_problem(prob)
            g.set_time_order(order)
            g.step(int(round(20.0 / dt)), dt)
            vb[order].append(g.mean_vm())
            assert g.check_finite()
            g.close()
    d1 = np.diff(vb[1]); d2 = np.diff(vb[2])
    p1 = np.log2(d1[:-1] / d1[1:]); p2 = np.log2(d2[:-1] / d2[1:])
    lim = vb[2][-1] + d2[-1] / 3.0                           # Richardson limit of the second-order sequence
    with capsys.disabled():
        print("slab dx=0.25 mm, v_bar(20 ms): first order %s -> observed order %s; second order %s -> observed order %s"
              % (np.round(vb[1], 4), np.round(p1, 2), np.round(vb[2], 4), np.round(p2, 2)))
        print("distance from the dt->0 limit %.4f mV: first order at dt=0.0025: %.2e, second order at dt=0.01: %.2e"
              % (lim, abs(vb[1][-1] - lim), abs(vb[2][1] - lim)))
    assert np.all((p1 > 0.8) & (p1 < 1.2)), p1
    assert np.all((p2 > 1.6) & (p2 < 2.4)), p2
    assert abs(vb[2][1] - lim) < abs(vb[1][-1] - lim)


def test_order_errors(ep):
    prob = make(5, coarsen=6.0)
    g = ep.Sim.from_problem(prob)                            # Courtemanche
    with pytest.raises(ep.EpError):
        g.set_time_order(2)
    with pytest.raises(ep.EpError):
        g.set_time_order(3)
    g.close()
