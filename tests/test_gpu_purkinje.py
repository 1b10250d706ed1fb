"""GPU parity of the two-dimensional medium: triangulated-surface finite volumes (ep_mesh_create_tri,
PAPER.md:170) with the Stewart Purkinje model (EP_MODEL_STEWART) against oracle/ep_oracle2d, and the
communication-node coupling of a Purkinje sheet to a ventricular slab across two handles.

Tolerances are north_star's: one step max|g-o|/max|o| <= 1e-11 per state variable, runs max|dVm| <= 1e-6 mV with
activation times equal to within one dt and identical activated sets."""
import numpy as np
import pytest

from ep_inputs import meshes as M
from ep_inputs import states
from ep_inputs.configs import make, purkinje_sheet, purkinje_strip
from ep_inputs.prng import uniform

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
def O2():
    from oracle import ep_oracle2d
    return ep_oracle2d


def _bumpy_problem():
    prob = purkinje_strip(0.3, lx=6.0, ly=4.2)
    M.jitter_interior_tri(prob.mesh, 0.06, 5, out_of_plane=0.05)
    cen = prob.mesh.centroids()
    th = np.deg2rad(10 + 50 * cen[:, 1] / 4.2)
    prob.mesh.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    prob.mesh.sigma_scale = uniform(14, np.arange(prob.mesh.n_tris), 0.1, 1.0)
    prob.sigma_l, prob.sigma_t = 30.0, 8.0
    return prob


@pytest.mark.parametrize("case", ["bumpy_sheet", "strip", "surface_coarse"])
def test_diffusion_operator_parity_2d(ep, O2, case):
    prob = {"bumpy_sheet": _bumpy_problem, "strip": lambda: purkinje_strip(0.25),
            "surface_coarse": lambda: purkinje_sheet(coarsen=4.0)}[case]()
    g = ep.Sim.from_problem(prob)
    o = O2.OracleSim2D.from_problem(prob)
    for seed in (1, 2):
        v = uniform(seed, np.arange(prob.mesh.n_tris), -90.0, 40.0)
        Dg, Do = g.apply_diffusion(v), o.apply_diffusion(v)
        assert np.abs(Dg - Do).max() <= 1e-12 * np.abs(Do).max()
    g.close()


def _one_step_err(g, o, S):
    errs = []
    for k in range(S):
        a, b = g.read_state(k), o.read_state(k)
        d = np.abs(a - b)
        scale = np.abs(b).max()
        errs.append(d.max() / scale)
        bad = d > 1e-10 * np.abs(b) + 1e-14 * scale           # per-cell bound, as in test_gpu_parity.py
        assert not bad.any(), (k, int(bad.sum()))
    return np.array(errs)


@pytest.mark.parametrize("case", ["bumpy_sheet", "strip"])
def test_stewart_one_step_random_states(ep, O2, case):
    """One explicit step from random physiological states (branch points of h / j and the I_CaL singularity planted),
    stimulus on for part of the cells; two more steps stay within 10x the tolerance."""
    prob = _bumpy_problem() if case == "bumpy_sheet" else purkinje_strip(0.25)
    n = prob.mesh.n_tris
    prob.stimuli[0].cell_ids = np.arange(0, n, 5, dtype=np.int64)
    g = ep.Sim.from_problem(prob)
    o = O2.OracleSim2D.from_problem(prob)
    y = states.random_states(2, 91, n)
    sv = states.special_voltages()
    y[0, : sv.size] = sv
    for k in range(20):
        g.write_state(k, y[k]); o.write_state(k, y[k])
    dt = 0.001
    g.step(1, dt); o.step(1, dt)
    err = _one_step_err(g, o, 20)
    assert err.max() <= ONE_STEP_TOL, err
    g.step(2, dt); o.step(2, dt)
    assert _one_step_err(g, o, 20).max() <= 10 * ONE_STEP_TOL
    g.close()


def test_stewart_beyond_physiological_voltages(ep, O2):
    """Reading T2: for |v| <= 200 mV the clamp of the transcendental arguments is inert."""
    prob = purkinje_strip(0.5)
    n = prob.mesh.n_tris
    g = ep.Sim.from_problem(prob)
    o = O2.OracleSim2D.from_problem(prob)
    y = states.random_states(2, 92, n)
    y[0] = uniform(93, np.arange(n), -200.0, 200.0)
    for k in range(20):
        g.write_state(k, y[k]); o.write_state(k, y[k])
    g.step(1, 0.001); o.step(1, 0.001)
    for k in range(20):
        a, b = g.read_state(k), o.read_state(k)
        assert np.abs(a - b).max() <= ONE_STEP_TOL * np.abs(b).max(), k
    g.close()


def test_purkinje_strip_run_and_conduction_velocity(ep, O2, capsys):
    """The paper's 2D benchmark rectangle with Table 2's Purkinje parameters, dx = 0.25 mm, dt below the
    explicit limit reported by ep_stable_dt: 6 ms of propagation against the oracle (graph replay path: 6,000 steps), then the
    conduction velocity between x = 5 and 15 mm on the GPU path alone: 4.0 m/s within 5 % (Table 2)."""
    prob = purkinje_strip(0.25)
    g = ep.Sim.from_problem(prob)
    o = O2.OracleSim2D.from_problem(prob)
    dt_max = g.stable_dt()
    dt = 0.001
    assert dt < 0.8 * dt_max, dt_max
    worst = 0.0
    for _ in range(6):
        g.step(1000, dt); o.step(1000, dt)
        worst = max(worst, np.abs(g.read_vm() - o.read_vm()).max())
    ta_g, ta_o = g.activation_times(), o.activation_times()
    assert worst <= RUN_TOL_MV, worst
    assert ((ta_g >= 0) == (ta_o >= 0)).all() and np.abs(ta_g - ta_o).max() <= dt + 1e-12
    assert abs(g.mean_vm() - o.mean_vm()) <= RUN_TOL_MV
    g.step(3000, dt)
    ta = g.activation_times()
    cen = prob.mesh.centroids()
    assert (ta >= 0).all() and g.check_finite()
    band = lambda x0: np.abs(cen[:, 0] - x0) < 0.25
    cv = 10.0 / (ta[band(15.0)].mean() - ta[band(5.0)].mean())
    with capsys.disabled():
        print("Purkinje strip dx=0.25 mm: %d cells, dt=%.4f ms (limit %.4f), 6 ms vs oracle max|dVm| = %.3e mV, "
              "CV = %.3f m/s (Table 2: 4.0)" % (prob.mesh.n_tris, dt, dt_max, worst, cv))
    assert cv == pytest.approx(4.0, rel=0.05)
    g.close()


def test_purkinje_sheet_window_on_the_full_surface(ep, O2, capsys):
    """The ~97,000-triangle endocardial Purkinje layer (54,000 / 108,000 triangles): 2,000 steps from the
    stimulus against the oracle on the full surface, then the GPU alone until the whole layer has fired."""
    prob = purkinje_sheet()
    g = ep.Sim.from_problem(prob)
    o = O2.OracleSim2D.from_problem(prob)
    dt_max = g.stable_dt()
    dt = 0.002 if 0.002 < 0.8 * dt_max else 0.001
    g.step(2000, dt); o.step(2000, dt)
    dv = np.abs(g.read_vm() - o.read_vm()).max()
    ta_g, ta_o = g.activation_times(), o.activation_times()
    assert dv <= RUN_TOL_MV and ((ta_g >= 0) == (ta_o >= 0)).all() and np.abs(ta_g - ta_o).max() <= dt + 1e-12
    n_act = int((ta_g >= 0).sum())
    g.step(int(round(60.0 / dt)) - 2000, dt)
    ta = g.activation_times()
    with capsys.disabled():
        print("Purkinje sheet: %d triangles, dt=%.4f ms (limit %.4f): 2,000 steps vs oracle max|dVm| = %.3e mV "
              "(%d cells activated); after 60 ms %d / %d activated, last at %.2f ms"
              % (prob.mesh.n_tris, dt, dt_max, dv, n_act, int((ta >= 0).sum()), ta.size, ta.max()))
    assert (ta >= 0).all() and g.check_finite()
    g.close()


def test_stewart_automaticity_on_the_gpu(ep, O2):
    """Unstimulated, uncoupled Purkinje cells fire spontaneously (I_f): the GPU path reproduces the oracle's first
    spontaneous upstroke (about 98 ms from the published initial state) to the step."""
    m = M.rect_tri(8, 8, 0.5)
    g = ep.Sim(m.xyz, m.tris, None, np.zeros(m.n_tris), 39.5, 39.5)
    g.state_init(ep.EP_MODEL_STEWART)
    dt = 0.01
    g.step(12000, dt)
    ta = g.activation_times()
    _, tr = O2.stw_run(O2.stw_init(), dt, 12000, trace=True)
    n_cross = int(np.nonzero((tr[:-1] <= 0) & (tr[1:] > 0))[0][0])
    assert np.all(ta == (n_cross + 1) * dt) and 90.0 < ta[0] < 110.0
    assert np.abs(g.read_vm() - tr[-1]).max() <= RUN_TOL_MV
    g.close()


def test_purkinje_muscle_junctions_couple_two_handles(ep, O2, oracle, capsys):
    """a wave on the 2D Purkinje sheet (Stewart, Table 2 conductivity) passes two communication nodes; each
    switches on, 5 ms later (the orthodromic delay of PAPER.md:196), a stimulus on the cells of a 3D ventricular slab (TP06,
    config 1's mesh) within R_S of its junction, and the two wavefronts started there spread through the slab.  GPU: two
    handles advanced in 1 ms slices with their own time steps (0.0025 / 0.02 ms), ep_trigger_set(slot = -1) + ep_couple.
    Oracle: the same protocol with the 2D and 3D oracles, the firing time taken from the 2D oracle's activation times.
    Firing times equal; both fields within 1e-6 mV; activation times within one dt, identical activated sets."""
    pp = purkinje_strip(0.5, lx=10.0, ly=3.5)
    pv = make(1)
    pv.stimuli = []
    cen2, cen3 = pp.mesh.centroids(), pv.mesh.centroids()
    junctions = [(4.0, 1.75), (8.0, 1.75)]
    targets = [np.array([1.2, 1.2, 0.5]), np.array([3.8, 3.8, 0.5])]
    monitors = [np.nonzero(np.hypot(cen2[:, 0] - x, cen2[:, 1] - y) < 0.5)[0].astype(np.int64) for x, y in junctions]
    regions = [np.nonzero(np.linalg.norm(cen3 - t, axis=1) < 0.75)[0].astype(np.int64) for t in targets]
    DELAY, AMP, DUR, NEVER = 5.0, -80.0, 1.5, 1.0e9
    dt2, dt3 = 0.0025, 0.02
    # --- GPU
    gp, gv = ep.Sim.from_problem(pp), ep.Sim.from_problem(pv)
    for k in range(2):
        gp.trigger_set(k, monitors[k], -1, 0.0)
        gv.stimulus_set(k, regions[k], AMP, NEVER, DUR)
    # --- oracle
    op = O2.OracleSim2D.from_problem(pp)
    ov = oracle.OracleSim.from_problem(pv)
    fired_o = [-1.0, -1.0]
    sched_g = [False, False]
    for ms in range(16):
        gp.step(400, dt2); gv.step(50, dt3)
        op.step(400, dt2); ov.step(50, dt3)
        for k in range(2):
            if not sched_g[k]:
                sched_g[k] = gp.couple(k, gv, k, DELAY)
            if fired_o[k] < 0:
                ta = op.activation_times()[monitors[k]]
                if (ta >= 0).any():
                    fired_o[k] = float(ta[ta >= 0].min())
                    ov.stimulus_set(k, regions[k], AMP, fired_o[k] + DELAY, DUR)
    fired_g = [gp.trigger_time(k) for k in range(2)]
    assert all(sched_g) and fired_g == fired_o and 0.0 < fired_g[0] < fired_g[1] < 4.0, (fired_g, fired_o)
    dvp = np.abs(gp.read_vm() - op.read_vm()).max()
    dvv = np.abs(gv.read_vm() - ov.read_vm()).max()
    ta_g, ta_o = gv.activation_times(), ov.activation_times()
    with capsys.disabled():
        print("PMJ coupling: junctions fired at %.4f / %.4f ms, slab stimulated 5 ms later; after 16 ms %d / %d slab cells "
              "activated; max|dVm| sheet %.3e mV, slab %.3e mV" % (fired_g[0], fired_g[1], int((ta_g >= 0).sum()), ta_g.size, dvp, dvv))
    assert dvp <= RUN_TOL_MV and dvv <= RUN_TOL_MV
    assert ((ta_g >= 0) == (ta_o >= 0)).all() and (ta_g >= 0).sum() > 0.5 * ta_g.size
    assert np.abs(ta_g - ta_o)[ta_g >= 0].max() <= dt3 + 1e-12
    first = ta_g[regions[0]]
    assert first[first >= 0].min() >= fired_g[0] + DELAY            # nothing in the slab fires before the delay has passed
    # polling too late is an error, not a silent shift
    gp2, gv2 = ep.Sim.from_problem(pp), ep.Sim.from_problem(pv)
    gp2.trigger_set(0, monitors[0], -1, 0.0)
    gv2.stimulus_set(0, regions[0], AMP, NEVER, DUR)
    gp2.step(4000, dt2); gv2.step(500, dt3)
    with pytest.raises(ep.EpError) as e:
        gp2.couple(0, gv2, 0, DELAY)
    assert e.value.code == -3
    for s in (gp, gv, gp2, gv2):
        s.close()
