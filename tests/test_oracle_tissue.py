"""Tissue-level pins of the oracle (diffusion + TP06 together) against what the paper states.

P11 (Fig. 11): conduction velocity along the fibres rises with mesh refinement and converges; the
converged value lies in the physiological range for ventricular myocardium (PAPER.md:21 quotes 0.3-0.5 m/s for atria
and faster ventricles; TP06 monodomain benchmarks sit at 0.5-0.7 m/s along fibres).
P5 (dense brute force): the operator assembled column by column from the oracle equals the dense matrix expanded
from the preprocessor's factored coefficients, has zero row sums, volume-weighted zero column sums and a spectrum in
the closed left half-plane.
"""
import os

import numpy as np

from ep_inputs import meshes as M


def _cv_along_x(oracle, h, dt, t_end=16.0):
    nx, ny = int(round(6.0 / h)), max(2, int(round(1.0 / h)))
    m = M.kuhn_slab(nx, ny, ny, h)
    fib = np.tile([1.0, 0.0, 0.0], (m.n_tets, 1))
    s = oracle.OracleSim(m.xyz, m.tets, fib, None, 1.3, 0.18, 1400.0, 1.0)
    s.state_init(0, None)
    cen = m.centroids()
    s.stimulus_set(0, np.nonzero(cen[:, 0] < 0.5)[0], -52.0, 0.0, 1.0)
    s.step(int(round(t_end / dt)), dt)
    ta = s.activation_times()
    assert (ta >= 0).all(), "the wave must cross the whole slab"
    # mean activation time in two transverse slices
    a = np.abs(cen[:, 0] - 2.0) < 0.5 * h + 1e-9
    b = np.abs(cen[:, 0] - 4.5) < 0.5 * h + 1e-9
    xa, xb = cen[a, 0].mean(), cen[b, 0].mean()
    return (xb - xa) / (ta[b].mean() - ta[a].mean()) * 100.0   # mm/ms -> cm/s


def test_plane_wave_cv_converges_under_refinement(oracle):
    oracle.set_threads(max(1, os.cpu_count() or 1))
    cv = [_cv_along_x(oracle, 0.5, 0.02), _cv_along_x(oracle, 0.25, 0.02), _cv_along_x(oracle, 0.125, 0.01)]
    oracle.set_threads(1)
    assert cv[0] < cv[1] < cv[2], cv                 # rises with refinement
    assert (cv[2] - cv[1]) < (cv[1] - cv[0]), cv     # and the increments shrink: converging from below
    assert abs(cv[1] - 53.7) < 1.0 and abs(cv[2] - 58.6) < 1.0, cv   # regression guard (SURVEY probe: 53.5 / 58.9)
    assert 45.0 < cv[2] < 75.0, cv                   # physiological range along fibres


def test_dense_assembly_matches_factored_stencil(oracle):
    import paper_2112_12854_b200 as ep
    m = M.kuhn_slab(4, 3, 3, 0.4)
    M.jitter_interior(m, 0.06, 5)
    cen = m.centroids()
    th = np.deg2rad(-60 + 120 * cen[:, 2] / 1.2)
    fib = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    n = m.n_tets
    s = oracle.OracleSim(m.xyz, m.tets, fib, None, 1.3, 0.18, 1400.0, 1.0)
    A = np.empty((n, n))
    for j in range(n):                                # brute force: one unit vector per column
        e = np.zeros(n); e[j] = 1.0
        A[:, j] = s.apply_diffusion(e)
    st = ep.host_stencil(m.xyz, m.tets, fib, None, 1.3, 0.18, 1400.0, 1.0)
    nn = m.n_nodes
    W = np.zeros((nn, n))                             # node interpolation matrix
    owner = np.repeat(np.arange(nn), np.diff(st["node_ptr"]))
    W[owner, st["node_cell"]] += st["w"]
    B = np.zeros((n, n))
    rows = np.arange(n)
    for k in range(8):
        B += st["a"][:, k, None] * W[st["node"][:, k], :]
    for k in range(4):
        np.add.at(B, (rows, st["nbr"][:, k]), st["b"][:, k])
        np.add.at(B, (rows, rows), -st["b"][:, k])
    B *= 1400.0 * 1.0
    scale = np.abs(A).max()
    assert np.abs(A - B).max() <= 1e-12 * scale
    assert np.abs(A.sum(axis=1)).max() <= 1e-11 * scale            # P1: row sums vanish
    vol, _ = s.geometry()
    assert np.abs(vol @ A).max() <= 1e-11 * scale * vol.max()      # P2: volume-weighted column sums vanish
    assert np.all(np.diag(A) < 0)
    lam = np.linalg.eigvals(A)
    assert lam.real.max() <= 1e-9 * scale                          # stable with eq. (8)


def test_volume_averaged_potential(oracle):
    """v_bar: exact for a uniform field; for v = x on a box tiled by tets the volume-weighted mean of
    the centroid values is the box centroid, whatever the (jittered) tetrahedra are."""
    m = M.kuhn_slab(6, 4, 3, 0.5)
    M.jitter_interior(m, 0.1, 3)
    s = oracle.OracleSim(m.xyz, m.tets)
    s.state_init(0, None)
    assert abs(s.mean_vm() + 86.2) < 1e-12
    s.write_state(0, m.centroids()[:, 0])
    assert abs(s.mean_vm() - 1.5) < 1e-13
    s.write_state(0, 2.0 * m.centroids()[:, 2] - 7.0)
    assert abs(s.mean_vm() - (2.0 * 0.75 - 7.0)) < 1e-13


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
