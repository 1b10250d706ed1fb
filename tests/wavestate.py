"""Seeded synthetic "wave in progress" initial states for the window parity tests (test infrastructure).

A window that starts from rest sees little besides the stimulus sites in its first 1,000 steps.  To put wavefronts,
plateau and repolarising tissue on the full-size meshes from step 0, every cell gets the state a single cell has at
a phase that falls off linearly with the distance to the nearest stimulated cell (a synthetic activation map): a chosen
fraction of the mesh is excited, from the front (phase 0) back to tissue that has already repolarised.  The per-phase states come from the ORACLE's single-cell runs (never
from the CUDA path); the same array is then written into both simulators, so parity is judged on identical inputs.
"""
import numpy as np
from scipy.spatial import cKDTree


def phase_table(oracle, model, cell_type, dt=0.01, t_max=400.0):
    """(phases [P] in ms after stimulus onset, states [P, S]) of one paced cell; fine sampling through the upstroke."""
    phases = np.concatenate([np.arange(0.0, 6.0, 0.05), np.arange(6.0, t_max + 1e-9, 1.0)])
    if model == 0:
        y = oracle.tp06_rest()
        run = lambda y, n, n0: oracle.tp06_run(y, cell_type, dt, n, -52.0, -n0, int(round(1.0 / dt)) - n0)[0]
    else:
        y = oracle.crn_rest()
        run = lambda y, n, n0: oracle.crn_run(y, dt, n, -20.0, -n0, int(round(2.0 / dt)) - n0)[0]
    out = np.empty((phases.size, y.size))
    n_done = 0
    for k, ph in enumerate(phases):
        n_to = int(round(ph / dt))
        if n_to > n_done:
            y = run(y, n_to - n_done, n_done)      # stimulus window expressed relative to the chunk start
            n_done = n_to
        out[k] = y
    return phases, out


def paint(oracle, prob, frac=0.45, t_span=350.0):
    """State array [S, n_tets] and the phase map: the fraction `frac` of the cells nearest to the stimulus sites is excited,
    at phases from 0 (the front, farthest of them) to t_span ms (next to a site, already repolarised for t_span beyond the
    action potential duration); everything farther away is at rest.  phase = t_span (1 - dist/d_frac)."""
    m = prob.mesh
    cen = m.centroids()
    src = np.concatenate([s.cell_ids for s in prob.stimuli])
    src = src[:: max(1, src.size // 4000)]
    dist, _ = cKDTree(cen[src]).query(cen, workers=-1)
    d_frac = np.quantile(dist, frac)
    phase = t_span * (1.0 - dist / d_frac)
    S = 19 if prob.model == 0 else 21
    y = np.empty((S, m.n_tets))
    types = m.cell_type if (prob.model == 0 and m.cell_type is not None) else np.zeros(m.n_tets, np.uint8)
    for t in np.unique(types):
        ph, tab = phase_table(oracle, prob.model, int(t), t_max=t_span)
        rest = tab[0]
        sel = np.nonzero(types == t)[0]
        idx = np.searchsorted(ph, np.maximum(phase[sel], 0.0), side="right") - 1
        vals = np.where((phase[sel] < 0.0)[:, None], rest[None, :], tab[idx])
        y[:, sel] = vals.T
    return y, phase
