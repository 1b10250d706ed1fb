"""Seeded random cell states inside physiological ranges, for one-step parity tests (no method arithmetic here).

Ranges cover what a ventricular / atrial cell visits during an action potential: Vm from below rest to the overshoot,
gates anywhere in [0,1], concentrations around their resting and peak values.  Order = the ABI's state order.
"""
from __future__ import annotations

import numpy as np

from .prng import uniform

# (lo, hi) per state variable, TP06 order: v m h j xr1 xr2 xs r s d f f2 fCass Rbar Ca_i Ca_SR Ca_SS Na_i K_i
TP06_RANGES = [(-95.0, 45.0)] + [(0.0, 1.0)] * 13 + [(4e-5, 1.5e-3), (0.5, 4.5), (4e-5, 5e-3), (6.0, 12.0),
                                                       (125.0, 142.0)]

# Courtemanche order: V m h j oa oi ua ui xr xs d f fCa u v w Na_i K_i Ca_i Ca_up Ca_rel
CRN98_RANGES = [(-90.0, 35.0)] + [(0.0, 1.0)] * 15 + [(9.0, 14.0), (130.0, 142.0), (6e-5, 1.2e-3), (0.8, 2.2),
                                                       (0.3, 2.0)]

# Stewart order: V y xr1 xr2 xs m h j d f f2 fCass s r R' Ca_i Ca_SR Ca_SS Na_i K_i
STEWART_RANGES = [(-95.0, 50.0)] + [(0.0, 1.0)] * 14 + [(4e-5, 1.5e-3), (0.5, 4.5), (4e-5, 5e-3), (6.0, 12.0),
                                                          (125.0, 142.0)]


def random_states(model: int, seed: int, n: int) -> np.ndarray:
    """[S, n] float64; variable k of cell c is uniform in its range, from counter k*n + c."""
    ranges = TP06_RANGES if model == 0 else (CRN98_RANGES if model == 1 else STEWART_RANGES)
    out = np.empty((len(ranges), n))
    ctr = np.arange(n, dtype=np.uint64)
    for k, (lo, hi) in enumerate(ranges):
        out[k] = uniform(seed, ctr + np.uint64(k) * np.uint64(n), lo, hi)
    return out


def special_voltages() -> np.ndarray:
    """Voltages at which the model has branch points or removable singularities (readings B6, B7)."""
    return np.array([-40.0, np.nextafter(-40.0, -100.0), np.nextafter(-40.0, 0.0), 15.0, 15.0 + 1e-9, 15.0 - 1e-9,
                     15.0 + 1e-6, 0.0, -86.2, -100.0, 60.0])
