"""The five BASELINE.json workloads as seeded synthetic problems (recipe: SURVEY.md section 8(d)).

These stand in for the paper's slab benchmark and heart meshes, which are not
available. `coarsen` multiplies the lattice spacing so that tests can run a small twin of the same geometry.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import meshes as M
from .prng import splitmix64

MODEL_TP06 = 0
MODEL_CRN98 = 1
MODEL_STEWART = 2


@dataclass
class Stimulus:
    cell_ids: np.ndarray   # int64
    amplitude: float       # uA/cm^2, negative depolarises (reading A15)
    t_start: float         # ms
    duration: float        # ms


@dataclass
class Trigger:
    """Communication-node coupling inside one mesh: the first monitored cell to exceed 0 mV switches
    stimulus slot `slot` on `delay` ms later (ep_trigger_set)."""
    monitor_ids: np.ndarray   # int64
    slot: int
    delay: float              # ms


@dataclass
class Problem:
    name: str
    mesh: M.TetMesh
    sigma_l: float = 1.3      # mS/cm
    sigma_t: float = 0.18     # mS/cm
    chi: float = 1400.0       # 1/cm
    Cm: float = 1.0           # uF/cm^2
    model: int = MODEL_TP06
    stimuli: list = field(default_factory=list)
    dt: float = 0.02          # ms
    n_steps: int = 1000
    notes: dict = field(default_factory=dict)
    triggers: list = field(default_factory=list)   # trigger k drives stimuli[triggers[k].slot]


def _pick(seed: int, pool: np.ndarray, k: int) -> np.ndarray:
    """k distinct entries of pool, chosen by sorting pool by a splitmix64 key."""
    key = splitmix64(seed, pool.astype(np.uint64))
    order = np.argsort(key, kind="stable")
    return pool[order[:k]]


def _balls(cent: np.ndarray, centres: np.ndarray, radius: float) -> np.ndarray:
    """Ids (ascending) of the cells whose centroid lies within `radius` of any of `centres`."""
    order = np.argsort(cent[:, 0], kind="stable")
    xs = cent[order, 0]
    hit = np.zeros(cent.shape[0], dtype=bool)
    for c in centres:
        lo, hi = np.searchsorted(xs, [c[0] - radius, c[0] + radius])
        idx = order[lo:hi]
        d2 = ((cent[idx] - c[None, :]) ** 2).sum(axis=1)
        hit[idx[d2 <= radius * radius]] = True
    return np.nonzero(hit)[0].astype(np.int64)


def config1(coarsen: float = 1.0) -> Problem:
    """C1: 5x5x1 mm slab, 20x20x4 cubes of 0.25 mm -> 9,600 tets; fibres along x; all endo; stimulus x<0.5 mm."""
    n = max(1, int(round(20 / coarsen)))
    nz = max(1, int(round(4 / coarsen)))
    mesh = M.kuhn_slab(n, n, nz, 5.0 / n)
    mesh.fibre = np.tile(np.array([1.0, 0.0, 0.0]), (mesh.n_tets, 1))
    mesh.cell_type = np.zeros(mesh.n_tets, dtype=np.uint8)
    cent = mesh.centroids()
    ids = np.nonzero(cent[:, 0] < 0.5)[0].astype(np.int64)
    return Problem("C1_tiny_slab", mesh, stimuli=[Stimulus(ids, -52.0, 0.0, 1.0)], dt=0.02, n_steps=1000)


def config2(coarsen: float = 1.0, seed: int = 1001, jitter: float = 0.2) -> Problem:
    """C2: the paper's 20x7x3 mm slab at dx=0.2 mm, interior nodes jittered +-20% dx per axis,
    fibre angle -60..+60 degrees through z, endo/mid/epi thirds in z, corner cube 1.5 mm stimulus."""
    dx = 0.2 * coarsen
    nx, ny, nz = int(round(20 / dx)), int(round(7 / dx)), int(round(3 / dx))
    mesh = M.kuhn_slab(nx, ny, nz, dx)
    M.jitter_interior(mesh, jitter * dx, seed)
    cent = mesh.centroids()
    zrel = np.clip(cent[:, 2] / (nz * dx), 0.0, 1.0)
    theta = np.deg2rad(-60.0 + 120.0 * zrel)
    mesh.fibre = np.stack([np.cos(theta), np.sin(theta), np.zeros_like(theta)], axis=1)
    mesh.cell_type = M.thirds(zrel)
    ids = np.nonzero(np.all(cent < 1.5, axis=1))[0].astype(np.int64)
    return Problem("C2_irregular_slab", mesh, stimuli=[Stimulus(ids, -52.0, 0.0, 1.0)], dt=0.02, n_steps=5000,
                   notes={"seed": seed, "dt_run": 0.005,
                          "dt_note": "nominal 0.02 ms is beyond the explicit stability limit of this jittered mesh "
                                     "(DESIGN.md reading S); runs use dt_run = 0.02/4 = the paper's finest dt"})


_LV_OUT = (35.0, 35.0, 60.0)
_LV_IN = (25.0, 25.0, 50.0)
_LV_ZCUT = 20.0


def _lv_inside(p):
    return M.in_ellipsoid(p, (0, 0, 0), _LV_OUT) & ~M.in_ellipsoid(p, (0, 0, 0), _LV_IN) & (p[:, 2] <= _LV_ZCUT)


def config3(coarsen: float = 1.0, seed: int = 1003, h: float = 0.72) -> Problem:
    """C3: truncated prolate LV shell (outer 35/35/60 mm, wall 10 mm, z<=20 mm), ~2M tets at h=0.72 mm; helical fibres
    +60 (endo) -> -60 (epi); endo/mid/epi thirds; 40 seeded endocardial stimulus balls of radius 1.5 mm, 1 ms."""
    h = h * coarsen
    mesh = M.carve_lattice(_lv_inside, (-35.0, -35.0, -60.0), (35.0, 35.0, _LV_ZCUT), h)
    cent = mesh.centroids()
    mesh.fibre, d = M.helical_fibres(cent, (0, 0, 0), _LV_IN, _LV_OUT)
    mesh.cell_type = M.thirds(d)
    pool = np.nonzero(d < 0.15)[0]
    pts = _pick(seed, pool, 40)
    ids = _balls(cent, cent[pts], max(1.5, 1.5 * coarsen))
    return Problem("C3_lv_ellipsoid", mesh, stimuli=[Stimulus(ids, -52.0, 0.0, 1.0)], dt=0.02, n_steps=20000,
                   notes={"seed": seed, "h": h})


_RV_C = (22.0, 0.0, 0.0)
_RV_OUT = (38.0, 32.0, 52.0)
_RV_IN = (34.0, 28.0, 48.0)


def _rv_inside(p):
    return (M.in_ellipsoid(p, _RV_C, _RV_OUT) & ~M.in_ellipsoid(p, _RV_C, _RV_IN)
            & ~M.in_ellipsoid(p, (0, 0, 0), _LV_OUT) & (p[:, 2] <= _LV_ZCUT))


def config4(coarsen: float = 1.0, seed: int = 1004, h: float = 0.345) -> Problem:
    """C4: C3's LV fused with a 4 mm crescent RV shell, ~20M tets; sigma scaled by 0.1 inside a 12 mm sphere centred at a
    seeded mid-wall LV point; 40 LV + 20 RV seeded endocardial stimulus balls; dt=0.01 ms, 5,000-step window."""
    h = h * coarsen

    def inside(p):
        return _lv_inside(p) | _rv_inside(p)

    mesh = M.carve_lattice(inside, (-35.0, -35.0, -60.0), (60.0, 35.0, _LV_ZCUT), h)
    cent = mesh.centroids()
    is_lv = _lv_inside(cent)
    mesh.fibre = np.empty((mesh.n_tets, 3))
    d = np.empty(mesh.n_tets)
    mesh.fibre[is_lv], d[is_lv] = M.helical_fibres(cent[is_lv], (0, 0, 0), _LV_IN, _LV_OUT)
    mesh.fibre[~is_lv], d[~is_lv] = M.helical_fibres(cent[~is_lv], _RV_C, _RV_IN, _RV_OUT)
    mesh.cell_type = M.thirds(d)
    mid_pool = np.nonzero(is_lv & (np.abs(d - 0.5) < 0.1))[0]
    scar_c = cent[_pick(seed + 7, mid_pool, 1)[0]]
    scale = np.ones(mesh.n_tets)
    scale[((cent - scar_c[None, :]) ** 2).sum(axis=1) <= 144.0] = 0.1
    mesh.sigma_scale = scale
    pts = np.concatenate([_pick(seed, np.nonzero(is_lv & (d < 0.15))[0], 40),
                          _pick(seed + 1, np.nonzero(~is_lv & (d < 0.3))[0], 20)])
    ids = _balls(cent, cent[pts], max(1.5, 1.5 * coarsen))
    return Problem("C4_biventricle_scar", mesh, stimuli=[Stimulus(ids, -52.0, 0.0, 1.0)], dt=0.01, n_steps=5000,
                   notes={"seed": seed, "h": h, "scar_centre": scar_c.tolist()})


_AT_OUT = (40.0, 40.0, 45.0)
_AT_IN = (38.0, 38.0, 43.0)
_AT_C = ((-45.0, 0.0, 0.0), (45.0, 0.0, 0.0))


def config5(coarsen: float = 1.0, seed: int = 1005, h: float = 0.55) -> Problem:
    """C5: two disjoint ellipsoidal atrial shells (outer 40/40/45 mm, wall 2 mm, centres 90 mm apart), ~3M tets;
    circumferential fibres; Courtemanche model (21 states); 2 mm stimulus ball at a seeded point of shell 1, 2.5 ms."""
    h = h * coarsen

    def inside(p):
        r = np.zeros(p.shape[0], dtype=bool)
        for c in _AT_C:
            r |= M.in_ellipsoid(p, c, _AT_OUT) & ~M.in_ellipsoid(p, c, _AT_IN)
        return r

    mesh = M.carve_lattice(inside, (-85.0, -40.0, -45.0), (85.0, 40.0, 45.0), h)
    cent = mesh.centroids()
    left = cent[:, 0] < 0
    c_of = np.where(left[:, None], np.array(_AT_C[0])[None, :], np.array(_AT_C[1])[None, :])
    _, circ, _ = M.ellipsoid_frame(cent - c_of, (0, 0, 0), _AT_OUT)
    mesh.fibre = circ
    mesh.cell_type = np.zeros(mesh.n_tets, dtype=np.uint8)
    pt = _pick(seed, np.nonzero(left)[0], 1)
    r = max(2.0, 2.0 * coarsen)
    ids = _balls(cent, cent[pt], r)
    stimuli = [Stimulus(ids, -52.0, 0.0, 2.5)]
    # Reading G1: the 2 mm patch alone excites the wall and the wave travels at ~0.3 m/s along the fibres, which reaches
    # ~5 % of the cells in 150 ms; in the paper the atria are activated within 140 ms because the 1D internodal pathways and
    # Bachmann's bundle (1.5 m/s) re-excite the myocardium through communication nodes.  Those
    # bundles are outside this path, so they are stood in for by two trigger-driven slots (ep_trigger_set): 12 seeded sites
    # on the shell of the sinus node 10 ms after the patch fires, 12 on the other shell 30 ms after it.
    triggers = []
    for k, (pool, delay) in enumerate(((np.nonzero(left)[0], 10.0), (np.nonzero(~left)[0], 30.0))):
        sites = _pick(seed + 1 + k, pool, 12)
        stimuli.append(Stimulus(_balls(cent, cent[sites], r), -52.0, 1e9, 2.5))
        triggers.append(Trigger(ids, 1 + k, delay))
    return Problem("C5_atrial_shell", mesh, model=MODEL_CRN98, stimuli=stimuli, dt=0.01, n_steps=15000,
                   notes={"seed": seed, "h": h}, triggers=triggers)


def paper_slab(dx: float = 0.1, coarsen: float = 1.0) -> Problem:
    """The paper's own benchmark slab (Table 1 :238-240): 20 x 7 x 3 mm, dx in {0.5, 0.2, 0.1} mm ->
    20,160 / 315,000 / 2,520,000 tets, fibres along x, corner cube of 1.5 mm stimulated, dt = 0.005 ms (the finest of
    PAPER.md:214, inside the explicit limit of all three meshes).  Un-jittered twin of config 2."""
    dx = dx * coarsen
    nx, ny, nz = int(round(20 / dx)), int(round(7 / dx)), int(round(3 / dx))
    mesh = M.kuhn_slab(nx, ny, nz, dx)
    mesh.fibre = np.tile(np.array([1.0, 0.0, 0.0]), (mesh.n_tets, 1))
    mesh.cell_type = np.zeros(mesh.n_tets, dtype=np.uint8)
    cent = mesh.centroids()
    ids = np.nonzero(np.all(cent < 1.5, axis=1))[0].astype(np.int64)
    return Problem("paper_slab_dx%g" % dx, mesh, stimuli=[Stimulus(ids, -52.0, 0.0, 2.0)], dt=0.005, n_steps=10000,
                   notes={"dx": dx})


# Table 2: 2D Purkinje network, Stewart model, isotropic monodomain, 3.95 mS/mm = 39.5 mS/cm
SIGMA_PURKINJE = 39.5


def purkinje_strip(dx: float = 0.2, jitter: float = 0.0, seed: int = 2001, lx: float = 20.0, ly: float = 7.0) -> Problem:
    """The paper's 2D benchmark domain (rectangle 20 x 7 mm, uniform grid) as a triangulated sheet with the
    Purkinje parameters of Table 2 (Stewart model, isotropic 39.5 mS/cm).  Stimulus: the strip x < 1.5 mm (the corner square
    of PAPER.md:214 does not reach the liminal size at this conductivity), -52 uA/cm^2 for 2 ms."""
    nx, ny = int(round(lx / dx)), int(round(ly / dx))
    mesh = M.rect_tri(nx, ny, dx)
    if jitter:
        M.jitter_interior_tri(mesh, jitter * dx, seed, out_of_plane=0.5 * jitter * dx)
    cent = mesh.centroids()
    ids = np.nonzero(cent[:, 0] < 1.5)[0].astype(np.int64)
    return Problem("purkinje_strip_dx%g" % dx, mesh, sigma_l=SIGMA_PURKINJE, sigma_t=SIGMA_PURKINJE, model=MODEL_STEWART,
                   stimuli=[Stimulus(ids, -52.0, 0.0, 2.0)], dt=0.001, n_steps=10000, notes={"dx": dx, "dim": 2})


def purkinje_sheet(coarsen: float = 1.0, seed: int = 2002, h: float = 0.45) -> Problem:
    """A Purkinje layer on the endocardium of config 3's left ventricle: the inner ellipsoid 25/25/50 mm below z = 20 mm as a
    triangulated surface, ~97,000 triangles at h = 0.45 mm (54,000 triangles at 0.45 mm for one ventricle,
    108,000 for both), Stewart model, isotropic 39.5 mS/cm.  Stimulus: the triangles within 3 mm of a seeded point on the
    base ring (where the bundle branch enters), 2 ms."""
    h = h * coarsen
    mesh = M.ellipsoid_surface(_LV_IN, _LV_ZCUT, h)
    cent = mesh.centroids()
    pool = np.nonzero(cent[:, 2] > _LV_ZCUT - 2.0)[0]
    pt = _pick(seed, pool, 1)
    ids = _balls(cent, cent[pt], 3.0)
    return Problem("purkinje_sheet", mesh, sigma_l=SIGMA_PURKINJE, sigma_t=SIGMA_PURKINJE, model=MODEL_STEWART,
                   stimuli=[Stimulus(ids, -52.0, 0.0, 2.0)], dt=0.001, n_steps=30000, notes={"seed": seed, "h": h, "dim": 2})


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5,
           6: lambda coarsen=1.0: paper_slab(0.5, coarsen), 7: lambda coarsen=1.0: paper_slab(0.2, coarsen),
           8: lambda coarsen=1.0: paper_slab(0.1, coarsen),
           9: lambda coarsen=1.0: purkinje_strip(0.2 * coarsen), 10: purkinje_sheet}


def make(cfg: int, coarsen: float = 1.0) -> Problem:
    return CONFIGS[cfg](coarsen=coarsen)
