"""Pins of the bidomain oracle (oracle/ep_oracle_bidomain.py; eq. (1)/(6)).

* "In the case the external and the internal conductivity tensors are parallel M_ext = lambda M_int the
  bidomain model reduces to the monodomain equation with M = lambda M_int/(1 + lambda)": the bidomain oracle run with such
  tensors must reproduce the (separately pinned) monodomain oracle run with that M, cell by cell, and
  v_ext = -v/(1 + lambda) + const.
* the elliptic equation is satisfied to round-off, v_ext has zero volume-weighted mean, the right-hand side is compatible
  (sum_c V_c b_c = 0: conservation), a constant added to v changes nothing.
* Table 2 conductivities: the unequal anisotropy ratios make the bidomain wave differ from the monodomain one
  (it is not a relabelled monodomain run), while the propagation speed along the fibres stays close to the monodomain
  value with sigma = sigma_i sigma_e/(sigma_i + sigma_e) (reading A10).
"""
import numpy as np
import pytest

from ep_inputs import meshes as M
from ep_inputs.prng import uniform
from oracle import ep_oracle as O
from oracle.ep_oracle_bidomain import BidomainOracle


def _slab(nx=10, ny=6, nz=3, h=0.25, jitter=0.0):
    m = M.kuhn_slab(nx, ny, nz, h)
    if jitter:
        M.jitter_interior(m, jitter * h, 31)
    m.fibre = np.tile(np.array([1.0, 0.0, 0.0]), (m.n_tets, 1))
    m.cell_type = np.zeros(m.n_tets, dtype=np.uint8)
    return m


def test_reduces_to_monodomain_when_tensors_are_proportional():
    lam = 2.5
    si = (1.2, 0.3)
    m = _slab(jitter=0.15)
    cen = m.centroids()
    ids = np.nonzero(cen[:, 0] < 0.5)[0].astype(np.int64)
    bd = BidomainOracle(m, si, (lam * si[0], lam * si[1]))
    bd.stimulus_set(0, ids, -52.0, 0.0, 1.0)
    mono = O.OracleSim(m.xyz, m.tets, m.fibre, None, lam * si[0] / (1 + lam), lam * si[1] / (1 + lam))
    mono.state_init(0, m.cell_type)
    mono.stimulus_set(0, ids, -52.0, 0.0, 1.0)
    dt = 0.02
    for _ in range(5):
        bd.step(40, dt); mono.step(40, dt)
        v = mono.read_vm()
        assert np.abs(bd.read_vm() - v).max() < 1e-8, np.abs(bd.read_vm() - v).max()
        vx = bd.read_vext()
        vol = bd.vol
        want = -(v - (vol * v).sum() / vol.sum()) / (1 + lam)
        assert np.abs(vx - want).max() < 1e-8
    assert v.max() > 0.0 and v.min() < -80.0          # a wave is under way: the comparison is not about a flat field
    assert np.array_equal(bd.activation_times() >= 0, mono.activation_times() >= 0)


def test_elliptic_equation_compatibility_and_gauge():
    m = _slab(nx=8, ny=5, nz=3, jitter=0.2)
    cen = m.centroids()
    th = np.deg2rad(-60 + 120 * cen[:, 2] / 0.75)
    m.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    bd = BidomainOracle(m, (1.7, 0.19), (6.2, 2.4))      # Table 2, mS/cm
    v = uniform(3, np.arange(m.n_tets), -85.0, 30.0)
    vx = bd.solve_vext(v)
    b = -bd.oi.apply_diffusion(v)
    assert abs((bd.vol * b).sum()) < 1e-12 * (bd.vol * np.abs(b)).sum()          # compatible right-hand side
    r = bd.oie.apply_diffusion(vx) - b
    assert np.abs(r).max() < 1e-9 * np.abs(b).max()                              # second equation of (6)
    assert abs((bd.vol * vx).sum()) < 1e-10 * (bd.vol * np.abs(vx)).sum()        # reading E1
    assert np.abs(bd.solve_vext(v + 17.0) - vx).max() < 1e-9 * np.abs(vx).max()  # constants are in the null space
    # v_ext opposes v (extracellular potential falls where the membrane depolarises): negative correlation
    assert np.corrcoef(vx, v)[0, 1] < -0.5
    # linearity
    v2 = uniform(4, np.arange(m.n_tets), -85.0, 30.0)
    assert np.abs(bd.solve_vext(2 * v - 3 * v2) - (2 * vx - 3 * bd.solve_vext(v2))).max() < 1e-8 * np.abs(vx).max()


def test_table2_bidomain_is_not_a_relabelled_monodomain():
    """Unequal anisotropy ratios (sigma_i 1.7/0.19, sigma_e 6.2/2.4 mS/cm): no single lambda exists; the bidomain front runs
    close to -- but not on -- the monodomain front with the harmonic-mean conductivities 1.334 / 0.176 mS/cm."""
    m = _slab(nx=20, ny=5, nz=2, h=0.25)
    cen = m.centroids()
    ids = np.nonzero(cen[:, 0] < 0.5)[0].astype(np.int64)
    si, se = (1.7, 0.19), (6.2, 2.4)
    bd = BidomainOracle(m, si, se)
    bd.stimulus_set(0, ids, -52.0, 0.0, 1.0)
    hm = tuple(a * b / (a + b) for a, b in zip(si, se))
    assert hm[0] == pytest.approx(1.334, abs=2e-3) and hm[1] == pytest.approx(0.176, abs=1e-3)     # reading A10
    mono = O.OracleSim(m.xyz, m.tets, m.fibre, None, hm[0], hm[1])
    mono.state_init(0, m.cell_type)
    mono.stimulus_set(0, ids, -52.0, 0.0, 1.0)
    bd.step(650, 0.02); mono.step(650, 0.02)
    ta_b, ta_m = bd.activation_times(), mono.activation_times()
    far = cen[:, 0] > 3.5
    assert (ta_b[far] >= 0).all() and (ta_m[far] >= 0).all()
    band = lambda x0: np.abs(cen[:, 0] - x0) < 0.25
    cv_b = 2.5 / (ta_b[band(4.0)].mean() - ta_b[band(1.5)].mean())
    cv_m = 2.5 / (ta_m[band(4.0)].mean() - ta_m[band(1.5)].mean())
    assert cv_b == pytest.approx(cv_m, rel=0.05) and 0.3 < cv_b < 0.8       # m/s, plane wave along the fibres
    assert np.abs(bd.read_vm() - mono.read_vm()).max() > 1e-3               # but it is a different solution
