"""Pins for the oracle's finite-volume diffusion operator (Fig. 8, eq. (7)-(8)).

None of these re-types the oracle's pipeline: they check it against invariants (row sums, conservation),
closed forms (linear field, cosine modes with the analytic -k^T M k eigenvalue, including the mm->cm unit factor and
the fibre-tensor orientation), a textbook identity (barycentric-gradient form of Gauss-Green) and spectral facts.
"""
import json
import os

import numpy as np
import pytest

from ep_inputs import meshes as M
from ep_inputs import make

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


def _uniform(oracle, n=6, h=1.0, fibre=(1.0, 0.0, 0.0), sl=1.3, st=0.18, dims=None):
    dims = dims or (n, n, n)
    m = M.kuhn_slab(*dims, h)
    f = np.tile(np.asarray(fibre, dtype=float), (m.n_tets, 1))
    return m, oracle.OracleSim(m.xyz, m.tets, f, None, sl, st)


def _jittered(oracle, seed=7):
    m = M.kuhn_slab(7, 5, 4, 0.3)
    M.jitter_interior(m, 0.2 * 0.3, seed)
    cen = m.centroids()
    th = np.deg2rad(-60 + 120 * cen[:, 2] / 1.2)
    m.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    from ep_inputs.prng import uniform
    scale = uniform(seed + 1, np.arange(m.n_tets), 0.1, 1.0)
    return m, oracle.OracleSim(m.xyz, m.tets, m.fibre, scale, 1.3, 0.18)


def test_mesh_generator_matches_paper_cell_counts():
    """PAPER.md:238-240 (Table 1): 20x7x3 mm at dx 0.5/0.2/0.1 mm -> 20,160 / 315,000 / 2,520,000 cells = 6 per cube."""
    for dx, n in GOLD["slab_cell_counts"]["value"].items():
        dx = float(dx)
        cubes = round(20 / dx) * round(7 / dx) * round(3 / dx)
        assert 6 * cubes == n
    assert make(2).mesh.n_tets == 315000
    assert make(6).mesh.n_tets == 20160 and make(7).mesh.n_tets == 315000      # the paper's own slab (configs 6-8)
    assert make(1).mesh.n_tets == 9600 and make(1).mesh.n_nodes == 2205


def test_geometry_volume_and_partition(oracle):
    m, s = _jittered(oracle)
    vol, cen = s.geometry()
    assert np.all(vol > 0)
    assert abs(vol.sum() - 7 * 5 * 4 * 0.3 ** 3) < 1e-12          # tets tile the box exactly
    assert np.allclose(cen, m.xyz[m.tets].mean(axis=1), atol=1e-15)
    # interior faces = (4*cells - boundary faces)/2
    info = M.validate(m)
    assert s.n_faces() == info["n_faces"] - info["n_boundary_faces"]


def test_uniform_field_gives_zero(oracle):
    """P1: weights sum to one, sum S n = 0, eq. (8) correction vanishes -> D(const) = 0."""
    for m, s in (_uniform(oracle), _jittered(oracle)):
        one = np.full(m.n_tets, -86.2)
        D = s.apply_diffusion(one)
        scale = np.abs(s.apply_diffusion(np.sin(np.arange(m.n_tets)))).max()
        assert np.abs(D).max() <= 1e-12 * scale


def test_conservation_no_flux(oracle):
    """P2: fluxes are single-valued on interior faces and zero on the boundary => sum V_c D_c = 0."""
    m, s = _jittered(oracle)
    vol, _ = s.geometry()
    rng = np.random.default_rng(3)
    for _ in range(3):
        v = rng.uniform(-90, 40, m.n_tets)
        D = s.apply_diffusion(v)
        assert abs((vol * D).sum()) <= 1e-13 * (vol * np.abs(D)).sum()


def test_linear_field_uniform_lattice(oracle):
    """P3: on the uniform Kuhn lattice node stars are centrally symmetric, so v = a.x+b gives grad v_c = a exactly for
    cells with no boundary node and D_c = 0 two cube layers inside. ('provided the grid is regular'.)"""
    n = 6
    m, s = _uniform(oracle, n=n)
    _, cen = s.geometry()
    a = np.array([0.7, -0.4, 0.9])
    v = cen @ a + 2.0
    g = s.cell_gradients(v)
    ijk = np.rint(m.xyz).astype(int)
    bnode = ((ijk == 0) | (ijk == n)).any(axis=1)
    inner = ~bnode[m.tets].any(axis=1)
    assert inner.sum() > 0
    assert np.abs(g[inner] - a).max() < 1e-13
    D = s.apply_diffusion(v)
    layer = np.minimum(np.floor(cen).min(axis=1), (n - 1 - np.floor(cen)).min(axis=1))
    assert np.abs(D[layer >= 2]).max() < 1e-10
    assert np.abs(D[layer == 0]).max() > 1.0     # the missing boundary flux shows up at the boundary layer


def test_gauss_green_equals_barycentric_gradient(oracle):
    """P4: (1/V) sum_j v_fj S_j n_j with v_f = mean of 3 nodal values == sum_n v_n grad(lambda_n), grad(lambda) = rows of
    inv([x1-x0, x2-x0, x3-x0]) (textbook P1 finite-element identity). Checks face/vertex indexing and orientation."""
    m, s = _jittered(oracle)
    rng = np.random.default_rng(5)
    v = rng.uniform(-90, 40, m.n_tets)
    vn = s.node_values(v)
    g = s.cell_gradients(v)
    x = m.xyz[m.tets]                                           # [N,4,3]
    E = np.stack([x[:, 1] - x[:, 0], x[:, 2] - x[:, 0], x[:, 3] - x[:, 0]], axis=1)   # rows = edges
    Einv = np.linalg.inv(E)                                     # columns = grad lambda_1..3
    dv = np.stack([vn[m.tets[:, k]] - vn[m.tets[:, 0]] for k in (1, 2, 3)], axis=1)
    g_ref = np.einsum("nij,nj->ni", Einv, dv)
    assert np.abs(g - g_ref).max() <= 1e-10 * np.abs(g_ref).max()


def test_node_interpolation_is_convex_inverse_distance(oracle):
    """v_n is a convex combination; for a field equal to 1 on one cell the weight is (1/d)/sum(1/d)."""
    m, s = _jittered(oracle)
    _, cen = s.geometry()
    c = 123
    e = np.zeros(m.n_tets)
    e[c] = 1.0
    w = s.node_values(e)
    touched = np.nonzero(w)[0]
    assert set(touched) == set(m.tets[c])
    for n in touched:
        star = np.nonzero((m.tets == n).any(axis=1))[0]
        invd = 1.0 / np.linalg.norm(cen[star] - m.xyz[n], axis=1)
        assert abs(w[n] - (1.0 / np.linalg.norm(cen[c] - m.xyz[n])) / invd.sum()) < 1e-14
    v = np.random.default_rng(0).uniform(-90, 40, m.n_tets)
    vn = s.node_values(v)
    assert vn.min() >= v.min() and vn.max() <= v.max()


@pytest.mark.parametrize("fibre,kdir", [((1.0, 0.0, 0.0), 0), ((0.0, 1.0, 0.0), 0), ((1.0, 0.0, 0.0), 1),
                                         ((np.sqrt(0.5), np.sqrt(0.5), 0.0), 0)])
def test_cosine_mode_closed_form_second_order(oracle, fibre, kdir):
    """P7 / PAPER.md:172,:232: for v = cos(pi x_k / L) (no-flux compatible) div(M grad v) = -(k^T M k) v with
    M = sigma_t I + (sigma_l - sigma_t) f f^T (eq. (2)-(3)); the discrete operator converges to it at ~2nd order.
    Units: sigma [mS/cm] * v [mV] / mm^2 * 100 = uA/cm^3. Catches wrong tensor orientation, sign, factor, units."""
    sl, st = 1.3, 0.18
    f = np.asarray(fibre)
    Mten = st * np.eye(3) + (sl - st) * np.outer(f, f)
    L = 4.0
    errs = []
    for n in (16, 32):
        h = L / n
        dims = [6, 6, 6]
        dims[kdir] = n
        m, s = _uniform(oracle, h=h, fibre=fibre, dims=tuple(dims))
        vol, cen = s.geometry()
        kvec = np.zeros(3)
        kvec[kdir] = np.pi / L
        v = np.cos(cen @ kvec)
        D = s.apply_diffusion(v)
        lam = -100.0 * kvec @ Mten @ kvec
        # Cell-centred FV on tets is not pointwise consistent (per-tet truncation error is O(1) on the Kuhn lattice) but
        # is supra-convergent in the mean: compare the volume-weighted Rayleigh quotient over cells >= 2 cube layers
        # from the boundary (where the one-sided node interpolation, reading A3, does not reach).
        ijk = np.floor(cen / h).astype(int)
        layer = np.minimum(ijk.min(axis=1), (np.array(dims) - 1 - ijk).min(axis=1))
        inner = layer >= 2
        lam_h = (vol * v * D)[inner].sum() / (vol * v * v)[inner].sum()
        errs.append(abs(lam_h / lam - 1.0))
    assert errs[0] < 0.02, errs
    assert errs[1] < 0.005 and errs[1] < errs[0] / 2.0, errs      # ~2nd order (ratio 4 ideal)


def test_spectrum_stable_only_with_eq8(oracle):
    """P5: dense operator by brute force (unit vectors). With eq. (8) every eigenvalue has Re <= 0 and the diagonal is
    negative; dropping the correction (PAPER.md:166 'improve the stability') produces a positive eigenvalue."""
    m, s = _uniform(oracle, n=4)
    N = m.n_tets
    A = np.zeros((N, N))
    A0 = np.zeros((N, N))
    for k in range(N):
        e = np.zeros(N)
        e[k] = 1.0
        A[:, k] = s.apply_diffusion(e)
        A0[:, k] = s.apply_diffusion(e, use_corr=False)
    vol, _ = s.geometry()
    assert np.abs(A.sum(axis=1)).max() < 1e-12 * np.abs(A).max()
    assert np.abs(vol @ A).max() < 1e-12 * np.abs(A).max() * vol.mean()
    assert (np.diag(A) < 0).all()
    ev = np.linalg.eigvals(A)
    assert ev.real.max() < 1e-9 * np.abs(ev).max()
    ev0 = np.linalg.eigvals(A0)
    assert ev0.real.max() > 1e-4 * np.abs(ev).max()      # clearly positive (round-off level is ~1e-15 rho)
    # linearity of the operator: A (a u + b w) = a A u + b A w
    rng = np.random.default_rng(1)
    u, w = rng.normal(size=N), rng.normal(size=N)
    assert np.allclose(s.apply_diffusion(2 * u - 3 * w), A @ (2 * u - 3 * w), rtol=0, atol=1e-10 * np.abs(A).max())


def test_stencil_reach(oracle):
    """P6 / PAPER.md:166: the face gradient uses 'all the cells sharing the nodes of the two cells c1 and c2'."""
    m, s = _uniform(oracle, n=6)
    _, cen = s.geometry()
    c = int(np.argmin(((cen - 3.0) ** 2).sum(axis=1)))
    e = np.zeros(m.n_tets)
    resp = np.zeros(m.n_tets, dtype=bool)
    # column probing is expensive; use the transpose trick on a few random fields instead: row c of A touches cell k iff
    # perturbing v_k changes D_c
    base = np.zeros(m.n_tets)
    D0 = s.apply_diffusion(base)[c]
    tets = m.tets
    nbrs = [k for k in range(m.n_tets) if k != c and len(set(tets[k]) & set(tets[c])) == 3]
    reach_nodes = set(tets[c])
    for k in nbrs:
        reach_nodes |= set(tets[k])
    reach = np.nonzero(np.isin(tets, list(reach_nodes)).any(axis=1))[0]
    for k in range(m.n_tets):
        e[:] = 0
        e[k] = 1.0
        resp[k] = abs(s.apply_diffusion(e)[c] - D0) > 0
    assert len(nbrs) == 4 and len(reach_nodes) == 8
    assert set(np.nonzero(resp)[0]) <= set(reach)
    assert resp.sum() >= 60


def test_scaling_and_isotropic_default(oracle):
    """sigma_scale multiplies the tensor (config 4 scar); fibre=None means isotropic sigma_l (ABI statement)."""
    m = M.kuhn_slab(4, 4, 4, 0.5)
    v = np.random.default_rng(2).uniform(-90, 40, m.n_tets)
    iso = oracle.OracleSim(m.xyz, m.tets, None, None, 0.7, 0.1)
    f = np.tile([0.0, 0.0, 1.0], (m.n_tets, 1))
    same = oracle.OracleSim(m.xyz, m.tets, f, None, 0.7, 0.7)
    assert np.allclose(iso.apply_diffusion(v), same.apply_diffusion(v), rtol=1e-13, atol=1e-9)
    half = oracle.OracleSim(m.xyz, m.tets, f, np.full(m.n_tets, 0.5), 0.7, 0.7)
    assert np.allclose(half.apply_diffusion(v), 0.5 * same.apply_diffusion(v), rtol=1e-13, atol=1e-9)
    # tet vertex order / orientation must not matter
    t2 = m.tets[:, [1, 0, 2, 3]].copy()
    flipped = oracle.OracleSim(m.xyz, t2, f, None, 0.7, 0.7)
    assert np.allclose(flipped.apply_diffusion(v), same.apply_diffusion(v), rtol=1e-12, atol=1e-9)
