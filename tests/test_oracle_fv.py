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


def test_two_tet_flux_by_hand(oracle):
    """Readings A6 (alpha weights) and A8 (M_f) pinned by a flux worked out by hand (numbers: tests/golden/two_tet_flux.json).

    Two tets share the face ABC, A=(0,0,0), B=(1,0,0), C=(0,1,0), in the plane z=0; cell 0 has apex P1=(0,0,1), cell 1 apex
    P2 below the plane.  v = (1, 0), sigma scale = (1, 0.1), sigma_l = 2, sigma_t = 0.5 mS/cm.  V_0 = 1/6; the area vector
    of the face outward of cell 0 is s = (0,0,-1/2); x_f = (1/3,1/3,0); x_c0 = (1/4,1/4,1/4), |x_f - x_c0| = sqrt(11)/12.

    Case A, P2=(0,0,-2), isotropic sigma_l: x_c1 = (1/4,1/4,-1/2), |x_f - x_c1| = sqrt(38)/12, so (A6)
      alpha_c1 = sqrt38/(sqrt11+sqrt38) = 0.65018...;  e = z-hat, d = 3/4.  Eq. (8) replaces the e-component of the averaged
      gradient by (v_c1 - v_c2)/d = 4/3 and e is parallel to s, so F = sigma_f (4/3)(-1/2) with (A8)
      sigma_f = 2 (alpha_c1 + 0.1 alpha_c2);  D_0 = 100 F / V_0 = -400 sigma_f = -548.132...,  D_1 = -100 F/V_1 = +200 sigma_f.
      (alpha swapped would give -331.9; a harmonic mean of the two tensors -192.8.)

    Case B, P2=(1,0,-2), fibre (1,0,1)/sqrt2 in both cells: x_c1 = (1/2,1/4,-1/2), V_1 = 1/3, e = (-1,0,3)/sqrt10, d = sqrt10/4,
      |x_f - x_c1| = sqrt(41)/12, alpha_c1 = sqrt41/(sqrt11+sqrt41) = 0.658775.
      Node values (P1 and P2 belong to one cell each): v_P1 = 1, v_P2 = 0,
        v_A = 3/(3+sqrt3) = 0.633975   (|A-x_c0| = sqrt3/4, |A-x_c1| = 3/4),
        v_B = 3/(3+sqrt11) = 0.474937  (sqrt11/4, 3/4),   v_C = sqrt17/(sqrt17+sqrt11) = 0.554201  (sqrt11/4, sqrt17/4).
      Gauss-Green with three-node face means = sum_n v_n grad(lambda_n):
        cell 0: lambda_B = x, lambda_C = y, lambda_P1 = z       -> grad v_c0 = (v_B-v_A, v_C-v_A, 1-v_A)
        cell 1: lambda_B = x+z/2, lambda_C = y, lambda_P2 = -z/2 -> grad v_c1 = (v_B-v_A, v_C-v_A, v_B/2)
      gbar = alpha_c1 grad v_c0 + alpha_c2 grad v_c1 = (-0.159037, -0.079774, 0.322159);
      eq. (8): g = gbar + [4/sqrt10 - gbar.e] e = (-0.446486, -0.079774, 1.184505);
      M_f = (alpha_c1 + 0.1 alpha_c2) [0.5 I + 1.5 f f^T]: (M g)_z = k (0.75 g_x + 1.25 g_z), k = 0.692898;
      F = (M_f g).s = -0.396949;  D_0 = 600 F = -238.169,  D_1 = -300 F = +119.085."""
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "two_tet_flux.json")))
    xyz = np.array(gold["nodes"], dtype=float)
    v = np.array(gold["v"])
    scale = np.array(gold["sigma_scale"])
    for case in ("case_A", "case_B"):
        g = gold[case]
        tets = np.array(g["tets"], np.int32)
        fib = None if g["fibre"] is None else np.tile(np.array(g["fibre"]), (2, 1))
        s = oracle.OracleSim(xyz, tets, fib, scale, g["sigma_l"], g["sigma_t"])
        D = s.apply_diffusion(v)
        assert D == pytest.approx(np.array(g["D"]), rel=1e-13), case
        if case == "case_B":
            vn = s.node_values(v)
            assert vn[:3] == pytest.approx(np.array(g["node_values_ABC"]), rel=1e-14)
            assert vn[3] == 1.0 and vn[5] == 0.0
            gr = s.cell_gradients(v)
            a1 = g["alpha_c1"]
            assert a1 * gr[0, 2] + (1 - a1) * gr[1, 2] == pytest.approx(g["gbar_z"], rel=1e-13)


def test_rotation_invariance(oracle):
    """div(M grad v) is a scalar: rotating the mesh and the fibres together (eq. (2)-(3): M = A M_hat A^T) must not change
    D_c.  Checked with the two proper axis permutations on the hand-worked two-tet case B (so that every component of
    M_f, not only the z row, meets the hand value) and with a general rotation on a jittered slab with conductivity
    contrasts (readings A8, A9)."""
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "two_tet_flux.json")))
    g = gold["case_B"]
    xyz = np.array(gold["nodes"], dtype=float)
    fib = np.tile(np.array(g["fibre"]), (2, 1))
    for perm in ([1, 2, 0], [2, 0, 1]):
        s = oracle.OracleSim(xyz[:, perm], np.array(g["tets"], np.int32), fib[:, perm], np.array(gold["sigma_scale"]),
                             g["sigma_l"], g["sigma_t"])
        assert s.apply_diffusion(np.array(gold["v"])) == pytest.approx(np.array(g["D"]), rel=1e-13), perm
    m, s0 = _jittered(oracle)
    from ep_inputs.prng import uniform
    scale = uniform(8, np.arange(m.n_tets), 0.1, 1.0)
    a, b, c = 0.7, -1.1, 0.4
    Rz = np.array([[np.cos(a), -np.sin(a), 0], [np.sin(a), np.cos(a), 0], [0, 0, 1]])
    Ry = np.array([[np.cos(b), 0, np.sin(b)], [0, 1, 0], [-np.sin(b), 0, np.cos(b)]])
    Rx = np.array([[1, 0, 0], [0, np.cos(c), -np.sin(c)], [0, np.sin(c), np.cos(c)]])
    R = Rz @ Ry @ Rx
    s1 = oracle.OracleSim(m.xyz @ R.T, m.tets, m.fibre @ R.T, scale, 1.3, 0.18)
    v = np.random.default_rng(9).uniform(-90, 40, m.n_tets)
    D0, D1 = s0.apply_diffusion(v), s1.apply_diffusion(v)
    assert np.abs(D0 - D1).max() <= 1e-10 * np.abs(D0).max()
