"""Pins of the two-dimensional cell-centred finite-volume operator in oracle/ep_oracle2d.cpp (the chain of
PAPER.md:164-168 on triangles) -- invariants, closed forms, a hand-worked two-triangle flux, a brute-force numpy assembly of
the same chain written independently, and the one number the paper prints for this medium: 3.95 mS/mm 'corresponding to a
velocity 4.0 m/s' (Table 2)."""
import numpy as np
import pytest

from ep_inputs import meshes as M
from ep_inputs.configs import purkinje_strip
from ep_inputs.prng import uniform
from oracle import ep_oracle2d as O2


def _flat(nx=12, ny=9, h=0.25, **kw):
    m = M.rect_tri(nx, ny, h)
    return m, O2.OracleSim2D(m.xyz, m.tris, **kw)


def _bumpy(seed=3):
    m = M.rect_tri(11, 8, 0.3)
    M.jitter_interior_tri(m, 0.06, seed, out_of_plane=0.05)
    cen = m.centroids()
    th = np.deg2rad(20 + 40 * cen[:, 0] / 3.3)
    m.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    m.sigma_scale = uniform(seed + 9, np.arange(m.n_tris), 0.2, 1.0)
    return m, O2.OracleSim2D(m.xyz, m.tris, m.fibre, m.sigma_scale, 2.0, 0.5)


def test_geometry():
    m, s = _flat()
    area, cen = s.geometry()
    assert np.allclose(area, 0.25 * 0.25 / 2, rtol=1e-14) and area.sum() == pytest.approx(12 * 9 * 0.0625, rel=1e-13)
    assert np.allclose(cen, m.centroids(), atol=1e-15)
    assert s.n_edges() == 3 * 12 * 9 - 12 - 9          # 2 nx ny diagonals+..., interior edges = (3 nx ny - nx - ny)


def test_uniform_field_gives_zero():
    for m, s in (_flat(), _bumpy()):
        D = s.apply_diffusion(np.full(m.n_tris, -86.2))
        scale = np.abs(s.apply_diffusion(uniform(1, np.arange(m.n_tris), -90, 30))).max()
        assert np.abs(D).max() < 1e-12 * scale


def test_conservation_under_no_flux():
    """sum_c A_c D_c = 0 for any field: interior edge fluxes are single-valued (reading D2), boundary edges carry none."""
    for m, s in (_flat(), _bumpy()):
        area, _ = s.geometry()
        v = uniform(4, np.arange(m.n_tris), -90.0, 40.0)
        D = s.apply_diffusion(v)
        assert abs((area * D).sum()) < 1e-12 * (area * np.abs(D)).sum()


def test_linear_field_on_the_uniform_flat_lattice():
    """v = a.x + b: node stars of the uniform lattice are centrally symmetric, so v_n is exact at interior nodes, the
    Gauss-Green gradient is exactly a in cells without a boundary node and D_c = 0 two squares away from the boundary."""
    m, s = _flat(nx=14, ny=11, h=0.2, sigma_l=1.7, sigma_t=1.7)
    a = np.array([0.7, -1.3, 0.0])
    cen = m.centroids()
    v = cen @ a + 2.0
    g = s.cell_gradients(v)
    onb = (m.xyz[:, 0] < 1e-9) | (m.xyz[:, 0] > 2.8 - 1e-9) | (m.xyz[:, 1] < 1e-9) | (m.xyz[:, 1] > 2.2 - 1e-9)
    inner = ~onb[m.tris].any(axis=1)
    assert np.abs(g[inner] - a).max() < 1e-12
    deep = (cen[:, 0] > 0.4) & (cen[:, 0] < 2.4) & (cen[:, 1] > 0.4) & (cen[:, 1] < 1.8)
    D = s.apply_diffusion(v)
    assert np.abs(D[deep]).max() < 1e-9 and np.abs(D[~deep]).max() > 1.0


def test_gauss_green_equals_the_barycentric_gradient():
    """(1/A) sum_j v_ej s_j with two-node edge means (reading D1) = gradient of the linear interpolant of the three nodal
    values, computed here by solving the 2 x 2 system in the triangle's own plane."""
    m, s = _bumpy()
    v = uniform(6, np.arange(m.n_tris), -80.0, 20.0)
    vn = s.node_values(v)
    g = s.cell_gradients(v)
    for c in range(0, m.n_tris, 7):
        p = m.xyz[m.tris[c]]
        e1, e2 = p[1] - p[0], p[2] - p[0]
        G = np.array([[e1 @ e1, e1 @ e2], [e1 @ e2, e2 @ e2]])
        rhs = np.array([vn[m.tris[c, 1]] - vn[m.tris[c, 0]], vn[m.tris[c, 2]] - vn[m.tris[c, 0]]])
        ab = np.linalg.solve(G, rhs)
        want = ab[0] * e1 + ab[1] * e2
        assert np.abs(g[c] - want).max() < 1e-10 * max(1.0, np.abs(want).max())


def test_node_values_are_inverse_distance_means():
    m, s = _bumpy()
    v = uniform(8, np.arange(m.n_tris), -80.0, 20.0)
    vn = s.node_values(v)
    cen = m.centroids()
    for n in (0, 5, 17, 40, m.n_nodes - 1):
        cells = np.nonzero((m.tris == n).any(axis=1))[0]
        w = 1.0 / np.linalg.norm(cen[cells] - m.xyz[n], axis=1)
        assert vn[n] == pytest.approx((w * v[cells]).sum() / w.sum(), rel=1e-13)


def test_two_triangle_flux_by_hand():
    """Unit square cut along its diagonal: T0 = (0,0),(1,0),(1,1), T1 = (0,0),(1,1),(0,1); v = (1, 0).
    Nodes: (0,0) and (1,1) are shared and equidistant from both centroids -> 1/2; (1,0) -> 1; (0,1) -> 0.  Both linear
    interpolants have gradient (1/2, -1/2).  Edge (0,0)-(1,1): s = (-1, 1) outward of T0, alpha = 1/2, centroids
    (2/3,1/3), (1/3,2/3): d = sqrt(2)/3, e = (1,-1)/sqrt(2); eq. (8): g = (1/2,-1/2) + [3/sqrt(2) - 1/sqrt(2)] e = (3/2,-3/2).
    M = diag(sl, st): flux = (M g).s = -(3/2)(sl + st); D_0 = 100 flux / (1/2) = -300 (sl + st), D_1 = +300 (sl + st)."""
    xyz = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0]], dtype=float)
    tris = np.array([[0, 1, 2], [0, 2, 3]], dtype=np.int32)
    fib = np.array([[1.0, 0, 0], [1.0, 0, 0]])
    sl, st = 1.3, 0.18
    s = O2.OracleSim2D(xyz, tris, fib, None, sl, st)
    v = np.array([1.0, 0.0])
    assert np.allclose(s.node_values(v), [0.5, 1.0, 0.5, 0.0], atol=1e-15)
    assert np.allclose(s.cell_gradients(v), [[0.5, -0.5, 0.0], [0.5, -0.5, 0.0]], atol=1e-14)
    D = s.apply_diffusion(v)
    assert D[0] == pytest.approx(-300.0 * (sl + st), rel=1e-13) and D[1] == pytest.approx(300.0 * (sl + st), rel=1e-13)
    D0 = s.apply_diffusion(v, use_corr=False)          # without eq. (8): g = (1/2,-1/2), flux = -(sl + st)/2
    assert D0[0] == pytest.approx(-100.0 * (sl + st), rel=1e-13)
    # swapped weights / tensors would show with unequal triangles: move node 3 to (0, 2)
    xyz2 = xyz.copy(); xyz2[3] = [0, 2, 0]
    s2 = O2.OracleSim2D(xyz2, tris, None, np.array([1.0, 3.0]), 1.0, 1.0)
    # T1 = (0,0),(1,1),(0,2): centroid (1/3, 1), area 1; edge midpoint (1/2,1/2): d0 = |(1/6,-1/6)| = sqrt(2)/6,
    # d1 = |(1/6,-1/2)| = sqrt(10)/6 -> alpha_0 = sqrt(10)/(sqrt(2)+sqrt(10)), M_f = alpha_0 * 1 + alpha_1 * 3
    a0 = np.sqrt(10.0) / (np.sqrt(2.0) + np.sqrt(10.0))
    Mf = a0 * 1.0 + (1 - a0) * 3.0
    vn = s2.node_values(v)
    w0 = np.array([3 / np.sqrt(5.0), 1.0])             # node (0,0): distances sqrt(5)/3 (T0) and sqrt(10)/3 (T1)
    w0 = np.array([1 / (np.sqrt(5.0) / 3), 1 / (np.sqrt(10.0) / 3)])
    assert vn[0] == pytest.approx(w0[0] / w0.sum(), rel=1e-14)
    g = s2.cell_gradients(v)
    gbar = a0 * g[0] + (1 - a0) * g[1]
    dc = np.array([2 / 3 - 1 / 3, 1 / 3 - 1.0, 0.0]); d = np.linalg.norm(dc); e = dc / d
    gf = gbar + ((1.0 - 0.0) / d - gbar @ e) * e
    flux = Mf * (gf @ np.array([-1.0, 1.0, 0.0]))
    D2 = s2.apply_diffusion(v)
    assert D2[0] == pytest.approx(100.0 * flux / 0.5, rel=1e-12) and D2[1] == pytest.approx(-100.0 * flux / 1.0, rel=1e-12)


def _numpy_operator(m, fibre, scale, sl, st):
    """The same chain assembled independently as a dense matrix with numpy (edge loop written from PAPER.md:164-168)."""
    nc, nn = m.n_tris, m.n_nodes
    X, T = m.xyz, m.tris
    cen = X[T].mean(axis=1)
    W = np.zeros((nn, nc))
    for c in range(nc):
        for n in T[c]:
            W[n, c] = 1.0 / np.linalg.norm(X[n] - cen[c])
    W /= W.sum(axis=1, keepdims=True)
    area = np.empty(nc); Gc = np.zeros((nc, 3, nn)); S = np.zeros((nc, 3, 3))
    for c in range(nc):
        p = X[T[c]]
        N = np.cross(p[1] - p[0], p[2] - p[0]); area[c] = 0.5 * np.linalg.norm(N); nu = N / np.linalg.norm(N)
        for j in range(3):
            a, b = [k for k in range(3) if k != j]
            sv = np.cross(p[b] - p[a], nu)
            if sv @ (0.5 * (p[a] + p[b]) - cen[c]) < 0:
                sv = -sv
            S[c, j] = sv
            for k in (a, b):
                Gc[c, :, T[c, k]] += 0.5 * sv / area[c]
    Gcell = Gc @ W                                          # [nc,3,nc]: cell gradient as a function of cell values
    Mten = np.empty((nc, 3, 3))
    for c in range(nc):
        f = fibre[c] / np.linalg.norm(fibre[c]) if fibre is not None else np.zeros(3)
        tt = st if fibre is not None else sl
        Mten[c] = (scale[c] if scale is not None else 1.0) * (tt * np.eye(3) + (sl - tt) * np.outer(f, f))
    A = np.zeros((nc, nc))
    edge = {}
    for c in range(nc):
        for j in range(3):
            a, b = [T[c, k] for k in range(3) if k != j]
            edge.setdefault((min(a, b), max(a, b)), []).append((c, j))
    for (a, b), lst in edge.items():
        if len(lst) != 2:
            continue
        (c1, j1), (c2, j2) = sorted(lst)
        xm = 0.5 * (X[a] + X[b])
        d1, d2 = np.linalg.norm(xm - cen[c1]), np.linalg.norm(xm - cen[c2])
        a1 = d2 / (d1 + d2); a2 = 1 - a1
        dc = cen[c1] - cen[c2]; d = np.linalg.norm(dc); e = dc / d
        gbar = a1 * Gcell[c1] + a2 * Gcell[c2]               # [3,nc]
        diff = np.zeros(nc); diff[c1] += 1.0 / d; diff[c2] -= 1.0 / d
        g = gbar + np.outer(e, diff - e @ gbar)
        Mf = a1 * Mten[c1] + a2 * Mten[c2]
        row = S[c1, j1] @ Mf @ g
        A[c1] += 100.0 * row / area[c1]
        A[c2] -= 100.0 * row / area[c2]
    return A


def test_dense_brute_force_against_independent_numpy_assembly():
    m, s = _bumpy(seed=11)
    A = _numpy_operator(m, m.fibre, m.sigma_scale, 2.0, 0.5)
    rng = np.random.default_rng(2)
    for _ in range(3):
        v = rng.normal(size=m.n_tris)
        assert np.allclose(s.apply_diffusion(v), A @ v, rtol=0, atol=1e-10 * np.abs(A).max())
    # spectrum: stable with eq. (8)
    ev = np.linalg.eigvals(A)
    assert ev.real.max() < 1e-9 * np.abs(ev).max() and (np.diag(A) < 0).all()


@pytest.mark.parametrize("kdir,fibre", [(0, (1.0, 0.0, 0.0)), (1, (1.0, 0.0, 0.0)), (0, (0.6, 0.8, 0.0))])
def test_cosine_mode_closed_form_second_order(kdir, fibre):
    """v = cos(pi x_k / L) is compatible with no-flux; div(M grad v) = -(k^T M k) v, M = st I + (sl - st) f f^T.  The
    Rayleigh quotient over cells two squares from the boundary converges at second order.  Fixes units, the
    tensor orientation and the area / length factors of the 2D chain."""
    sl, st = 2.0, 0.5
    f = np.array(fibre)
    Mten = st * np.eye(3) + (sl - st) * np.outer(f, f)
    L = 4.0
    errs = []
    for n in (16, 32):
        h = L / n
        dims = [8, 8]; dims[kdir] = n
        m = M.rect_tri(dims[0], dims[1], h)
        s = O2.OracleSim2D(m.xyz, m.tris, np.tile(f, (m.n_tris, 1)), None, sl, st)
        area, cen = s.geometry()
        k = np.zeros(3); k[kdir] = np.pi / L
        v = np.cos(cen @ k)
        D = s.apply_diffusion(v)
        lam = -100.0 * k @ Mten @ k
        ij = np.floor(cen[:, :2] / h).astype(int)
        layer = np.minimum(ij.min(axis=1), (np.array(dims) - 1 - ij).min(axis=1))
        inner = layer >= 2
        errs.append(abs((area * v * D)[inner].sum() / (area * v * v)[inner].sum() / lam - 1.0))
    assert errs[0] < 0.02 and errs[1] < 0.005 and errs[1] < errs[0] / 2.5, errs


def test_rotating_the_sheet_in_space_changes_nothing():
    """Reading D2: nothing in the chain refers to the global axes; a rigidly rotated flat sheet gives the same operator."""
    m, s = _bumpy(seed=4)
    th = 0.7
    R = np.array([[np.cos(th), 0, np.sin(th)], [0, 1, 0], [-np.sin(th), 0, np.cos(th)]]) @ \
        np.array([[1, 0, 0], [0, np.cos(1.1), -np.sin(1.1)], [0, np.sin(1.1), np.cos(1.1)]])
    s2 = O2.OracleSim2D(m.xyz @ R.T, m.tris, m.fibre @ R.T, m.sigma_scale, 2.0, 0.5)
    v = uniform(12, np.arange(m.n_tris), -80.0, 30.0)
    a, b = s.apply_diffusion(v), s2.apply_diffusion(v)
    assert np.abs(a - b).max() < 1e-10 * np.abs(a).max()


def test_purkinje_conduction_velocity_matches_table_2():
    """Table 2: '2D Purkinje network, Stewart, isotropic monodomain, 3.95 mS/mm, corresponding to a velocity
    4.0 m/s'.  Plane wave along the 20 x 7 mm sheet at dx = 0.5 mm: 4.0 m/s within 5 %.  (chi = 140 /mm, C_m = 0.01 uF/mm^2,
    PAPER.md:113.)  Pins the 2D operator, the Stewart upstroke and the unit chain together against a number the paper prints."""
    prob = purkinje_strip(0.5)
    o = O2.OracleSim2D.from_problem(prob)
    o.step(3200, 0.0025)                                # 8 ms
    ta = o.activation_times()
    cen = prob.mesh.centroids()
    assert (ta >= 0).all()
    band = lambda x0: np.abs(cen[:, 0] - x0) < 0.5
    cv = 10.0 / (ta[band(15.0)].mean() - ta[band(5.0)].mean())      # mm/ms = m/s
    assert cv == pytest.approx(4.0, rel=0.05), cv


def test_step_level_semantics_on_uncoupled_cells():
    """sigma_scale = 0 uncouples the cells, so each one must follow the single-cell recurrence exactly: stimulus window on
    integer steps [n_on, n_off) (A16), I_s/C_m (C_m = 2 here), activation time = (n+1) dt of the first step that exceeds 0 mV
    (A18), -1 where it never does within the run."""
    m = M.rect_tri(2, 1, 0.5)
    m.xyz[3, 0] += 0.2                                       # node (1,1) moved: unequal areas, the stimulated cell included
    s = O2.OracleSim2D(m.xyz, m.tris, None, np.zeros(m.n_tris), 1.0, 1.0, chi=1400.0, Cm=2.0)
    s.state_init()
    dt = 0.01
    s.stimulus_set(0, [1], -104.0, 0.5, 1.0)                 # -104 uA/cm^2 over C_m = 2 -> -52 uA/uF on steps 50..149
    s.step(400, dt)
    y1, tr1 = O2.stw_run(O2.stw_init(), dt, 400, istim=-52.0, n_on=50, n_off=150, trace=True)
    y0, tr0 = O2.stw_run(O2.stw_init(), dt, 400, trace=True)
    assert s.read_vm()[1] == y1[0] and s.read_vm()[0] == y0[0] and s.read_vm()[2] == y0[0]
    for k in range(20):
        assert s.read_state(k)[1] == y1[k]
    n_cross = int(np.nonzero((tr1[:-1] <= 0) & (tr1[1:] > 0))[0][0])
    ta = s.activation_times()
    assert ta[1] == (n_cross + 1) * dt and ta[0] == -1.0 and ta[3] == -1.0
    p = m.xyz[m.tris]
    area = 0.5 * np.abs(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0])[:, 2])
    assert area.max() > 1.5 * area.min()
    v = np.array([y0[0], y1[0], y0[0], y0[0]])
    assert s.mean_vm() == pytest.approx((area * v).sum() / area.sum(), rel=1e-14)
