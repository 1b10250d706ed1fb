"""Host preprocessor (ep_host_stencil, no GPU): the factored 8-node + 4-neighbour gather must reproduce the oracle's
literal Fig. 8 pipeline on random fields, and its tables must have the structure DESIGN.md states."""
import numpy as np
import pytest

from ep_inputs import make
from ep_inputs import meshes as M
from ep_inputs.prng import uniform


def _apply(st, v, chi_cm):
    """Evaluate the factored stencil with numpy (test code; the product evaluates it in the CUDA kernels)."""
    nn = st["node_ptr"].size - 1
    deg = np.diff(st["node_ptr"])
    owner = np.repeat(np.arange(nn), deg)
    vn = np.zeros(nn)
    np.add.at(vn, owner, st["w"] * v[st["node_cell"]])
    dv = (st["a"] * vn[st["node"]]).sum(axis=1) + (st["b"] * (v[st["nbr"]] - v[:, None])).sum(axis=1)
    return dv * chi_cm, vn


def _cases():
    m = M.kuhn_slab(7, 5, 4, 0.3)
    M.jitter_interior(m, 0.06, 11)
    cen = m.centroids()
    th = np.deg2rad(-60 + 120 * cen[:, 2] / 1.2)
    m.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    m.sigma_scale = uniform(12, np.arange(m.n_tets), 0.1, 1.0)
    yield "jittered_slab", m
    p3 = make(3, coarsen=6.0).mesh
    yield "lv_shell_coarse", p3
    p5 = make(5, coarsen=4.0).mesh
    yield "atrial_shell_coarse", p5


@pytest.mark.parametrize("name,mesh", list(_cases()))
def test_factored_stencil_equals_oracle_operator(oracle, name, mesh):
    import paper_2112_12854_b200 as ep
    chi, Cm = 1400.0, 1.0
    st = ep.host_stencil(mesh.xyz, mesh.tets, mesh.fibre, mesh.sigma_scale, 1.3, 0.18, chi, Cm)
    osim = oracle.OracleSim(mesh.xyz, mesh.tets, mesh.fibre, mesh.sigma_scale, 1.3, 0.18, chi, Cm)
    for seed in (1, 2):
        v = uniform(seed, np.arange(mesh.n_tets), -90.0, 40.0)
        D_o = osim.apply_diffusion(v)
        D_h, vn = _apply(st, v, chi * Cm)
        scale = np.abs(D_o).max()
        assert np.abs(D_h - D_o).max() <= 1e-12 * scale, name
        assert np.abs(vn - osim.node_values(v)).max() <= 1e-13 * 90.0
    # structure
    nc = mesh.n_tets
    assert np.all(st["node"][:, :4] == mesh.tets)                  # own nodes first
    bnd = st["nbr"] == np.arange(nc)[:, None]
    assert np.all(st["b"][bnd] == 0.0)                             # no-flux boundary faces (reading A11)
    assert np.mean(st["b"][~bnd] > 0.0) > 0.9                      # two-point part: mostly positive weights
    # neighbour relation is symmetric
    for j in range(4):
        nb = st["nbr"][:, j]
        back = (st["nbr"][nb] == np.arange(nc)[:, None]).any(axis=1)
        assert np.all(back)
    # row sums vanish (uniform field -> zero), weights are convex
    assert np.abs(st["a"].sum(axis=1)).max() <= 1e-12 * np.abs(st["a"]).max()
    assert np.all(st["w"] > 0)
    # permutation is a bijection
    assert np.array_equal(np.sort(st["perm"]), np.arange(nc))


def test_morton_order_is_local():
    """Cells adjacent in device order are close in space (what the gather locality of the kernels relies on)."""
    import paper_2112_12854_b200 as ep
    p = make(1)
    st = ep.host_stencil(p.mesh.xyz, p.mesh.tets, p.mesh.fibre)
    cen = p.mesh.centroids()[st["perm"]]
    step = np.linalg.norm(np.diff(cen, axis=0), axis=1)
    assert np.median(step) < 0.25 and np.mean(step) < 0.5          # cube edge is 0.25 mm; slab is 5 mm wide
    inv = np.empty_like(st["perm"])
    inv[st["perm"]] = np.arange(inv.size)
    bnd = st["nbr"] == np.arange(inv.size)[:, None]
    dist = np.abs(inv[st["nbr"]] - inv[:, None])[~bnd]
    assert np.median(dist) <= 8


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


def _tri_cases():
    m = M.rect_tri(13, 9, 0.3)
    M.jitter_interior_tri(m, 0.06, 5, out_of_plane=0.05)
    cen = m.centroids()
    th = np.deg2rad(10 + 50 * cen[:, 1] / 2.7)
    m.fibre = np.stack([np.cos(th), np.sin(th), 0 * th], axis=1)
    m.sigma_scale = uniform(14, np.arange(m.n_tris), 0.1, 1.0)
    yield "bumpy_sheet", m, 2.0, 0.5
    yield "purkinje_surface_coarse", M.ellipsoid_surface((25.0, 25.0, 50.0), 20.0, 3.0), 39.5, 39.5


@pytest.mark.parametrize("name,mesh,sl,st_", list(_tri_cases()))
def test_factored_stencil_of_a_triangulated_surface_equals_the_2d_oracle(name, mesh, sl, st_):
    """ep_host_stencil_tri against the edge-walking 2D oracle on random fields; table structure."""
    import paper_2112_12854_b200 as ep
    from oracle import ep_oracle2d as O2
    chi, Cm = 1400.0, 1.0
    st = ep.host_stencil_tri(mesh.xyz, mesh.tris, mesh.fibre, mesh.sigma_scale, sl, st_, chi, Cm)
    osim = O2.OracleSim2D(mesh.xyz, mesh.tris, mesh.fibre, mesh.sigma_scale, sl, st_, chi, Cm)
    for seed in (1, 2):
        v = uniform(seed, np.arange(mesh.n_tris), -90.0, 40.0)
        D_o = osim.apply_diffusion(v)
        D_h, vn = _apply(st, v, chi * Cm)
        assert np.abs(D_h - D_o).max() <= 1e-12 * np.abs(D_o).max(), name
        assert np.abs(vn - osim.node_values(v)).max() <= 1e-13 * 90.0
    nc = mesh.n_tris
    assert np.all(st["node"][:, :3] == mesh.tris)                  # own nodes first
    assert np.all(st["a"][:, 6:] == 0.0) and np.all(st["b"][:, 3] == 0.0)     # 3 + 3 nodes, 3 neighbours
    bnd = st["nbr"] == np.arange(nc)[:, None]
    assert np.all(st["b"][bnd] == 0.0)
    assert np.abs(st["a"].sum(axis=1)).max() <= 1e-9 * np.abs(st["a"]).max()  # uniform field -> zero
    deg = np.diff(st["node_ptr"])
    assert deg.sum() == 3 * nc and deg.min() >= 1
    assert sorted(st["perm"].tolist()) == list(range(nc))


def test_triangle_mesh_errors():
    import paper_2112_12854_b200 as ep
    m = M.rect_tri(2, 2, 1.0)
    bad = m.tris.copy(); bad[0, 0] = 99
    with pytest.raises(ep.EpError) as e:
        ep.host_stencil_tri(m.xyz, bad)
    assert e.value.code == -2
    flat = m.xyz.copy(); flat[:, 1] = 0.0                          # every triangle degenerate
    with pytest.raises(ep.EpError):
        ep.host_stencil_tri(flat, m.tris)
    three = np.vstack([m.tris, [[0, 1, 8]], [[0, 1, 7]]]).astype(np.int32)     # edge (0,1) now in three triangles
    with pytest.raises(ep.EpError):
        ep.host_stencil_tri(m.xyz, three)
