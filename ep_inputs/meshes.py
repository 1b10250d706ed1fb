"""Seeded synthetic tetrahedral meshes shaped like the paper's workloads.

Everything here is input generation only: lattice points, the Kuhn/Freudenthal split of a cube into six
tetrahedra (reading A12: only the counts 20,160 / 315,000 / 2,520,000 = 6 x cubes are printed),
carving of ellipsoidal shells out of the lattice, fibre fields by the paper's transmural rule
(alpha = alpha_endo*d + alpha_epi*(1-d), +-60 degrees) and cell-type bands.
No finite-volume or cell-model arithmetic lives here; both the oracle tests and the CUDA path consume these arrays.
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

from .prng import uniform

# The six Kuhn simplices of the unit cube: one per permutation of the axes; all share the (0,0,0)-(1,1,1) diagonal.
_KUHN_PERMS = list(itertools.permutations((0, 1, 2)))


@dataclass
class TetMesh:
    xyz: np.ndarray            # [n_nodes,3] float64, mm
    tets: np.ndarray           # [n_tets,4] int32, 0-based
    fibre: np.ndarray | None = None        # [n_tets,3] float64 (unit) or None = isotropic
    cell_type: np.ndarray | None = None    # [n_tets] uint8: 0 endo, 1 mid, 2 epi
    sigma_scale: np.ndarray | None = None  # [n_tets] float64 or None
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def n_tets(self) -> int:
        return int(self.tets.shape[0])

    def centroids(self) -> np.ndarray:
        return self.xyz[self.tets].mean(axis=1)


def _kuhn_tets_of_cubes(ci, cj, ck, nx, ny, nz) -> np.ndarray:
    """Tets (node ids in the full (nx+1)(ny+1)(nz+1) lattice, x fastest) of the listed cubes. [6*M,4] int64."""
    sx, sy, sz = 1, nx + 1, (nx + 1) * (ny + 1)
    strides = np.array([sx, sy, sz], dtype=np.int64)
    base = ci.astype(np.int64) * sx + cj.astype(np.int64) * sy + ck.astype(np.int64) * sz
    out = np.empty((base.shape[0], 6, 4), dtype=np.int64)
    for t, p in enumerate(_KUHN_PERMS):
        out[:, t, 0] = base
        out[:, t, 1] = base + strides[p[0]]
        out[:, t, 2] = base + strides[p[0]] + strides[p[1]]
        out[:, t, 3] = base + sx + sy + sz
    return out.reshape(-1, 4)


def lattice_nodes(nx, ny, nz, h, origin=(0.0, 0.0, 0.0)) -> np.ndarray:
    k, j, i = np.meshgrid(np.arange(nz + 1), np.arange(ny + 1), np.arange(nx + 1), indexing="ij")
    xyz = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1).astype(np.float64) * h
    return xyz + np.asarray(origin, dtype=np.float64)


def kuhn_slab(nx: int, ny: int, nz: int, h: float) -> TetMesh:
    """Box [0,nx*h]x[0,ny*h]x[0,nz*h] cut into nx*ny*nz cubes of edge h, six Kuhn tets each."""
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    tets = _kuhn_tets_of_cubes(i.ravel(), j.ravel(), k.ravel(), nx, ny, nz)
    xyz = lattice_nodes(nx, ny, nz, h)
    return TetMesh(xyz=xyz, tets=tets.astype(np.int32), meta={"kind": "kuhn_slab", "dims": (nx, ny, nz), "h": h})


def jitter_interior(mesh: TetMesh, amplitude: float, seed: int) -> None:
    """Move interior lattice nodes by U(-amplitude, amplitude) per axis (reading G3); boundary nodes stay put."""
    nx, ny, nz = mesh.meta["dims"]
    h = mesh.meta["h"]
    ijk = np.rint(mesh.xyz / h).astype(np.int64)
    interior = ((ijk[:, 0] > 0) & (ijk[:, 0] < nx) & (ijk[:, 1] > 0) & (ijk[:, 1] < ny)
                & (ijk[:, 2] > 0) & (ijk[:, 2] < nz))
    n = mesh.n_nodes
    ctr = np.arange(n, dtype=np.uint64)
    for ax in range(3):
        d = uniform(seed, ctr * np.uint64(3) + np.uint64(ax), -amplitude, amplitude)
        mesh.xyz[:, ax] += np.where(interior, d, 0.0)
    mesh.meta["jitter"] = amplitude


def carve_lattice(inside, lo, hi, h: float) -> TetMesh:
    """Keep the cubes of an h-lattice over the box [lo,hi] whose centre satisfies inside(xyz)->bool; Kuhn-split
    them; renumber the nodes that are used. Conforming by construction (same split in every cube)."""
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    dims = np.maximum(1, np.ceil((hi - lo) / h - 1e-9).astype(np.int64))
    nx, ny, nz = (int(d) for d in dims)
    keep_i, keep_j, keep_k = [], [], []
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    for k in range(nz):  # slab by slab keeps the temporary arrays small for the 20M-cell config
        c = np.stack([lo[0] + (ii.ravel() + 0.5) * h, lo[1] + (jj.ravel() + 0.5) * h,
                      np.full(ii.size, lo[2] + (k + 0.5) * h)], axis=1)
        m = inside(c)
        keep_i.append(ii.ravel()[m])
        keep_j.append(jj.ravel()[m])
        keep_k.append(np.full(int(m.sum()), k, dtype=np.int64))
    ci, cj, ck = np.concatenate(keep_i), np.concatenate(keep_j), np.concatenate(keep_k)
    tets_full = _kuhn_tets_of_cubes(ci, cj, ck, nx, ny, nz)
    used, inv = np.unique(tets_full.ravel(), return_inverse=True)
    tets = inv.reshape(-1, 4).astype(np.int32)
    sy, sz = nx + 1, (nx + 1) * (ny + 1)
    xyz = np.stack([used % sy, (used // sy) % (ny + 1), used // sz], axis=1).astype(np.float64) * h + lo
    return TetMesh(xyz=xyz, tets=tets, meta={"kind": "carved", "h": h, "dims": (nx, ny, nz), "n_cubes": int(ci.size)})


# ----------------------------------------------------------------------------------------------------------
# ellipsoidal shells


def shell_depth(p: np.ndarray, centre, inner, outer, iters: int = 60) -> np.ndarray:
    """Transmural coordinate d in [0,1] (0 = inner/endocardial surface, 1 = outer/epicardial): the t for which p
    lies on the ellipsoid with semi-axes inner + t*(outer-inner). Bisection; values outside the wall are clipped.
    Worked through in cache-sized chunks (the 20M-cell config calls this on every cell)."""
    c = np.asarray(centre, dtype=np.float64)
    a0 = np.asarray(inner, dtype=np.float64)
    da = np.asarray(outer, dtype=np.float64) - a0
    n = p.shape[0]
    out = np.empty(n)
    chunk = 1 << 15

    def work(s):
        q = p[s:s + chunk] - c
        qx, qy, qz = (np.ascontiguousarray(q[:, k]) for k in range(3))
        lo = np.full(qx.shape[0], -0.5)
        hi = np.full(qx.shape[0], 1.5)
        for _ in range(iters):
            mid = 0.5 * (lo + hi)
            # >0: p is outside the level-mid ellipsoid => the true t is larger
            g = ((qx / (a0[0] + mid * da[0])) ** 2 + (qy / (a0[1] + mid * da[1])) ** 2) + (qz / (a0[2] + mid * da[2])) ** 2 - 1.0
            up = g > 0
            lo = np.where(up, mid, lo)
            hi = np.where(up, hi, mid)
        out[s:s + chunk] = 0.5 * (lo + hi)

    starts = range(0, n, chunk)
    if n > 8 * chunk:      # numpy releases the GIL inside its loops: chunks are independent, the result is the same
        from concurrent.futures import ThreadPoolExecutor
        import os
        with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
            list(ex.map(work, starts))
    else:
        for s0 in starts:
            work(s0)
    return np.clip(out, 0.0, 1.0)


def ellipsoid_frame(p: np.ndarray, centre, axes):
    """Unit (normal, circumferential, longitudinal) directions of the ellipsoid family through p; the long axis is z."""
    q = p - np.asarray(centre, dtype=np.float64)
    n = q / (np.asarray(axes, dtype=np.float64) ** 2)[None, :]
    n /= np.maximum(np.linalg.norm(n, axis=1, keepdims=True), 1e-300)
    zhat = np.array([0.0, 0.0, 1.0])
    circ = np.cross(zhat[None, :], n)
    nc = np.linalg.norm(circ, axis=1)
    bad = nc < 1e-9
    circ[bad] = np.array([1.0, 0.0, 0.0])  # poles: fall back to x-hat
    circ /= np.where(bad, 1.0, nc)[:, None]
    lon = np.cross(n, circ)
    lon /= np.maximum(np.linalg.norm(lon, axis=1, keepdims=True), 1e-300)
    return n, circ, lon


def helical_fibres(p, centre, inner, outer, alpha_endo_deg=60.0, alpha_epi_deg=-60.0):
    """alpha = alpha_endo*(1-d) + alpha_epi*d with d=0 at the endocardium (labels as in SURVEY 8(d) C3);
    f = cos(alpha) e_circ + sin(alpha) e_long. Returns (fibre [n,3], d [n])."""
    d = shell_depth(p, centre, inner, outer)
    mid_axes = 0.5 * (np.asarray(inner, dtype=np.float64) + np.asarray(outer, dtype=np.float64))
    _, circ, lon = ellipsoid_frame(p, centre, mid_axes)
    alpha = np.deg2rad(alpha_endo_deg * (1.0 - d) + alpha_epi_deg * d)
    f = np.cos(alpha)[:, None] * circ + np.sin(alpha)[:, None] * lon
    f /= np.linalg.norm(f, axis=1, keepdims=True)
    return f, d


def thirds(d: np.ndarray) -> np.ndarray:
    """endo / mid / epi bands by thirds of the transmural coordinate (0 endo, 1 mid, 2 epi)."""
    return np.minimum(2, np.floor(d * 3.0)).astype(np.uint8)


def in_ellipsoid(p, centre, axes) -> np.ndarray:
    q = (p - np.asarray(centre, dtype=np.float64)) / np.asarray(axes, dtype=np.float64)
    return (q * q).sum(axis=1) <= 1.0


def validate(mesh: TetMesh) -> dict:
    """Harness-side sanity checks: positive volumes after orientation is ignored, every face
    shared by at most two cells. Returns counts; raises on failure."""
    x = mesh.xyz[mesh.tets]
    vol = np.abs(np.einsum("ij,ij->i", np.cross(x[:, 1] - x[:, 0], x[:, 2] - x[:, 0]), x[:, 3] - x[:, 0])) / 6.0
    if not (vol > 0).all():
        raise ValueError("degenerate tetrahedron")
    t = mesh.tets.astype(np.int64)
    faces = np.concatenate([np.sort(np.delete(t, j, axis=1), axis=1) for j in range(4)], axis=0)
    nn = np.int64(mesh.n_nodes)
    key = (faces[:, 0] * nn + faces[:, 1]) * nn + faces[:, 2]
    _, cnt = np.unique(key, return_counts=True)
    if cnt.max() > 2:
        raise ValueError("face shared by more than two cells")
    return {"n_faces": int(cnt.size), "n_boundary_faces": int((cnt == 1).sum()), "min_vol": float(vol.min()),
            "mean_vol": float(vol.mean())}


# ---------------------------------------------------------------------------------------------------------------------
# Triangulated surfaces: the two-dimensional media of the paper (Purkinje network).
@dataclass
class TriMesh:
    xyz: np.ndarray            # [n_nodes,3] float64, mm (a flat mesh has z = 0)
    tris: np.ndarray           # [n_tris,3] int32, 0-based
    fibre: np.ndarray | None = None        # [n_tris,3] or None = isotropic (Table 2)
    sigma_scale: np.ndarray | None = None  # [n_tris] or None
    cell_type: np.ndarray | None = None
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def n_tris(self) -> int:
        return int(self.tris.shape[0])

    @property
    def n_tets(self) -> int:       # "number of cells" under the name the 3D code paths use
        return self.n_tris

    def centroids(self) -> np.ndarray:
        return self.xyz[self.tris].mean(axis=1)


def rect_tri(nx: int, ny: int, h: float) -> TriMesh:
    """nx x ny squares of side h in the plane z = 0, each cut along its (0,0)-(1,1) diagonal: 2 nx ny triangles (the
    paper's 2D benchmark domain is such a rectangle, 20 x 7 mm)."""
    i, j = np.meshgrid(np.arange(nx + 1), np.arange(ny + 1), indexing="ij")
    xyz = np.stack([i.ravel() * h, j.ravel() * h, np.zeros(i.size)], axis=1).astype(np.float64)
    nid = lambda a, b: a * (ny + 1) + b
    ci, cj = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")
    ci, cj = ci.ravel(), cj.ravel()
    t1 = np.stack([nid(ci, cj), nid(ci + 1, cj), nid(ci + 1, cj + 1)], axis=1)
    t2 = np.stack([nid(ci, cj), nid(ci + 1, cj + 1), nid(ci, cj + 1)], axis=1)
    tris = np.empty((2 * ci.size, 3), dtype=np.int32)
    tris[0::2] = t1
    tris[1::2] = t2
    return TriMesh(xyz, tris, meta={"kind": "rect", "nx": nx, "ny": ny, "h": h})


def jitter_interior_tri(mesh: TriMesh, amplitude: float, seed: int, out_of_plane: float = 0.0) -> None:
    """Move the interior nodes of a rect_tri mesh by U(-a, a) per in-plane axis (and optionally out of the plane)."""
    nx, ny, h = mesh.meta["nx"], mesh.meta["ny"], mesh.meta["h"]
    x, y = mesh.xyz[:, 0], mesh.xyz[:, 1]
    interior = (x > 0.5 * h) & (x < (nx - 0.5) * h) & (y > 0.5 * h) & (y < (ny - 0.5) * h)
    ids = np.nonzero(interior)[0]
    for d, amp in ((0, amplitude), (1, amplitude), (2, out_of_plane)):
        if amp:
            mesh.xyz[ids, d] += uniform(seed + d, ids, -amp, amp)


def ellipsoid_surface(axes, z_cut: float, h: float, apex_hole: float = 1.0) -> TriMesh:
    """Triangulated open ellipsoidal surface x^2/a^2 + y^2/b^2 + z^2/c^2 = 1 between the plane z = z_cut (base) and a small
    hole around the apex (lowest point), on a structured (ring, azimuth) grid whose rings are about h apart and whose rings
    carry a number of points proportional to their circumference (rounded to a multiple of 8).  Stand-in for the Purkinje
    layer on a ventricular endocardium (a thin layer in the subendocardium)."""
    a, b, c = axes
    t_top = np.arccos(np.clip(z_cut / c, -1.0, 1.0))              # polar angle from +z of the base ring
    t_bot = np.pi - apex_hole / max(a, b)                         # ring of radius ~apex_hole around the apex
    # arc length along a meridian, numerically, to place rings ~h apart
    tt = np.linspace(t_top, t_bot, 4001)
    ds = np.hypot(a * np.cos(tt), c * np.sin(tt))
    s = np.concatenate([[0.0], np.cumsum(0.5 * (ds[1:] + ds[:-1]) * np.diff(tt))])
    n_rings = max(2, int(round(s[-1] / h)) + 1)
    ring_t = np.interp(np.linspace(0.0, s[-1], n_rings), s, tt)
    pts, ring_start, ring_n = [], [], []
    for t in ring_t:
        r = 0.5 * (a + b) * np.sin(t)
        n = max(8, int(round(2.0 * np.pi * r / h / 8.0)) * 8)
        ph = 2.0 * np.pi * np.arange(n) / n
        ring_start.append(sum(ring_n))
        ring_n.append(n)
        pts.append(np.stack([a * np.sin(t) * np.cos(ph), b * np.sin(t) * np.sin(ph), np.full(n, c * np.cos(t))], axis=1))
    xyz = np.concatenate(pts, axis=0)
    tris = []
    for k in range(n_rings - 1):        # stitch ring k (n0 points) to ring k+1 (n1 points) by advancing the lagging side
        n0, n1, s0, s1 = ring_n[k], ring_n[k + 1], ring_start[k], ring_start[k + 1]
        i = j = 0
        while i < n0 or j < n1:
            # next azimuth on each ring (as a fraction of the circle)
            fi, fj = (i + 1) / n0, (j + 1) / n1
            if j >= n1 or (i < n0 and fi <= fj):
                tris.append((s0 + i % n0, s0 + (i + 1) % n0, s1 + j % n1))
                i += 1
            else:
                tris.append((s0 + i % n0, s1 + (j + 1) % n1, s1 + j % n1))
                j += 1
    return TriMesh(xyz.astype(np.float64), np.array(tris, dtype=np.int32),
                   meta={"kind": "ellipsoid_surface", "axes": tuple(axes), "z_cut": z_cut, "h": h})
