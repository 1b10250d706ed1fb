"""Bidomain oracle -- CPU, TEST INFRASTRUCTURE ONLY (plain numpy / scipy on top of oracle/ep_oracle.cpp's operator).

Eq. (1) / (6) of the paper with the time stepping of PAPER.md:176-178: v^{n+1} is an explicit
function of v, v_ext, I_ion, I_s at t^n,

    v^{n+1} = v^n + dt [ (A_i v^n + A_i v_ext^n)/(chi C_m) - i_ion - I_s/C_m ],          s^{n+1} from s^n (Rush-Larsen / FE),

and "once v(t^{n+1}) is solved, the external potential v_ext(t^{n+1}) is obtained by solving the linear system given by the
second equation of the system (6)":   A_ie v_ext^{n+1} = -A_i v^{n+1},   A_i = div(M_int grad .), A_ie = div((M_int+M_ext) grad .),
both discretised by the finite-volume chain of PAPER.md:164-168 (the C++ oracle's apply_diffusion, with the respective tensor).

The paper solves that system "through an iterative GMRES method with restart"; its solution has a plain definition, so this
oracle IS that definition: A_ie is assembled column by column (operator applied to unit vectors) and the system is solved
DIRECTLY (sparse LU).  Readings: E1 the system is singular under no-flux boundaries (constants are
in the null space, the cell volumes span the left null space): v_ext is the solution with zero volume-weighted mean,
imposed through a bordered system; E2 v_ext^0 solves the same equation for v^0 (zero for a uniform initial potential).
Only tests/ may import this module.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from . import ep_oracle as O


class BidomainOracle:
    def __init__(self, mesh, sig_int, sig_ext, chi=1400.0, Cm=1.0, model=0):
        """sig_int = (l, t), sig_ext = (l, t) in mS/cm along / across the fibres (Table 2)."""
        self.mesh, self.chi, self.Cm = mesh, chi, Cm
        self.oi = O.OracleSim(mesh.xyz, mesh.tets, mesh.fibre, mesh.sigma_scale, sig_int[0], sig_int[1], chi, Cm)
        self.oie = O.OracleSim(mesh.xyz, mesh.tets, mesh.fibre, mesh.sigma_scale, sig_int[0] + sig_ext[0],
                               sig_int[1] + sig_ext[1], chi, Cm)
        self.oi.state_init(model, mesh.cell_type)
        self.n = mesh.n_tets
        self.vol, _ = self.oi.geometry()
        self._lu = None
        self.vext = np.zeros(self.n)
        self._valid = False

    def stimulus_set(self, *a):
        self.oi.stimulus_set(*a)

    def _factor(self):
        if self._lu is None:
            n = self.n
            cols = []
            e = np.zeros(n)
            for k in range(n):                       # A_ie column by column: the operator applied to unit vectors
                e[k] = 1.0
                c = self.oie.apply_diffusion(e)
                e[k] = 0.0
                nz = np.nonzero(c)[0]
                cols.append((nz, c[nz]))
            rows = np.concatenate([nz for nz, _ in cols])
            colid = np.concatenate([np.full(nz.size, k) for k, (nz, _) in enumerate(cols)])
            vals = np.concatenate([v for _, v in cols])
            A = sp.csc_matrix((vals, (rows, colid)), shape=(n, n))
            self.A_ie = A
            # bordered system (reading E1): [A 1; V^T 0] [x; mu] = [b; 0]
            K = sp.bmat([[A, sp.csc_matrix(np.ones((n, 1)))], [sp.csc_matrix(self.vol[None, :]), None]], format="csc")
            self._lu = spla.splu(K)
        return self._lu

    def solve_vext(self, v):
        """v_ext with A_ie v_ext = -A_i v and sum_c V_c v_ext,c = 0 (direct solve)."""
        b = -self.oi.apply_diffusion(v)
        x = self._factor().solve(np.concatenate([b, [0.0]]))
        return x[:-1]

    def step(self, n_steps, dt):
        for _ in range(n_steps):
            if not self._valid:                       # reading E2
                self.vext = self.solve_vext(self.oi.read_vm())
                self._valid = True
            self.oi.set_source(self.oi.apply_diffusion(self.vext) / (self.chi * self.Cm))
            self.oi.step(1, dt)
            self.vext = self.solve_vext(self.oi.read_vm())

    def read_vm(self):
        return self.oi.read_vm()

    def read_state(self, k):
        return self.oi.read_state(k)

    def write_state(self, k, arr):
        self.oi.write_state(k, arr)
        if k == 0:
            self._valid = False

    def read_vext(self):
        if not self._valid:
            self.vext = self.solve_vext(self.oi.read_vm())
            self._valid = True
        return self.vext.copy()

    def activation_times(self):
        return self.oi.activation_times()

    def close(self):
        self.oi.close(); self.oie.close()
