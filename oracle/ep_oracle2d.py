"""ctypes wrapper around oracle/ep_oracle2d.cpp -- CPU ORACLE of the 2D (Purkinje) medium, TEST INFRASTRUCTURE ONLY.

Triangulated-surface finite volumes + Stewart 2009 Purkinje cell model.  Only tests/
may import this module; it never imports the CUDA package.  The shared object is built on demand with g++.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ep_oracle2d.cpp")
_LIB = os.path.join(_HERE, "libep_oracle2d.so")
_LIB_OVERRIDE = os.environ.get("EP_ORACLE2D_LIB")      # mutation test: a deliberately broken build
_lib = None
_dp = C.POINTER(C.c_double)

STW_STATES = ["V", "y", "xr1", "xr2", "xs", "m", "h", "j", "d", "f", "f2", "fCass", "s", "r", "Rprime", "Ca_i", "Ca_SR",
              "Ca_SS", "Na_i", "K_i"]
STW_GATES = STW_STATES[1:14]
STW_CURRENTS = ["IfNa", "IfK", "IK1", "Ito", "Isus", "IKr", "IKs", "ICaL", "INaK", "INa", "IbNa", "INaCa", "IbCa", "IpK",
                "IpCa", "iion", "Irel", "Ileak", "Iup", "Ixfer", "dR"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_LIB_OVERRIDE if _LIB_OVERRIDE else build())
        L.orc2_create.restype = C.c_void_p
        L.orc2_create.argtypes = [C.c_int64, _dp, C.c_int64, C.POINTER(C.c_int32), _dp, _dp, C.c_double, C.c_double,
                                  C.c_double, C.c_double]
        L.orc2_destroy.argtypes = [C.c_void_p]
        L.orc2_n_edges.restype = C.c_int64
        L.orc2_n_edges.argtypes = [C.c_void_p]
        L.orc2_geometry.argtypes = [C.c_void_p, _dp, _dp]
        L.orc2_node_values.argtypes = [C.c_void_p, _dp, _dp]
        L.orc2_cell_gradients.argtypes = [C.c_void_p, _dp, _dp]
        L.orc2_apply_diffusion.argtypes = [C.c_void_p, _dp, _dp, C.c_int]
        L.orc2_state_init.argtypes = [C.c_void_p, _dp]
        L.orc2_stimulus_set.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_int64), C.c_double, C.c_double,
                                        C.c_double]
        L.orc2_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.orc2_get_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc2_set_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc2_activation_times.argtypes = [C.c_void_p, _dp]
        L.orc2_mean_vm.restype = C.c_double
        L.orc2_mean_vm.argtypes = [C.c_void_p]
        L.orc2_stw_init.argtypes = [_dp]
        L.orc2_stw_gates.argtypes = [C.c_double, C.c_double, _dp, _dp]
        L.orc2_stw_currents.argtypes = [_dp, _dp]
        L.orc2_stw_step.argtypes = [_dp, C.c_double, C.c_double, C.c_double, _dp]
        L.orc2_stw_run.argtypes = [_dp, C.c_double, C.c_int64, C.c_double, C.c_int64, C.c_int64, _dp, C.c_int]
        _lib = L
    return _lib


class OracleSim2D:
    """Oracle handle for a triangulated surface with the Stewart model; mirrors the ep_* call list."""

    def __init__(self, xyz, tris, fibre=None, sigma_scale=None, sigma_l=39.5, sigma_t=39.5, chi=1400.0, Cm=1.0):
        L = lib()
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        tris = np.ascontiguousarray(tris, dtype=np.int32)
        fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
        sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
        self.n_nodes, self.n_tris = int(xyz.shape[0]), int(tris.shape[0])
        self._h = L.orc2_create(self.n_nodes, _p(xyz), self.n_tris, _p(tris, C.c_int32), _p(fibre), _p(sigma_scale),
                                sigma_l, sigma_t, chi, Cm)
        if not self._h:
            raise ValueError("oracle2d: invalid mesh")
        self.n_states = 20

    @classmethod
    def from_problem(cls, prob):
        m = prob.mesh
        s = cls(m.xyz, m.tris, m.fibre, m.sigma_scale, prob.sigma_l, prob.sigma_t, prob.chi, prob.Cm)
        s.state_init()
        for k, st in enumerate(prob.stimuli):
            s.stimulus_set(k, st.cell_ids, st.amplitude, st.t_start, st.duration)
        return s

    def close(self):
        if self._h:
            lib().orc2_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def n_edges(self):
        return int(lib().orc2_n_edges(self._h))

    def geometry(self):
        area = np.empty(self.n_tris)
        cen = np.empty((self.n_tris, 3))
        lib().orc2_geometry(self._h, _p(area), _p(cen))
        return area, cen

    def node_values(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n_nodes)
        lib().orc2_node_values(self._h, _p(v), _p(out))
        return out

    def cell_gradients(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty((self.n_tris, 3))
        lib().orc2_cell_gradients(self._h, _p(v), _p(out))
        return out

    def apply_diffusion(self, v, use_corr=True):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n_tris)
        lib().orc2_apply_diffusion(self._h, _p(v), _p(out), 1 if use_corr else 0)
        return out

    def state_init(self, y0=None):
        y0 = None if y0 is None else np.ascontiguousarray(y0, dtype=np.float64)
        lib().orc2_state_init(self._h, _p(y0))

    def stimulus_set(self, slot, cell_ids, amplitude, t_start, duration):
        ids = np.ascontiguousarray(cell_ids, dtype=np.int64)
        rc = lib().orc2_stimulus_set(self._h, slot, ids.size, _p(ids, C.c_int64), amplitude, t_start, duration)
        if rc:
            raise ValueError(f"oracle2d: stimulus_set rc={rc}")

    def step(self, n_steps, dt):
        rc = lib().orc2_step(self._h, int(n_steps), float(dt))
        if rc:
            raise ValueError(f"oracle2d: step rc={rc}")

    def read_state(self, var):
        out = np.empty(self.n_tris)
        lib().orc2_get_state(self._h, var, _p(out))
        return out

    def write_state(self, var, arr):
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        assert arr.size == self.n_tris
        lib().orc2_set_state(self._h, var, _p(arr))

    def read_vm(self):
        return self.read_state(0)

    def mean_vm(self):
        return float(lib().orc2_mean_vm(self._h))

    def activation_times(self):
        out = np.empty(self.n_tris)
        lib().orc2_activation_times(self._h, _p(out))
        return out


def stw_init():
    y = np.empty(20)
    lib().orc2_stw_init(_p(y))
    return y


def stw_gates(v, Ca_SS=4.46818714055411e-4):
    inf, tau = np.empty(13), np.empty(13)
    lib().orc2_stw_gates(float(v), float(Ca_SS), _p(inf), _p(tau))
    return inf, tau


def stw_currents(y):
    y = np.ascontiguousarray(y, dtype=np.float64)
    out = np.empty(21)
    lib().orc2_stw_currents(_p(y), _p(out))
    return dict(zip(STW_CURRENTS, out))


def stw_step(y, dt, istim=0.0, dv_diff=0.0):
    y = np.ascontiguousarray(y, dtype=np.float64)
    yn = np.empty(20)
    lib().orc2_stw_step(_p(y), float(dt), float(istim), float(dv_diff), _p(yn))
    return yn


def stw_run(y, dt, n_steps, istim=0.0, n_on=0, n_off=0, trace=False, freeze_v=False):
    y = np.array(y, dtype=np.float64)
    tr = np.empty(n_steps + 1) if trace else None
    lib().orc2_stw_run(_p(y), float(dt), int(n_steps), float(istim), int(n_on), int(n_off), _p(tr), 1 if freeze_v else 0)
    return y, tr
