"""ctypes wrapper around oracle/ep_oracle.cpp -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It never imports the CUDA package. The shared object is built on demand with g++ (see build()).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ep_oracle.cpp")
_LIB = os.path.join(_HERE, "libep_oracle.so")
# tests/test_oracle_mutations.py points this at a deliberately broken build to prove that the pins notice it
_LIB_OVERRIDE = os.environ.get("EP_ORACLE_LIB")
_lib = None

_dp = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    """g++ -O2 -ffp-contract=off (no FMA contraction, so the arithmetic is what the source says)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.check_call(cmd)
    return _LIB


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        if _LIB_OVERRIDE:
            L = C.CDLL(_LIB_OVERRIDE)
        else:
            build()
            L = C.CDLL(_LIB)
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int64, _dp, C.c_int64, C.POINTER(C.c_int32), _dp, _dp, C.c_double, C.c_double,
                                 C.c_double, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        L.orc_n_faces.restype = C.c_int64
        L.orc_n_faces.argtypes = [C.c_void_p]
        L.orc_geometry.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_node_values.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_cell_gradients.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_apply_diffusion.argtypes = [C.c_void_p, _dp, _dp, C.c_int]
        L.orc_state_init.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_uint8), _dp]
        L.orc_stimulus_set.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_int64), C.c_double, C.c_double,
                                       C.c_double]
        L.orc_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.orc_set_source.argtypes = [C.c_void_p, _dp]
        L.orc_trigger_set.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_int64), C.c_int, C.c_double]
        L.orc_trigger_time.argtypes = [C.c_void_p, C.c_int]
        L.orc_trigger_time.restype = C.c_double
        L.orc_n_states.argtypes = [C.c_void_p]
        L.orc_step_count.argtypes = [C.c_void_p]
        L.orc_step_count.restype = C.c_int64
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc_set_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc_activation_times.argtypes = [C.c_void_p, _dp]
        L.orc_mean_vm.restype = C.c_double
        L.orc_mean_vm.argtypes = [C.c_void_p]
        L.orc_tp06_rest.argtypes = [_dp]
        L.orc_tp06_gates.argtypes = [C.c_double, C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.orc_tp06_currents.argtypes = [_dp, C.c_int, _dp]
        L.orc_tp06_run.argtypes = [_dp, C.c_int, C.c_double, C.c_int64, C.c_double, C.c_int64, C.c_int64, _dp, C.c_int]
        L.orc_crn_rest.argtypes = [_dp]
        L.orc_crn_gates.argtypes = [C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_crn_currents.argtypes = [_dp, _dp]
        L.orc_crn_run.argtypes = [_dp, C.c_double, C.c_int64, C.c_double, C.c_int64, C.c_int64, _dp, C.c_int]
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def get_threads() -> int:
    return int(lib().orc_get_threads())


class OracleSim:
    """Oracle simulation handle; mirrors the ep_* C-ABI call list (ep_mesh_create ... ep_activation_times)."""

    def __init__(self, xyz, tets, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0):
        L = lib()
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        tets = np.ascontiguousarray(tets, dtype=np.int32)
        fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
        sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
        self.n_nodes, self.n_tets = int(xyz.shape[0]), int(tets.shape[0])
        self._h = L.orc_create(self.n_nodes, _p(xyz), self.n_tets, _p(tets, C.c_int32), _p(fibre), _p(sigma_scale),
                               sigma_l, sigma_t, chi, Cm)
        if not self._h:
            raise ValueError("oracle: invalid mesh")
        self.chi, self.Cm = chi, Cm

    @classmethod
    def from_problem(cls, prob):
        m = prob.mesh
        s = cls(m.xyz, m.tets, m.fibre, m.sigma_scale, prob.sigma_l, prob.sigma_t, prob.chi, prob.Cm)
        s.state_init(prob.model, m.cell_type)
        for k, st in enumerate(prob.stimuli):
            s.stimulus_set(k, st.cell_ids, st.amplitude, st.t_start, st.duration)
        for k, tr in enumerate(getattr(prob, "triggers", [])):
            s.trigger_set(k, tr.monitor_ids, tr.slot, tr.delay)
        return s

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # geometry / operator pieces
    def n_faces(self):
        return int(lib().orc_n_faces(self._h))

    def geometry(self):
        vol = np.empty(self.n_tets)
        cen = np.empty((self.n_tets, 3))
        lib().orc_geometry(self._h, _p(vol), _p(cen))
        return vol, cen

    def node_values(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n_nodes)
        lib().orc_node_values(self._h, _p(v), _p(out))
        return out

    def cell_gradients(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty((self.n_tets, 3))
        lib().orc_cell_gradients(self._h, _p(v), _p(out))
        return out

    def apply_diffusion(self, v, use_corr=True):
        """div(M grad v) in uA/cm^3."""
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n_tets)
        lib().orc_apply_diffusion(self._h, _p(v), _p(out), 1 if use_corr else 0)
        return out

    # time stepping
    def state_init(self, model=0, cell_type=None, y0=None):
        ct = None if cell_type is None else np.ascontiguousarray(cell_type, dtype=np.uint8)
        y0 = None if y0 is None else np.ascontiguousarray(y0, dtype=np.float64)
        rc = lib().orc_state_init(self._h, model, _p(ct, C.c_uint8), _p(y0))
        if rc:
            raise ValueError(f"oracle: state_init rc={rc}")
        self.n_states = int(lib().orc_n_states(self._h))

    def stimulus_set(self, slot, cell_ids, amplitude, t_start, duration):
        ids = np.ascontiguousarray(cell_ids, dtype=np.int64)
        rc = lib().orc_stimulus_set(self._h, slot, ids.size, _p(ids, C.c_int64), amplitude, t_start, duration)
        if rc:
            raise ValueError(f"oracle: stimulus_set rc={rc}")

    def trigger_set(self, trigger, monitor_ids, slot, delay):
        ids = np.ascontiguousarray(monitor_ids, dtype=np.int64)
        rc = lib().orc_trigger_set(self._h, int(trigger), ids.size, _p(ids, C.c_int64), int(slot), float(delay))
        if rc:
            raise ValueError(f"oracle: trigger_set rc={rc}")

    def trigger_time(self, trigger):
        return float(lib().orc_trigger_time(self._h, int(trigger)))

    def set_source(self, src):
        """Extra right-hand side per cell in mV/ms (bidomain: div(M_int grad v_ext)/(chi C_m)); None removes it."""
        src = None if src is None else np.ascontiguousarray(src, dtype=np.float64)
        assert src is None or src.size == self.n_tets
        lib().orc_set_source(self._h, _p(src))

    def step(self, n_steps, dt):
        rc = lib().orc_step(self._h, int(n_steps), float(dt))
        if rc:
            raise ValueError(f"oracle: step rc={rc}")

    def read_state(self, var):
        out = np.empty(self.n_tets)
        lib().orc_get_state(self._h, var, _p(out))
        return out

    def write_state(self, var, arr):
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        assert arr.size == self.n_tets
        lib().orc_set_state(self._h, var, _p(arr))

    def read_vm(self):
        return self.read_state(0)

    def mean_vm(self):
        return float(lib().orc_mean_vm(self._h))

    def activation_times(self):
        out = np.empty(self.n_tets)
        lib().orc_activation_times(self._h, _p(out))
        return out


# ---- single-cell helpers
def tp06_rest():
    y = np.empty(19)
    lib().orc_tp06_rest(_p(y))
    return y


def tp06_gates(v, cell_type=0, Ca_SS=7e-5, Ca_SR=1.3):
    inf, tau = np.empty(13), np.empty(13)
    lib().orc_tp06_gates(float(v), int(cell_type), float(Ca_SS), float(Ca_SR), _p(inf), _p(tau))
    return inf, tau


def tp06_currents(y, cell_type=0):
    y = np.ascontiguousarray(y, dtype=np.float64)
    out = np.empty(17)
    lib().orc_tp06_currents(_p(y), int(cell_type), _p(out))
    names = ["INa", "ICaL", "Ito", "IKr", "IKs", "IK1", "INaCa", "INaK", "IpCa", "IpK", "IbNa", "IbCa", "iion",
             "Irel", "Ileak", "Iup", "Ixfer"]
    return dict(zip(names, out))


def tp06_run(y, cell_type, dt, n_steps, istim=0.0, n_on=0, n_off=0, trace=False, freeze_v=False):
    """Advance one cell n_steps; returns (y_final, v_trace or None)."""
    y = np.array(y, dtype=np.float64)
    tr = np.empty(n_steps + 1) if trace else None
    lib().orc_tp06_run(_p(y), int(cell_type), float(dt), int(n_steps), float(istim), int(n_on), int(n_off), _p(tr),
                       1 if freeze_v else 0)
    return y, tr


# ---- Courtemanche single-cell helpers
CRN_CURRENTS = ["INa", "IK1", "Ito", "IKur", "IKr", "IKs", "ICaL", "IpCa", "INaK", "INaCa", "IbNa", "IbCa", "iion", "Irel",
                "Itr", "Iup", "Iupleak", "Fn"]


def crn_rest():
    y = np.empty(21)
    lib().orc_crn_rest(_p(y))
    return y


def crn_gates(V, Cai=1.013e-4, Fn=0.0):
    inf, tau = np.empty(15), np.empty(15)
    lib().orc_crn_gates(float(V), float(Cai), float(Fn), _p(inf), _p(tau))
    return inf, tau


def crn_currents(y):
    y = np.ascontiguousarray(y, dtype=np.float64)
    out = np.empty(18)
    lib().orc_crn_currents(_p(y), _p(out))
    return dict(zip(CRN_CURRENTS, out))


def crn_run(y, dt, n_steps, istim=0.0, n_on=0, n_off=0, trace=False, freeze_v=False):
    y = np.array(y, dtype=np.float64)
    tr = np.empty(n_steps + 1) if trace else None
    lib().orc_crn_run(_p(y), float(dt), int(n_steps), float(istim), int(n_on), int(n_off), _p(tr), 1 if freeze_v else 0)
    return y, tr
