"""ctypes wrapper around oracle/ep_oracle_o2.cpp -- CPU ORACLE of the second-order time stepping (Adams-Bashforth
for the non-gating variables + second-order Rush-Larsen), TEST INFRASTRUCTURE ONLY.  The library is ep_oracle.cpp plus the
second-order step; this wrapper talks to its own copy, never to libep_oracle.so, and never imports the CUDA package."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ep_oracle_o2.cpp")
_DEP = os.path.join(_HERE, "ep_oracle.cpp")
_LIB = os.path.join(_HERE, "libep_oracle_o2.so")
_lib = None
_dp = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_DEP))
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < newest:
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.c_int64, _dp, C.c_int64, C.POINTER(C.c_int32), _dp, _dp, C.c_double, C.c_double,
                                 C.c_double, C.c_double]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_state_init.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_uint8), _dp]
        L.orc_stimulus_set.argtypes = [C.c_void_p, C.c_int, C.c_int64, C.POINTER(C.c_int64), C.c_double, C.c_double,
                                       C.c_double]
        L.orc_get_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc_set_state.argtypes = [C.c_void_p, C.c_int, _dp]
        L.orc_activation_times.argtypes = [C.c_void_p, _dp]
        L.orc_mean_vm.restype = C.c_double
        L.orc_mean_vm.argtypes = [C.c_void_p]
        L.orc_o2_attach.restype = C.c_void_p
        L.orc_o2_attach.argtypes = [C.c_void_p]
        L.orc_o2_detach.argtypes = [C.c_void_p]
        L.orc_o2_reset.argtypes = [C.c_void_p]
        L.orc_o2_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.orc_step.argtypes = [C.c_void_p, C.c_int64, C.c_double]
        L.orc_tp06_rest.argtypes = [_dp]
        L.orc_tp06_run.argtypes = [_dp, C.c_int, C.c_double, C.c_int64, C.c_double, C.c_int64, C.c_int64, _dp, C.c_int]
        L.orc_tp06_run_o2.argtypes = [_dp, C.c_int, C.c_double, C.c_int64, C.c_double, C.c_int64, C.c_int64, _dp]
        L.orc_tp06_rhs.argtypes = [_dp, C.c_int, C.c_double, _dp]
        L.orc_tp06_step_o2.argtypes = [_dp, C.c_int, C.c_double, C.c_double, C.c_double, _dp, C.c_int, _dp]
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


class OracleSimO2:
    """Tissue oracle advanced by the second-order scheme (TP06 only)."""

    def __init__(self, xyz, tets, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0, cell_type=None):
        L = lib()
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        tets = np.ascontiguousarray(tets, dtype=np.int32)
        fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
        sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
        self.n_tets = int(tets.shape[0])
        self._h = L.orc_create(int(xyz.shape[0]), _p(xyz), self.n_tets, _p(tets, C.c_int32), _p(fibre), _p(sigma_scale),
                               sigma_l, sigma_t, chi, Cm)
        if not self._h:
            raise ValueError("oracle: invalid mesh")
        ct = None if cell_type is None else np.ascontiguousarray(cell_type, dtype=np.uint8)
        L.orc_state_init(self._h, 0, _p(ct, C.c_uint8), None)
        self._o = L.orc_o2_attach(self._h)

    @classmethod
    def from_problem(cls, prob):
        m = prob.mesh
        s = cls(m.xyz, m.tets, m.fibre, m.sigma_scale, prob.sigma_l, prob.sigma_t, prob.chi, prob.Cm, m.cell_type)
        for k, st in enumerate(prob.stimuli):
            s.stimulus_set(k, st.cell_ids, st.amplitude, st.t_start, st.duration)
        return s

    def stimulus_set(self, slot, cell_ids, amplitude, t_start, duration):
        ids = np.ascontiguousarray(cell_ids, dtype=np.int64)
        lib().orc_stimulus_set(self._h, slot, ids.size, _p(ids, C.c_int64), amplitude, t_start, duration)

    def step(self, n_steps, dt):
        rc = lib().orc_o2_step(self._o, int(n_steps), float(dt))
        if rc:
            raise ValueError(f"oracle o2: step rc={rc}")

    def read_state(self, var):
        out = np.empty(self.n_tets)
        lib().orc_get_state(self._h, var, _p(out))
        return out

    def write_state(self, var, arr):
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        lib().orc_set_state(self._h, var, _p(arr))
        lib().orc_o2_reset(self._o)          # a rewritten state has no history

    def read_vm(self):
        return self.read_state(0)

    def mean_vm(self):
        return float(lib().orc_mean_vm(self._h))

    def activation_times(self):
        out = np.empty(self.n_tets)
        lib().orc_activation_times(self._h, _p(out))
        return out

    def close(self):
        if getattr(self, "_o", None):
            lib().orc_o2_detach(self._o); self._o = None
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h); self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def tp06_rest():
    y = np.empty(19)
    lib().orc_tp06_rest(_p(y))
    return y


def tp06_run(y, cell_type, dt, n_steps, istim=0.0, n_on=0, n_off=0):
    y = np.array(y, dtype=np.float64)
    lib().orc_tp06_run(_p(y), int(cell_type), float(dt), int(n_steps), float(istim), int(n_on), int(n_off), None, 0)
    return y


def tp06_run_o2(y, cell_type, dt, n_steps, istim=0.0, n_on=0, n_off=0, trace=False):
    y = np.array(y, dtype=np.float64)
    tr = np.empty(n_steps + 1) if trace else None
    lib().orc_tp06_run_o2(_p(y), int(cell_type), float(dt), int(n_steps), float(istim), int(n_on), int(n_off), _p(tr))
    return (y, tr) if trace else y


def tp06_rhs(y, cell_type=0, dv_diff=0.0):
    """Right-hand sides of v, Ca_i, Ca_SR, Ca_SS, Na_i, K_i at y, WITHOUT the stimulus."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    f = np.empty(6)
    lib().orc_tp06_rhs(_p(y), int(cell_type), float(dv_diff), _p(f))
    return f


def tp06_step_o2(y, cell_type, dt, istim, dv_diff, hist9, have):
    y = np.ascontiguousarray(y, dtype=np.float64)
    hist9 = np.array(hist9, dtype=np.float64)
    yn = np.empty(19)
    lib().orc_tp06_step_o2(_p(y), int(cell_type), float(dt), float(istim), float(dv_diff), _p(hist9), int(have), _p(yn))
    return yn, hist9
