"""ctypes binding of libep.so: same names as include/ep.h, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

EP_MODEL_TP06, EP_MODEL_CRN98, EP_MODEL_STEWART = 0, 1, 2
_dp = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_i64p = C.POINTER(C.c_int64)
_u8p = C.POINTER(C.c_uint8)
_vp = C.c_void_p

# name -> (restype, argtypes); tests/test_abi.py checks this table against include/ep.h
SIGNATURES = {
    "ep_model_n_states": (C.c_int, [C.c_int]),
    "ep_mesh_create": (C.c_int, [C.POINTER(_vp), C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double,
                                 C.c_double, C.c_double]),
    "ep_mesh_create_tri": (C.c_int, [C.POINTER(_vp), C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double,
                                     C.c_double, C.c_double]),
    "ep_mesh_create_bidomain": (C.c_int, [C.POINTER(_vp), C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double,
                                          C.c_double, C.c_double, C.c_double, C.c_double]),
    "ep_bidomain_solver": (C.c_int, [_vp, C.c_int, C.c_int, C.c_double]),
    "ep_read_vext": (C.c_int, [_vp, _dp]),
    "ep_bidomain_stats": (C.c_int, [_vp, _i64p, _i64p, _i64p, _dp]),
    "ep_shard_plan": (C.c_int, [C.c_int64, _dp, C.c_int64, _i32p, C.c_int, C.c_int, _i64p, _i64p, _i64p, _i64p, _i64p, _i64p]),
    "ep_shard_create": (C.c_int, [C.POINTER(_vp), C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double,
                                  C.c_double, C.c_double, C.c_int, C.c_int]),
    "ep_shard_info": (C.c_int, [_vp, _i64p, _i64p, _i64p, _i64p, _i64p]),
    "ep_shard_buffers": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "ep_halo_pack": (C.c_int, [_vp]),
    "ep_halo_unpack": (C.c_int, [_vp]),
    "ep_halo_exchange_local": (C.c_int, [C.POINTER(_vp), C.c_int]),
    "ep_state_init": (C.c_int, [_vp, C.c_int, _u8p, _dp]),
    "ep_stimulus_set": (C.c_int, [_vp, C.c_int, C.c_int64, _i64p, C.c_double, C.c_double, C.c_double]),
    "ep_trigger_set": (C.c_int, [_vp, C.c_int, C.c_int64, _i64p, C.c_int, C.c_double]),
    "ep_trigger_time": (C.c_int, [_vp, C.c_int, _dp]),
    "ep_couple": (C.c_int, [_vp, C.c_int, _vp, C.c_int, C.c_double, C.POINTER(C.c_int)]),
    "ep_set_time_order": (C.c_int, [_vp, C.c_int]),
    "ep_step": (C.c_int, [_vp, C.c_int64, C.c_double]),
    "ep_synchronize": (C.c_int, [_vp]),
    "ep_read_vm": (C.c_int, [_vp, _dp]),
    "ep_read_state": (C.c_int, [_vp, C.c_int, _dp]),
    "ep_write_state": (C.c_int, [_vp, C.c_int, _dp]),
    "ep_write_states": (C.c_int, [_vp, _dp]),
    "ep_read_states": (C.c_int, [_vp, _dp]),
    "ep_activation_times": (C.c_int, [_vp, _dp]),
    "ep_set_step_count": (C.c_int, [_vp, C.c_int64, C.c_double]),
    "ep_write_activation_times": (C.c_int, [_vp, _dp]),
    "ep_trigger_restore": (C.c_int, [_vp, C.c_int, C.c_double]),
    "ep_mean_vm": (C.c_int, [_vp, _dp]),
    "ep_apply_diffusion": (C.c_int, [_vp, _dp, _dp]),
    "ep_stable_dt": (C.c_int, [_vp, _dp]),
    "ep_check_finite": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "ep_set_stream": (C.c_int, [_vp, _vp]),
    "ep_device_vm": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "ep_n_cells": (C.c_int64, [_vp]),
    "ep_n_nodes": (C.c_int64, [_vp]),
    "ep_step_count": (C.c_int64, [_vp]),
    "ep_time": (C.c_double, [_vp]),
    "ep_device_bytes": (C.c_int64, [_vp]),
    "ep_step_bytes": (C.c_int64, [_vp]),
    "ep_launch_count": (C.c_int64, [_vp]),
    "ep_kernel_bytes": (C.c_int64, [_vp, C.c_int]),
    "ep_profile": (C.c_int, [_vp, C.c_int]),
    "ep_profile_read": (C.c_int, [_vp, _dp]),
    "ep_math_eval": (C.c_int, [C.c_int, C.c_int64, _dp, _dp]),
    "ep_fp64_rate": (C.c_int, [_dp]),
    "ep_weighted_mean_noalloc": (C.c_int, [_vp, _vp, C.c_int64, _vp, _vp]),
    "ep_destroy": (None, [_vp]),
    "ep_last_error": (C.c_char_p, []),
    "ep_host_stencil": (C.c_int, [C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                  C.c_double, _i32p, _dp, _i32p, _dp, _i64p, _i32p, _dp, _i32p]),
    "ep_host_stencil_tri": (C.c_int, [C.c_int64, _dp, C.c_int64, _i32p, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                      C.c_double, _i32p, _dp, _i32p, _dp, _i64p, _i32p, _dp, _i32p]),
}

_lib = None


class EpError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libep error {code}: {msg}")
        self.code = code


def lib():
    """Load (building if stale) libep.so.  Raises if it cannot be built or loaded: there is no fallback."""
    global _lib
    if _lib is None:
        path = os.environ.get("EP_LIB_OVERRIDE") or _build.build()   # override: A/B builds of the same ABI
        L = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        L._path = path
        _lib = L
    return _lib


def _chk(rc: int) -> None:
    if rc != 0:
        raise EpError(rc, lib().ep_last_error().decode())


def _p(a, ct=C.c_double):
    return a.ctypes.data_as(C.POINTER(ct)) if a is not None else None


def math_eval(fn: int, x):
    """ep_math_eval: the kernels' own exp (0), log (1), rcp (2), rsqrt (3) on the device."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    _chk(lib().ep_math_eval(int(fn), x.size, _p(x), _p(y)))
    return y


def fp64_rate() -> float:
    """ep_fp64_rate: measured warp-wide DFMA instructions per second of the current device's fp64 pipe."""
    r = C.c_double(0.0)
    _chk(lib().ep_fp64_rate(C.byref(r)))
    return float(r.value)


NOALLOC_MAX_N = 33554432   # EP_NOALLOC_MAX_N of include/ep.h


def weighted_mean_noalloc(v_dptr: int, w_dptr: int, n: int, out_dptr: int, stream=None) -> None:
    """ep_weighted_mean_noalloc: out[0] = sum(w v) / sum(w), out[1] = sum(w) of DEVICE arrays (raw pointers, double[n] /
    double[2]); allocates nothing, asynchronous on `stream` (a cudaStream_t as int, None: the default stream)."""
    _chk(lib().ep_weighted_mean_noalloc(_vp(v_dptr), _vp(w_dptr), int(n), _vp(out_dptr), _vp(stream) if stream else None))


def model_n_states(model: int) -> int:
    return int(lib().ep_model_n_states(model))


def host_stencil(xyz, tets, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0):
    """ep_host_stencil: the preprocessor's factored stencil in the caller's numbering (no GPU needed)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    tets = np.ascontiguousarray(tets, dtype=np.int32)
    fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
    sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
    nn, nc = xyz.shape[0], tets.shape[0]
    out = dict(node=np.empty((nc, 8), np.int32), a=np.empty((nc, 8)), nbr=np.empty((nc, 4), np.int32),
               b=np.empty((nc, 4)), node_ptr=np.empty(nn + 1, np.int64), node_cell=np.empty(4 * nc, np.int32),
               w=np.empty(4 * nc), perm=np.empty(nc, np.int32))
    _chk(lib().ep_host_stencil(nn, _p(xyz), nc, _p(tets, C.c_int32), _p(fibre), _p(sigma_scale), sigma_l, sigma_t,
                               chi, Cm, _p(out["node"], C.c_int32), _p(out["a"]), _p(out["nbr"], C.c_int32),
                               _p(out["b"]), _p(out["node_ptr"], C.c_int64), _p(out["node_cell"], C.c_int32),
                               _p(out["w"]), _p(out["perm"], C.c_int32)))
    return out


def host_stencil_tri(xyz, tris, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0):
    """ep_host_stencil_tri: the factored stencil of a triangulated surface in the caller's numbering (no GPU needed)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    tris = np.ascontiguousarray(tris, dtype=np.int32)
    fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
    sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
    nn, nc = xyz.shape[0], tris.shape[0]
    out = dict(node=np.empty((nc, 8), np.int32), a=np.empty((nc, 8)), nbr=np.empty((nc, 4), np.int32),
               b=np.empty((nc, 4)), node_ptr=np.empty(nn + 1, np.int64), node_cell=np.empty(3 * nc, np.int32),
               w=np.empty(3 * nc), perm=np.empty(nc, np.int32))
    _chk(lib().ep_host_stencil_tri(nn, _p(xyz), nc, _p(tris, C.c_int32), _p(fibre), _p(sigma_scale), sigma_l, sigma_t,
                                   chi, Cm, _p(out["node"], C.c_int32), _p(out["a"]), _p(out["nbr"], C.c_int32),
                                   _p(out["b"]), _p(out["node_ptr"], C.c_int64), _p(out["node_cell"], C.c_int32),
                                   _p(out["w"]), _p(out["perm"], C.c_int32)))
    return out


def shard_plan(xyz, tets, part, n_parts):
    """ep_shard_plan: the host-only partitioner (no GPU needed).  Returns n_owned, the global ids of the local cells (owned
    first), and the per-peer segments + global cell ids of the send and receive buffers."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    tets = np.ascontiguousarray(tets, dtype=np.int32)
    nc = tets.shape[0]
    counts = np.zeros(4, np.int64)
    local = np.empty(nc, np.int64); sg = np.empty(nc, np.int64); rg = np.empty(nc, np.int64)
    sp = np.empty(n_parts + 1, np.int64); rp = np.empty(n_parts + 1, np.int64)
    _chk(lib().ep_shard_plan(xyz.shape[0], _p(xyz), nc, _p(tets, C.c_int32), int(part), int(n_parts), _p(counts, C.c_int64),
                             _p(local, C.c_int64), _p(sp, C.c_int64), _p(sg, C.c_int64), _p(rp, C.c_int64), _p(rg, C.c_int64)))
    return dict(n_owned=int(counts[0]), local_cells=local[:counts[1]].copy(), send_ptr=sp, send_global=sg[:counts[2]].copy(),
                recv_ptr=rp, recv_global=rg[:counts[3]].copy())


def halo_exchange_local(sims):
    """ep_halo_exchange_local: pack, exchange and unpack the halos of all parts of one sharding living in this process."""
    arr = (_vp * len(sims))(*[s._h for s in sims])
    _chk(lib().ep_halo_exchange_local(arr, len(sims)))


class Sim:
    """One simulation handle (ep_sim*).  Method names follow the C-ABI calls.  cells [n,4]: tetrahedra (ep_mesh_create);
    cells [n,3]: a triangulated surface (ep_mesh_create_tri)."""

    def __init__(self, xyz, tets, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0,
                 sigma_ext=None):
        """sigma_ext = (l, t): bidomain (ep_mesh_create_bidomain); sigma_l / sigma_t are then the intracellular values."""
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        tets = np.ascontiguousarray(tets, dtype=np.int32)
        fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
        sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
        self._h = _vp()
        if sigma_ext is not None:
            _chk(lib().ep_mesh_create_bidomain(C.byref(self._h), xyz.shape[0], _p(xyz), tets.shape[0], _p(tets, C.c_int32),
                                               _p(fibre), _p(sigma_scale), sigma_l, sigma_t, float(sigma_ext[0]),
                                               float(sigma_ext[1]), chi, Cm))
        else:
            create = lib().ep_mesh_create if tets.shape[1] == 4 else lib().ep_mesh_create_tri
            _chk(create(C.byref(self._h), xyz.shape[0], _p(xyz), tets.shape[0], _p(tets, C.c_int32),
                        _p(fibre), _p(sigma_scale), sigma_l, sigma_t, chi, Cm))
        self.n_tets = int(lib().ep_n_cells(self._h))
        self.n_nodes = int(lib().ep_n_nodes(self._h))
        self.n_states = 0

    @classmethod
    def shard(cls, xyz, tets, part, n_parts, fibre=None, sigma_scale=None, sigma_l=1.3, sigma_t=0.18, chi=1400.0, Cm=1.0):
        """ep_shard_create: part `part` of an n_parts-way sharding of the GLOBAL mesh.  The handle is numbered locally;
        self.global_ids[k] is the global id of local cell k, the first self.n_owned are the owned ones."""
        xyz = np.ascontiguousarray(xyz, dtype=np.float64)
        tets = np.ascontiguousarray(tets, dtype=np.int32)
        fibre = None if fibre is None else np.ascontiguousarray(fibre, dtype=np.float64)
        sigma_scale = None if sigma_scale is None else np.ascontiguousarray(sigma_scale, dtype=np.float64)
        s = cls.__new__(cls)
        s._h = _vp()
        _chk(lib().ep_shard_create(C.byref(s._h), xyz.shape[0], _p(xyz), tets.shape[0], _p(tets, C.c_int32), _p(fibre),
                                   _p(sigma_scale), sigma_l, sigma_t, chi, Cm, int(part), int(n_parts)))
        s.n_tets = int(lib().ep_n_cells(s._h))
        s.n_nodes = int(lib().ep_n_nodes(s._h))
        s.n_states = 0
        no, nl = C.c_int64(), C.c_int64()
        s.global_ids = np.empty(s.n_tets, np.int64)
        s.send_ptr = np.empty(n_parts + 1, np.int64); s.recv_ptr = np.empty(n_parts + 1, np.int64)
        _chk(lib().ep_shard_info(s._h, C.byref(no), C.byref(nl), _p(s.global_ids, C.c_int64), _p(s.send_ptr, C.c_int64),
                                 _p(s.recv_ptr, C.c_int64)))
        s.n_owned = int(no.value)
        return s

    def shard_buffers(self):
        """Device pointers (ints) of the send and receive buffers."""
        a, b = _vp(), _vp()
        _chk(lib().ep_shard_buffers(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def halo_pack(self):
        _chk(lib().ep_halo_pack(self._h))

    def halo_unpack(self):
        _chk(lib().ep_halo_unpack(self._h))

    @classmethod
    def from_problem(cls, prob):
        m = prob.mesh
        cells = m.tets if hasattr(m, "tets") else m.tris          # TetMesh or TriMesh (ep_inputs.meshes)
        s = cls(m.xyz, cells, m.fibre, m.sigma_scale, prob.sigma_l, prob.sigma_t, prob.chi, prob.Cm)
        s.state_init(prob.model, m.cell_type)
        for k, st in enumerate(prob.stimuli):
            s.stimulus_set(k, st.cell_ids, st.amplitude, st.t_start, st.duration)
        for k, tr in enumerate(getattr(prob, "triggers", [])):
            s.trigger_set(k, tr.monitor_ids, tr.slot, tr.delay)
        return s

    def close(self):
        if getattr(self, "_h", None):
            lib().ep_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def state_init(self, model=EP_MODEL_TP06, cell_type=None, y0=None):
        ct = None if cell_type is None else np.ascontiguousarray(cell_type, dtype=np.uint8)
        y0 = None if y0 is None else np.ascontiguousarray(y0, dtype=np.float64)
        _chk(lib().ep_state_init(self._h, model, _p(ct, C.c_uint8), _p(y0)))
        self.n_states = model_n_states(model)

    def stimulus_set(self, slot, cell_ids, amplitude, t_start, duration):
        ids = np.ascontiguousarray(cell_ids, dtype=np.int64)
        _chk(lib().ep_stimulus_set(self._h, slot, ids.size, _p(ids, C.c_int64), amplitude, t_start, duration))

    def trigger_set(self, trigger, monitor_ids, slot, delay):
        ids = np.ascontiguousarray(monitor_ids, dtype=np.int64)
        _chk(lib().ep_trigger_set(self._h, int(trigger), ids.size, _p(ids, C.c_int64), int(slot), float(delay)))

    def trigger_time(self, trigger):
        d = C.c_double()
        _chk(lib().ep_trigger_time(self._h, int(trigger), C.byref(d)))
        return d.value

    def bidomain_solver(self, restart=30, max_cycles=200, rel_tol=1e-10):
        _chk(lib().ep_bidomain_solver(self._h, int(restart), int(max_cycles), float(rel_tol)))

    def read_vext(self, out=None):
        out = np.empty(self.n_tets) if out is None else out
        _chk(lib().ep_read_vext(self._h, _p(out)))
        return out

    def bidomain_stats(self):
        a, b, c, r = C.c_int64(), C.c_int64(), C.c_int64(), C.c_double()
        _chk(lib().ep_bidomain_stats(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(r)))
        return {"iters_last": a.value, "iters_total": b.value, "solves": c.value, "rel_res_last": r.value}

    def couple(self, trigger, dst, slot, delay):
        """ep_couple(self -> dst): True once dst's slot has been scheduled."""
        f = C.c_int()
        _chk(lib().ep_couple(self._h, int(trigger), dst._h, int(slot), float(delay), C.byref(f)))
        return bool(f.value)

    def set_time_order(self, order):
        _chk(lib().ep_set_time_order(self._h, int(order)))

    def step(self, n_steps, dt):
        _chk(lib().ep_step(self._h, int(n_steps), float(dt)))

    def synchronize(self):
        _chk(lib().ep_synchronize(self._h))

    def read_vm(self, out=None):
        out = np.empty(self.n_tets) if out is None else out
        _chk(lib().ep_read_vm(self._h, _p(out)))
        return out

    def read_state(self, var, out=None):
        out = np.empty(self.n_tets) if out is None else out
        _chk(lib().ep_read_state(self._h, int(var), _p(out)))
        return out

    def write_state(self, var, arr):
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        assert arr.size == self.n_tets
        _chk(lib().ep_write_state(self._h, int(var), _p(arr)))

    def write_states(self, arr):
        """All S rows at once, [S, n_tets] row-major (pinned memory makes the copies asynchronous)."""
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        assert arr.size == self.n_states * self.n_tets
        _chk(lib().ep_write_states(self._h, _p(arr)))

    def read_states(self, out=None):
        out = np.empty((self.n_states, self.n_tets)) if out is None else out
        assert out.size == self.n_states * self.n_tets and out.flags.c_contiguous
        _chk(lib().ep_read_states(self._h, _p(out)))
        return out

    def set_step_count(self, step_count, dt):
        _chk(lib().ep_set_step_count(self._h, int(step_count), float(dt)))

    def write_activation_times(self, arr):
        arr = np.ascontiguousarray(arr, dtype=np.float64)
        assert arr.size == self.n_tets
        _chk(lib().ep_write_activation_times(self._h, _p(arr)))

    def trigger_restore(self, trigger, t_fire):
        _chk(lib().ep_trigger_restore(self._h, int(trigger), float(t_fire)))

    def activation_times(self, out=None):
        out = np.empty(self.n_tets) if out is None else out
        _chk(lib().ep_activation_times(self._h, _p(out)))
        return out

    def mean_vm(self):
        d = C.c_double()
        _chk(lib().ep_mean_vm(self._h, C.byref(d)))
        return d.value

    def apply_diffusion(self, v):
        v = np.ascontiguousarray(v, dtype=np.float64)
        out = np.empty(self.n_tets)
        _chk(lib().ep_apply_diffusion(self._h, _p(v), _p(out)))
        return out

    def stable_dt(self):
        d = C.c_double()
        _chk(lib().ep_stable_dt(self._h, C.byref(d)))
        return d.value

    def check_finite(self):
        f = C.c_int()
        rc = lib().ep_check_finite(self._h, C.byref(f))
        if rc not in (0, -6):
            _chk(rc)
        return bool(f.value)

    def set_stream(self, cuda_stream: int | None):
        _chk(lib().ep_set_stream(self._h, _vp(cuda_stream) if cuda_stream else None))

    def device_vm(self):
        vm, perm = _vp(), _vp()
        _chk(lib().ep_device_vm(self._h, C.byref(vm), C.byref(perm)))
        return vm.value, perm.value

    def profile(self, enable: bool):
        _chk(lib().ep_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """{steps, ms_node, ms_cell}: per-kernel CUDA-event totals since ep_profile(1)."""
        out = np.zeros(4)
        _chk(lib().ep_profile_read(self._h, _p(out)))
        return {"steps": int(out[0]), "ms_node": float(out[1]), "ms_cell": float(out[2])}

    def kernel_bytes(self, kernel: int) -> int:
        return int(lib().ep_kernel_bytes(self._h, int(kernel)))

    @property
    def step_count(self):
        return int(lib().ep_step_count(self._h))

    @property
    def time(self):
        return float(lib().ep_time(self._h))

    @property
    def device_bytes(self):
        return int(lib().ep_device_bytes(self._h))

    @property
    def step_bytes(self):
        return int(lib().ep_step_bytes(self._h))

    @property
    def launch_count(self):
        return int(lib().ep_launch_count(self._h))
