#!/usr/bin/env python
"""bench.py -- fp64 cell-updates/s of the fused monodomain + TP06 step (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--inner 25] [--impl ours|reference]

One bench "step" = one ep_step(inner, dt) call = `inner` explicit time steps of the whole hot path (node gather + fused
cell kernel) over the whole synthetic mesh of the chosen BASELINE config (default: config 3, the
~2M-cell left-ventricle shell, the smallest of the ">= 2M cell" meshes the metric's 60 % target is quoted on).
Prints ONE JSON line (rank 0).  N > 1: independent replicas, one per GPU ("replicas only").
--impl reference times the CPU oracle (as it stands) on the host cores on a bounded sample of the same workload.

"e2e" is the same metric through the C-ABI with HOST buffers: every bench step is a self-contained job -- the config's initial
state (all S rows) and cleared activation times are copied in from pinned host memory (ep_write_states, ep_set_step_count,
ep_write_activation_times), `inner` time steps run, Vm and the activation times are read back -- with all copies inside the
timed region.  By default the jobs alternate between two handles of the same mesh so that the copies of one job overlap the
kernels of the other (what a caller with a stream of independent jobs does); `value_one_handle` is the same through one handle,
strictly in turn, and --e2e-handles 1 reports only that.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 cell-updates/sec (monodomain+TP06 step)"
UNIT = "cell-updates/s"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs (profiling recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, pw, reasons = [], [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        hi = [x for x in sm if x >= 0.5 * max(sm)]
        return {"sm_mhz": statistics.median(hi), "sm_max_mhz": max(smax), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def _run_dt(prob) -> float:
    """Time step the benchmark runs: the config's nominal dt, except where DESIGN.md reading S overrides it."""
    return float(prob.notes.get("dt_run", prob.dt))


def _oracle_leg(prob, budget_s: float, threads: int):
    """Time the oracle, as it stands, on this host: whole mesh, as many steps as fit the budget (at least 1)."""
    if hasattr(prob.mesh, "tris"):          # 2D medium: the triangle / Stewart oracle (OpenMP, all cores)
        from oracle import ep_oracle2d as O2
        o = O2.OracleSim2D.from_problem(prob)
    else:
        from oracle import ep_oracle as O
        O.set_threads(threads)
        o = O.OracleSim.from_problem(prob)
    t0 = time.perf_counter()
    o.step(1, _run_dt(prob))
    t1 = time.perf_counter() - t0
    n = max(1, min(400, int(budget_s / max(t1, 1e-6)) - 1))
    t0 = time.perf_counter()
    o.step(n, _run_dt(prob))
    t = time.perf_counter() - t0
    o.close()
    return prob.mesh.n_tets * n / t, n, t


def run_reference(args):
    """--impl reference: the oracle on the host cores; each bench step = --inner oracle time steps on the full mesh (fewer if they do not fit)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from ep_inputs import make
    from oracle import ep_oracle as O
    prob = make(args.config)
    cores = os.cpu_count() or 1
    O.set_threads(cores)
    o = O.OracleSim.from_problem(prob)
    # one bench step = the same `--inner` explicit time steps as the GPU arm's bench step when the whole run (warm-up included)
    # fits in about four minutes of oracle time on this host; otherwise as many as fit (at least one).  --ref-inner overrides.
    t0 = time.perf_counter()
    o.step(1, _run_dt(prob))
    t1 = max(time.perf_counter() - t0, 1e-6)
    fit = int(240.0 / (t1 * (args.steps + args.warmup)))
    per = args.ref_inner if args.ref_inner > 0 else max(1, min(args.inner, fit))
    for _ in range(args.warmup):
        o.step(per, _run_dt(prob))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(per, _run_dt(prob))
    t = time.perf_counter() - t0
    o.close()
    val = prob.mesh.n_tets * per * args.steps / t
    sample = f"config {args.config} full mesh ({prob.mesh.n_tets} cells), {per} oracle time step(s) per bench step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config(prob, _run_dt(prob), per, 1, int(os.environ.get("WORLD_SIZE", "1")), _step_bytes_formula(prob)),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def _step_bytes_formula(prob):
    """Algorithmic HBM bytes of one first-order time step (what ep_step_bytes returns), for the arm that
    has no handle: nc (16 S + 194) + 16 nn on a tetrahedral mesh."""
    S = {0: 19, 1: 21, 2: 20}[prob.model]
    return prob.mesh.n_tets * (16 * S + 194) + 16 * prob.mesh.n_nodes


def _config(prob, dt, inner, order, world, step_bytes):
    """The `config` object: the same keys and values in both arms (it names the workload, not the run)."""
    return {"workload": prob.name, "cells": prob.mesh.n_tets, "nodes": prob.mesh.n_nodes, "dt_ms": dt,
            "dt_nominal_ms": prob.dt, "dt_divisor": int(round(prob.dt / dt)), "time_steps_per_step": inner,
            "states": "config initial condition (rest + stimulus at t=0), window starts after warm-up",
            "l2": ("inputs larger than L2 (%.0f MB touched per time step)" if step_bytes > 126e6 else
                   "working set of %.0f MB per time step fits in L2 and is not flushed: a parity-size config, not a bench line")
                  % (step_bytes / 1e6),
            "time_order": order, "parallelism": "replicas" if world > 1 else "single"}


def max_over_ranks(x: float, dist, device) -> float:
    """MAX all-reduce of one timing scalar (the only collective of the N > 1 path: replicas share no data)."""
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, cells: int, inner: int, steps: int, ms_max: float) -> float:
    """cell-updates/s of all replicas together: every rank advances `cells` cells by inner*steps time steps."""
    return world * cells * inner * steps / (ms_max * 1e-3)


def run_disttest(args):
    """CPU-only check of the N > 1 plumbing (gloo): rank r reports (r + 1) ms; the job value uses the slowest rank."""
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist.init_process_group("gloo")
    dist.barrier()
    ms_max = max_over_ranks(float(rank + 1), dist, "cpu")
    val = whole_job_value(world, 1000, 10, 2, ms_max)
    if rank == 0:
        print(json.dumps({"impl": "disttest", "n_gpus": world, "ms_max": ms_max, "value": val, "scaling": "weak"}))
    dist.destroy_process_group()


def run_ours(args):
    import numpy as np
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libep has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    import paper_2112_12854_b200 as ep
    from ep_inputs import make
    prob = make(args.config)
    mesh = prob.mesh
    nc = mesh.n_tets
    sim = ep.Sim.from_problem(prob)
    stream = torch.cuda.Stream()
    sim.set_stream(stream.cuda_stream)
    if args.order == 2:
        sim.set_time_order(2)     # PAPER.md:232 variant (TP06 only); not the headline configuration
    S = sim.n_states
    # explicit stability (reading S): config 2 runs at dt = nominal/4; ep_stable_dt confirms the choice
    dt_max = sim.stable_dt()
    dt = _run_dt(prob)
    dt_k = int(round(prob.dt / dt))
    if dt > dt_max:
        raise SystemExit(f"bench.py: dt = {dt} ms exceeds the explicit stability limit {dt_max:.5f} ms of this mesh")
    inner = args.inner
    # the config as specified: every cell at the model's resting state, the config's stimulus armed at t = 0; the
    # timed window is the start of that simulation (stimulus on, wave leaving the stimulus sites)
    pinned = torch.empty((S, nc), dtype=torch.float64).pin_memory()
    sim.read_states(pinned.numpy())
    out_vm = torch.empty(nc, dtype=torch.float64).pin_memory()
    out_ta = torch.empty(nc, dtype=torch.float64).pin_memory()

    tact0 = torch.full((nc,), -1.0, dtype=torch.float64).pin_memory()

    def upload(h=None):
        # one self-contained job: the config's initial state, clock at t = 0, no cell activated yet
        h = h or sim
        h.write_states(pinned.numpy())        # all S rows, one call: pipelined copies + permutation kernels, one sync
        h.set_step_count(0, dt)
        h.write_activation_times(tact0.numpy())
        for k in range(len(getattr(prob, "triggers", []))):
            h.trigger_restore(k, -1.0)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident arm
    for _ in range(args.warmup):
        sim.step(inner, dt)
    sim.synchronize()
    l0 = sim.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clocks = ClockSampler(local) if rank == 0 else None
    with torch.cuda.stream(stream):
        e0.record(stream)
        for _ in range(args.steps):
            sim.step(inner, dt)
        e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches_timed = sim.launch_count - l0
    # second, identical pass with a CUDA-event pair around every kernel launch (ep_profile): per-kernel durations for
    # the roofline.  Kept out of the pass above because the extra event records cost a few us per time step.
    sim.profile(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        p0.record(stream)
        for _ in range(args.steps):
            sim.step(inner, dt)
        p1.record(stream)
    barrier()
    ms_profiled = p0.elapsed_time(p1)
    clk = clocks.stop() if clocks else None
    prof = sim.profile_read()
    sim.profile(False)
    launches = launches_timed
    finite = sim.check_finite()
    ms_max = max_over_ranks(ms, dist, "cuda")
    value = whole_job_value(world, nc, inner, args.steps, ms_max)

    # ---------------- end-to-end arm: host state in, Vm + activation times out, every bench step
    def e2e_step():
        upload()
        sim.step(inner, dt)
        sim.read_vm(out_vm.numpy())
        sim.activation_times(out_ta.numpy())

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    n_e2e = max(3, min(args.steps, 10))
    for _ in range(n_e2e):
        e2e_step()
    barrier()
    e2e_one = whole_job_value(world, nc, inner, n_e2e, 1e3 * max_over_ranks(time.perf_counter() - t0, dist, "cuda"))
    e2e_val, e2e_handles = e2e_one, 1
    if args.e2e_handles == 2:
        # the same jobs through TWO handles of the same mesh, double-buffered: while one handle advances its `inner` time
        # steps the other one takes the next job's host state (ep_write_states) and hands back the previous job's result
        # (ep_read_vm, ep_activation_times).  Every job still copies all its inputs in and its result out, from / to pinned
        # host memory, inside the timed region; the copies of one job overlap the kernels of the other.
        sim_b = ep.Sim.from_problem(prob)
        if args.order == 2:
            sim_b.set_time_order(2)
        pair = (sim, sim_b)
        out_b = (torch.empty(nc, dtype=torch.float64).pin_memory(), torch.empty(nc, dtype=torch.float64).pin_memory())
        outs = ((out_vm, out_ta), out_b)

        def submit(k):
            upload(pair[k % 2])
            pair[k % 2].step(inner, dt)

        def collect(k):
            pair[k % 2].read_vm(outs[k % 2][0].numpy())
            pair[k % 2].activation_times(outs[k % 2][1].numpy())

        def pipeline(n):
            submit(0)
            for k in range(n):
                if k + 1 < n:
                    submit(k + 1)
                collect(k)

        pipeline(2)
        barrier()
        t0 = time.perf_counter()
        pipeline(n_e2e)
        barrier()
        e2e_val = whole_job_value(world, nc, inner, n_e2e, 1e3 * max_over_ranks(time.perf_counter() - t0, dist, "cuda"))
        e2e_handles = 2
        same = bool(np.array_equal(outs[0][0].numpy(), outs[1][0].numpy()) and np.array_equal(outs[0][1].numpy(), outs[1][1].numpy()))
        if not same:
            raise SystemExit("bench.py: the two handles of the end-to-end arm disagree")
        sim_b.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak, peak_src, _ = _peaks()
    cell_bytes = sim.kernel_bytes(1)
    cell_ms = prof["ms_cell"] / max(1, prof["steps"])
    node_ms = prof["ms_node"] / max(1, prof["steps"])
    achieved = cell_bytes / (cell_ms * 1e-3) / 1e9
    # figures read from the committed ncu capture of this workload (profiles/traffic.json names the capture): DRAM bytes
    # per launch and fp64 warp instructions per warp (= fp64 instructions per cell-step) of the dominant kernel
    cap = {}
    try:
        cap = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(prob.name, {})
    except Exception:
        cap = {}
    traffic = args.traffic if args.traffic is not None else cap.get("bytes_per_launch")
    fp64_inst = cap.get("fp64_inst_per_cell_step")
    hbm_floor_ms = cell_bytes / (peak * 1e9) * 1e3
    # the other roof (t_roof = max(bytes / BW_HBM, I_alg / R_fp64)): fp64 instructions the kernel executes
    # (ncu) over the DFMA issue rate of this GPU measured in this run, after the timed region, at whatever clock the
    # power cap then allows (ep_fp64_rate: a DFMA-only kernel)
    fp64_rate = ep.fp64_rate()
    fp64_floor_ms = (nc / 32.0) * fp64_inst / fp64_rate * 1e3 if fp64_inst else None
    roof_ms = max(hbm_floor_ms, fp64_floor_ms or 0.0)
    roofline = {"bound": "hbm", "kernel": "cell_step_kernel<%d>" % prob.model, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src, "traffic": traffic,
                "alg_bytes_per_launch": cell_bytes, "alg_bytes_per_cell": cell_bytes / nc,
                "avg_launch_ms": cell_ms, "node_kernel_avg_launch_ms": node_ms,
                "kernel_share_of_step": cell_ms / max(1e-12, cell_ms + node_ms),
                "profiled_pass_ms_per_step": ms_profiled / args.steps,
                "hbm_floor_ms": hbm_floor_ms,
                "fp64": {"warp_dfma_per_s_measured": fp64_rate, "tflops_measured": fp64_rate * 64 / 1e12,
                         "inst_per_cell_step": fp64_inst, "inst_source": cap.get("source"),
                         "floor_ms": fp64_floor_ms,
                         "frac": (fp64_floor_ms / cell_ms) if fp64_floor_ms else None},
                "roof": "fp64" if (fp64_floor_ms or 0.0) > hbm_floor_ms else "hbm",
                "roof_ms": roof_ms, "roof_frac": roof_ms / cell_ms,
                "whole_step_frac": sim.step_bytes / (ms_max * 1e-3 / (inner * args.steps)) / 1e9 / peak}
    cores = os.cpu_count() or 1
    cpu_val, cpu_n, cpu_t = _oracle_leg(prob, args.cpu_budget, cores)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": _config(prob, dt, inner, args.order, world, sim.step_bytes),
        "dt_stable_max_ms": dt_max,
        "simulated_ms_per_wall_s": dt * inner * args.steps / (ms_max * 1e-3),
        "us_per_time_step": 1e3 * ms_max / (inner * args.steps),
        "clocks": clk, "gpu_launches": launches, "all_finite": bool(finite),
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 8 * (S + 1) * nc, "d2h_bytes_per_step": 16 * nc,
                "steps": n_e2e, "handles": e2e_handles, "value_one_handle": e2e_one,
                "how": ("two handles, double-buffered: the copies of one job overlap the kernels of the other"
                        if e2e_handles == 2 else "one handle: upload, step, read back, strictly in turn")},
        "roofline": roofline,
        "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"config {args.config} full mesh ({nc} cells), {cpu_n} time steps, {cpu_t:.1f} s"},
    }
    print(json.dumps(out))
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "disttest"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..5; 6/7/8 = the paper's Table-1 slab at dx 0.5/0.2/0.1 mm; 9/10 = Purkinje strip / sheet (2D, Stewart)")
    ap.add_argument("--inner", type=int, default=100, help="explicit time steps per bench step")
    ap.add_argument("--e2e-handles", type=int, default=2, choices=(1, 2),
                    help="end-to-end arm: 2 = jobs alternate between two handles so that copies overlap compute (default); 1 = serial")
    ap.add_argument("--ref-inner", type=int, default=0,
                    help="oracle time steps per bench step (--impl reference); 0 = --inner if the run fits in ~4 minutes, else fewer")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--order", type=int, default=1, choices=[1, 2],
                    help="time-stepping order: 1 = the paper's Rush-Larsen + forward Euler (headline), 2 = AB2 + second-order Rush-Larsen")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "disttest":
        run_disttest(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
