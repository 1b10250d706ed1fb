"""N > 1 path of bench.py on CPU (gloo, world size 2): replicas only, no data-path collective."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(extra, port):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--gpus", "2"] + extra
    env = dict(os.environ, OMP_NUM_THREADS="2")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout          # rank 0 alone prints, exactly one JSON line
    return json.loads(lines[0])


def test_max_over_ranks_and_whole_job_value():
    d = _torchrun(["--impl", "disttest"], 29631)
    assert d["n_gpus"] == 2 and d["ms_max"] == 2.0            # slowest rank decides
    assert d["value"] == 2 * 1000 * 10 * 2 / 2.0e-3           # both replicas' cell-updates over that time
    assert d["scaling"] == "weak"


def test_reference_arm_under_torchrun_runs_on_rank0_only():
    d = _torchrun(["--impl", "reference", "--config", "1", "--steps", "3", "--warmup", "3"], 29632)
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "C1_tiny_slab" and d["unit"] == "cell-updates/s"


def test_whole_job_value_formula():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(1, 2_000_000, 100, 20, 500.0) == 2_000_000 * 100 * 20 / 0.5
    assert bench.whole_job_value(8, 10, 1, 1, 1.0) == 8 * 10 / 1e-3
