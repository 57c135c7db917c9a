"""Host-side logic of bench.py's N > 1 path ("replicas only"), run as two gloo processes on CPU, and the
reference arm's rank handling.  No GPU."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["LBM_ROOT"])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
t = bench.reduce_max([1.0 + rank, 5.0 - rank], world, "cpu")
assert t == [float(world), 5.0], t
v = bench.whole_job_mlups(1000, 10, world, t[0])
assert abs(v - world * 1000 * 10 / world / 1e6) < 1e-12
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"ok{rank}\n"); sys.stdout.flush()
"""


def test_max_over_ranks_and_whole_job_value_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, LBM_ROOT=ROOT, OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29653", str(script)],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "ok0" in out.stdout and "ok1" in out.stdout


def test_reference_arm_prints_one_line_on_rank0_only():
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "3",
           "--warmup", "3", "--gpus", "2"]
    r0 = subprocess.run(cmd, env=dict(os.environ, RANK="0", WORLD_SIZE="2"), capture_output=True, text=True, timeout=300)
    r1 = subprocess.run(cmd, env=dict(os.environ, RANK="1", WORLD_SIZE="2"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0 and r1.returncode == 0 and r1.stdout.strip() == ""
    line = json.loads(r0.stdout.strip())
    assert line["impl"] == "reference" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"] == "rt_double_64x128" and line["dtype"] == "f64"


def test_our_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--steps", "3"], capture_output=True,
                       text=True, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in (r.stderr + r.stdout)
