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


SLAB_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["LBM_ROOT"])
import torch, torch.distributed as dist
from paper_1405_1253_b200.slab_ring import partition, exchange_messages
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
Lx = 24
parts = partition(70, world)
z0, nz = parts[rank]
# a message is 26 population-rows of Lx doubles; the payload names its sender and direction
up = torch.full((26 * Lx,), 100.0 + rank, dtype=torch.float64)
dn = torch.full((26 * Lx,), 200.0 + rank, dtype=torch.float64)
below, above = torch.zeros(26 * Lx, dtype=torch.float64), torch.zeros(26 * Lx, dtype=torch.float64)
for step in range(3):
    up += 1000.0; dn += 1000.0
    for r in exchange_messages(up, dn, below, above, rank, world):
        r.wait()
    if rank > 0:
        assert torch.all(below == 100.0 + (rank - 1) + 1000.0 * (step + 1)), (rank, step, below[0])
    else:
        assert torch.all(below == 0)
    if rank + 1 < world:
        assert torch.all(above == 200.0 + (rank + 1) + 1000.0 * (step + 1)), (rank, step, above[0])
    else:
        assert torch.all(above == 0)
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"ok{rank}:{z0}+{nz}\n"); sys.stdout.flush()
"""


def test_slab_partition_and_message_ring_world3(tmp_path):
    """Host logic of the z-slab path (bench.py --slabs): balanced contiguous partition, and the per-step exchange
    pattern -- up-message to rank+1's lower ghost rows, down-message to rank-1's upper ghost rows, nothing across the
    walls -- as three gloo processes on CPU."""
    sys.path.insert(0, ROOT)
    from paper_1405_1253_b200.slab_ring import partition
    assert partition(8192, 8) == [(1024 * r, 1024) for r in range(8)]
    p = partition(70, 3)
    assert p == [(0, 24), (24, 23), (47, 23)] and sum(n for _, n in p) == 70
    with pytest.raises(ValueError):
        partition(17, 3)                      # slabs must hold both edge zones: at least 6 rows
    script = tmp_path / "slab_worker.py"
    script.write_text(SLAB_WORKER)
    env = dict(os.environ, LBM_ROOT=ROOT, OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=3",
                          "--master-addr", "127.0.0.1", "--master-port", "29654", str(script)],
                         env=env, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert "ok0:0+24" in out.stdout and "ok1:24+23" in out.stdout and "ok2:47+23" in out.stdout


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
