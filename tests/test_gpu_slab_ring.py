"""SURVEY 8(f)4 / VERDICT r2 items 2-3: the rank-to-rank schedule of the z-slab path, executed.

Two processes (torch.distributed.run) share the one GPU of the box; their group is gloo, so SlabRing stages the
messages through pinned host buffers -- everything else (pack on the exchange stream, interior rows on the main stream
while the messages travel, unpack, edge rows; pairs of steps with the two-step kernel, single steps with the one-step
kernel) is the schedule an NCCL group runs.  Each rank compares its own rows bit for bit with a whole-lattice run of its
own.  The ranks' kernels never wait on one another on the device: every transfer completes on the host first."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["LBM_ROOT"])
import torch, torch.distributed as dist
import paper_1405_1253_b200 as pkg
import synthetic_inputs as si
from paper_1405_1253_b200.slab_ring import SlabRing
torch.cuda.set_device(0)
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
Lx, Lz, tau, g = int(os.environ["LBM_LX"]), int(os.environ["LBM_LZ"]), 0.75, 2e-4
fields = si.sweep_fields_torch(Lx, Lz, 21, "cuda")
checked = 0
for wall_kind in (0, 1):
    kw = dict(wall_kind=wall_kind, T_wall=(1.02, 0.97))
    for fused in (True, False):
        whole = pkg.Lattice(Lx, Lz, tau, g, **kw)
        whole.init_equilibrium(*fields)
        ring = SlabRing(Lx, Lz, tau, g, rank, world, **kw)
        assert ring.staged
        rows = slice(ring.z0, ring.z0 + ring.nz)
        ring.slab.init_equilibrium(*[x[rows].contiguous() for x in fields])
        for n in (1, 2, 7, 20):
            whole.step(n)
            ring.step(n, fused=fused)
            torch.cuda.synchronize()
            assert torch.equal(ring.slab.get_populations(), whole.get_populations()[:, rows]), (rank, wall_kind, fused, n)
            checked += 1
        ring.close(); whole.close()
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"ok{rank}:{checked}\n"); sys.stdout.flush()
"""


@pytest.mark.gpu
@pytest.mark.parametrize("Lx,Lz,world", [(200, 150, 2), (520, 96, 3)])
def test_slab_ring_steps_between_processes_equal_the_whole_lattice(tmp_path, Lx, Lz, world):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import __graft_entry__ as g
    g.build()
    script = tmp_path / "ring_worker.py"
    script.write_text(WORKER)
    env = dict(os.environ, LBM_ROOT=ROOT, OMP_NUM_THREADS="1", LBM_LX=str(Lx), LBM_LZ=str(Lz))
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={world}",
                          "--master-addr", "127.0.0.1", "--master-port", "29671", str(script)],
                         env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, (out.stdout[-1500:], out.stderr[-3000:])
    for r in range(world):
        assert f"ok{r}:16" in out.stdout, out.stdout


@pytest.mark.gpu
def test_bench_slabs_runs_between_two_processes_on_one_gpu():
    """bench.py --slabs (run_slabs), the strong-scaling mode, with `--backend gloo`: two ranks on the one GPU."""
    import json
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29672", os.path.join(ROOT, "bench.py"),
                          "--slabs", "--backend", "gloo", "--config", "2", "--steps", "20", "--warmup", "4", "--gpus", "2"],
                         env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, (out.stdout[-1500:], out.stderr[-3000:])
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["scaling"] == "strong" and line["n_gpus"] == 2 and line["value"] > 0 and line["gpu_launches"] > 0
    assert 2.0 < line["config"]["L_u"] < 20.0 and 2.0 < line["config"]["L_d"] < 20.0
