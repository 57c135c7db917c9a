#!/usr/bin/env python
"""bench.py -- MLUPS (FP64) of the fused thermal D2Q37 LB step on B200, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4] [--variant V]

One "step" = one pass of the whole hot path (periodic wrap + propagate + bc + collide + swap, SURVEY 8(a)
a1-a5) over the resident lattice; the diagnostics row a6 (mixing widths, eq. 12) runs once per timed
region and is inside it.  N = 1 workload: BASELINE.json configs[3], the 4096x8192 single-front RT lattice
the headline metric is quoted on (~20 GB of populations resident).  N > 1: the path does not shard in this
deliverable ("replicas only"): every rank runs an independent replica with its own seed, no
data-path collective, weak scaling.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synthetic_inputs as si  # noqa: E402

BYTES_PER_SITE = 592          # 37 x 8 B read + 37 x 8 B written per site per step
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel at 4096x8192, from the committed
# `ncu --set full` capture (profiles/); None until a capture exists for the default variant.
NCU_TRAFFIC_BYTES = None


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, device_index: int):
        super().__init__(daemon=True)
        self.samples, self.mask, self.max_mhz, self.ok = [], 0, None, False
        self._stop = threading.Event()
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            uuid = str(torch.cuda.get_device_properties(device_index).uuid)
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.nv = pynvml
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        while self.ok and not self._stop.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            time.sleep(0.02)

    def finish(self) -> dict:
        self._stop.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "samples": len(s),
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b]}


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_sample_rate(cfg, budget_s: float, threads: int | None = None):
    """Times the CPU oracle, as it stands, on a bounded sample of `cfg`: a slab of full width Lx and `rows`
    rows around the interface, stepped until ~budget_s of CPU time is spent.  Returns (MLUPS, cores, text)."""
    from oracle import lbm_oracle as orc
    cores = threads or orc.max_threads()
    orc.set_threads(cores)
    rows = 64
    sub = si.scaled(cfg, cfg.Lx, rows)
    f = orc.init_rt(sub.Lx, sub.Lz, sub.g, si.DEFAULT_SEED, **sub.rt_args())
    t0 = time.perf_counter(); f = orc.step(f, sub.tau, sub.g, nsteps=1); t1 = time.perf_counter() - t0
    n = max(2, int(budget_s / max(t1, 1e-6)))
    t0 = time.perf_counter(); orc.step(f, sub.tau, sub.g, nsteps=n); dt = time.perf_counter() - t0
    mlups = sub.Lx * rows * n / dt / 1e6
    return mlups, cores, f"{sub.Lx}x{rows} slab of {cfg.name} around the interface, {n} steps, {dt:.1f} s"


def run_reference(args):
    """--impl reference: the oracle on the host cores, one bounded slab step per bench 'step'."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import lbm_oracle as orc
    cfg = si.rt_config(args.config)
    cores = orc.max_threads()
    orc.set_threads(cores)
    probe = si.scaled(cfg, cfg.Lx, 16)
    f = orc.init_rt(probe.Lx, probe.Lz, probe.g, si.DEFAULT_SEED, **probe.rt_args())
    t0 = time.perf_counter(); orc.step(f, probe.tau, probe.g, nsteps=1); t1 = time.perf_counter() - t0
    rate = probe.Lx * 16 / t1                                  # sites / s
    total = args.steps + args.warmup
    rows = int(min(cfg.Lz, max(8, rate * 120.0 / total / cfg.Lx)))   # whole run ~2 minutes
    sub = si.scaled(cfg, cfg.Lx, rows)
    f = orc.init_rt(sub.Lx, sub.Lz, sub.g, si.DEFAULT_SEED, **sub.rt_args())
    f = orc.step(f, sub.tau, sub.g, nsteps=args.warmup)
    t0 = time.perf_counter(); orc.step(f, sub.tau, sub.g, nsteps=args.steps); dt = time.perf_counter() - t0
    mlups = sub.Lx * rows * args.steps / dt / 1e6
    sample = f"{sub.Lx}x{rows} slab of {cfg.name} around the interface per step"
    print(json.dumps({
        "impl": "reference", "metric": "MLUPS (FP64)", "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "Lx": cfg.Lx, "Lz": cfg.Lz, "tau": cfg.tau, "g": cfg.g, "sample": sample},
        "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
