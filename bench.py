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
FLOPS_PER_SITE = 559          # FP64 flops of one collision as the KERNEL evaluates it, FMA = 2: 196 DFMA + 89 DADD + 78 DMUL in the SASS
FLOPS_PER_SITE_ORACLE = 2939  # FP64 operations per site-step of the ORACLE as written (oracle/lbm_oracle.c: site_moments 596, shift 8,
                              # orc_feq 4 + 37 x 59, relaxation 37 x 4), every arithmetic operator counted once, FMA = 2
FALLBACK_HBM_GBS = 6650.0     # /opt/skills/guides/B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel from the committed `ncu --set full`
# captures under profiles/ -- NOT measured in this run: reported with its source file, and only when this run's launch
# (workload, steps per launch, strip width, rows per chunk) is the one that was captured; null otherwise.
# The key ends with the git blob hash of the kernel's source file at capture time: an edit to the kernel nulls the figure
# until the capture is redone.
NCU_TRAFFIC = {
    ("rt_single_4096x8192", 1, None, None, "lbm_step.cuh", "f0747db8b6c7e93d7466d3f6ff90472b7d15c26c"): (19.839e9, "profiles/r2_step_kernels_full.md"),
    ("rt_single_4096x8192", 2, 56, 410, "lbm_step2s.cuh", "18b59ca29fdd9930f533092bc42a60318d81d938"): (20.210e9, "profiles/r3_step2s_kernel_full.md"),
}


def git_blob_hash(path: str) -> str:
    """What `git hash-object` prints for the file (sha1 of "blob <size>\\0" + contents)."""
    import hashlib
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_traffic(workload, spl, strip_w, zchunk):
    src = "lbm_step2s.cuh" if spl > 1 else "lbm_step.cuh"
    blob = git_blob_hash(os.path.join(ROOT, "paper_1405_1253_b200", "csrc", src))
    key = (workload, spl, strip_w if spl > 1 else None, zchunk if spl > 1 else None, src, blob)
    return NCU_TRAFFIC.get(key, (None, None))


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
        self._halt = threading.Event()
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
        while self.ok and not self._halt.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
            except Exception:
                pass
            time.sleep(0.002)

    def mark(self):
        """The timed region starts here: only later samples (and their throttle reasons) are reported."""
        self._first = len(self.samples)
        self.mask = 0

    def finish(self) -> dict:
        self._halt.set()
        if self.is_alive():
            self.join()
        mine = self.samples[getattr(self, "_first", 0):]
        if not mine:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        s = sorted(mine)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "samples": len(s), "period_ms": 2,
                "reasons": [n for b, n in self.REASONS.items() if self.mask & b]}


# ------------------------------------------------------------------------------------------ oracle legs
_HOST_CORES = None


def host_cores() -> int:
    """Threads the oracle's OpenMP loops get by default on this box (asked once, before any orc_set_threads)."""
    global _HOST_CORES
    if _HOST_CORES is None:
        from oracle import lbm_oracle as orc
        _HOST_CORES = orc.max_threads()
    return _HOST_CORES


def oracle_sample_rate(cfg, budget_s: float, threads: int | None = None):
    """Times the CPU oracle, as it stands, on a bounded sample of `cfg`: a slab of full width Lx and `rows`
    rows around the interface, stepped until ~budget_s of CPU time is spent.  Returns (MLUPS, cores, text)."""
    from oracle import lbm_oracle as orc
    cores = threads or host_cores()
    orc.set_threads(cores)
    rows = 64
    sub = si.scaled(cfg, cfg.Lx, rows)
    f = orc.init_rt(sub.Lx, sub.Lz, sub.g, si.DEFAULT_SEED, **sub.rt_args())
    f = orc.step(f, sub.tau, sub.g, nsteps=2)                     # untimed: thread start-up, page faults
    n, dt, batch = 0, 0.0, 8
    while dt < budget_s:                                          # doubling batches until the budget is spent
        t0 = time.perf_counter(); f = orc.step(f, sub.tau, sub.g, nsteps=batch); dt += time.perf_counter() - t0
        n += batch
        batch = min(2 * batch, max(8, int(n / max(dt, 1e-6) * max(budget_s - dt, 0.0)) + 1))
    mlups = sub.Lx * rows * n / dt / 1e6
    return mlups, cores, f"{sub.Lx}x{rows} slab of {cfg.name} around the interface, {n} steps, {dt:.1f} s"


def oracle_named_samples():
    """The two oracle timings SURVEY 8(d) / BASELINE.md section 3 name: config 1 (64x128, 100 steps) and 512x1024 for
    10 steps, each single-threaded and on all host cores.  Returns a list of dicts (MLUPS)."""
    from oracle import lbm_oracle as orc
    out = []
    allc = host_cores()
    for idx, steps in ((1, 100), (2, 10)):
        cfg = si.rt_config(idx)
        f0 = orc.init_rt(cfg.Lx, cfg.Lz, cfg.g, si.DEFAULT_SEED, **cfg.rt_args())
        for threads in (1, allc):
            orc.set_threads(threads)
            orc.step(f0, cfg.tau, cfg.g, nsteps=1)                 # untimed: thread start-up, page faults
            t0 = time.perf_counter(); orc.step(f0, cfg.tau, cfg.g, nsteps=steps); dt = time.perf_counter() - t0
            out.append({"sample": f"{cfg.name}, {steps} steps", "threads": threads,
                        "value": cfg.Lx * cfg.Lz * steps / dt / 1e6, "unit": "MLUPS", "seconds": dt})
    orc.set_threads(allc)
    return out


def run_reference(args):
    """--impl reference: the oracle on the host cores, one bounded slab step per bench 'step'."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import lbm_oracle as orc
    cfg = si.rt_config(args.config)
    cores = host_cores()
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


# ------------------------------------------------------------------------------------------ our arm
def reduce_max(values, world: int, device: str):
    """MAX over ranks of a list of per-rank timings (one process per GPU; gloo on CPU in the tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def whole_job_mlups(sites_per_rank: int, steps: int, world: int, seconds_max: float) -> float:
    """Replicas only: every rank updates its own lattice; the job's rate is all sites over the slowest rank."""
    return world * sites_per_rank * steps / seconds_max / 1e6


def a6_kernel_times(lat, cfg, stream, torch, reps: int = 5):
    """Row a6 kernels at this workload, timed with CUDA events outside the driver's timed region: moments_kernel (reads
    the 37 populations, writes rho, u_x, u_z, T: 328 B per site) and the one-pass diagnostics
    (row_diagnostics_kernel<false> + final_diagnostics_kernel: 296 B per site read; <true> re-reads each row for the
    squared deviations, from L2).  Peak: the measured copy bandwidth.  Traffic: profiles/r3_a6_kernels.md."""
    peak, peak_kind = measured_peak()
    sites = cfg.Lx * cfg.Lz
    fields = [torch.empty((cfg.Lz, cfg.Lx), dtype=torch.float64, device="cuda") for _ in range(4)]

    def timed(fn):
        fn(); torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream); torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    out = {"peak": peak, "peak_kind": peak_kind, "unit": "GB/s", "bound": "hbm"}
    for name, nbytes, fn in (
            ("moments_kernel", 328, lambda: lat.moments(*fields)),
            ("row_diagnostics_kernel<false>+final", 296, lambda: lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u, profiles=False)),
            ("row_diagnostics_kernel<true>+final", 296, lambda: lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u, profiles=True, rms=True))):
        t = timed(fn)
        out[name] = {"bytes_per_site": nbytes, "ms": t * 1e3, "achieved": nbytes * sites / t / 1e9,
                     "frac": nbytes * sites / t / 1e9 / peak}
    out["note"] = "the diagnostics calls copy their results to the host and synchronise: their time includes that"
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    import __graft_entry__ as entry
    import paper_1405_1253_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        entry.build()
    if world > 1:
        dist.barrier()

    cfg = si.rt_config(args.config)
    if args.lx and args.lz:
        cfg = si.scaled(cfg, args.lx, args.lz)
    sites = cfg.Lx * cfg.Lz
    stream = torch.cuda.current_stream()
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, wall_kind=args.wall_kind, T_wall=(cfg.T_d, cfg.T_u))
    if args.variant is not None:
        lat.set_variant(args.variant)
    if args.zchunk:
        lat.set_zchunk(args.zchunk)
    lat.init_rt(si.DEFAULT_SEED + rank, **cfg.rt_args())     # replicas differ only by their seed
    fused, strip_w, zchunk = lat.plan()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps + one widths call
    sampler = ClockSampler(local)                            # running before the warm-up, so that it is sampling at
    sampler.start()                                          # full rate when the (short) timed region begins
    lat.step(args.warmup)
    lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u, want_tbar=False)
    barrier()
    sampler.mark()
    l0 = lat.kernel_launches
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    ev[0].record(stream)
    lat.step(args.steps)                                     # K (one-step) or K/2 (two-step kernel) launches
    ev[1].record(stream)
    step_launches = lat.kernel_launches - l0
    widths = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u, want_tbar=False)   # a6, synchronises
    ev[2].record(stream)
    barrier()
    clocks = sampler.finish()
    launches = lat.kernel_launches - l0
    t_steps = ev[0].elapsed_time(ev[1]) * 1e-3
    t_total = ev[0].elapsed_time(ev[2]) * 1e-3
    t_total, t_steps = reduce_max([t_total, t_steps], world, "cuda")
    value = whole_job_mlups(sites, args.steps, world, t_total)

    # ---- sustained leg (not the driver's timed region): the contract's K steps can be a burst of a few tens of
    # milliseconds at full boost, while a long run settles at the clock the 1 kW power cap allows.  The same call is
    # repeated for >= `--sustain` seconds (default 3 s, >= 200 steps) and timed with CUDA events the same way.
    sustained = None
    if args.sustain > 0:
        n_sus = max(200, int(args.sustain / max(t_steps / args.steps, 1e-6)) // 2 * 2)
        barrier()
        s2 = ClockSampler(local)
        s2.start()
        ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev2[0].record(stream)
        lat.step(n_sus)
        ev2[1].record(stream)
        barrier()
        c2 = s2.finish()
        t_sus = reduce_max([ev2[0].elapsed_time(ev2[1]) * 1e-3], world, "cuda")[0]
        sustained = {"value": whole_job_mlups(sites, n_sus, world, t_sus), "unit": "MLUPS", "steps": n_sus,
                     "seconds": t_sus, "ms_per_step": t_sus / n_sus * 1e3, "sm_mhz": c2.get("sm_mhz"),
                     "reasons": c2.get("reasons")}

    # ---- end to end through lbm_run_host: pinned host fields in, K steps, host fields out
    a6 = a6_kernel_times(lat, cfg, stream, torch) if rank == 0 else None
    host_in = [x.cpu().pin_memory() for x in lat.kinetic_moments()]     # what lbm_run_host takes (lbm_kinetic_moments)
    host_out = tuple(torch.empty_like(x).pin_memory() for x in host_in)
    fp64_peak = max(pkg.fp64_peak() for _ in range(2))                  # TFLOP/s, DFMA chains on all SMs (clock under load)
    e2e_steps = args.e2e_steps or args.steps
    lat.run_host(*host_in, n=min(3, e2e_steps), outs=host_out)          # warm-up (allocates staging)
    barrier()
    t0 = time.perf_counter()
    lat.run_host(*host_in, n=e2e_steps, outs=host_out)                   # synchronous
    t_e2e = reduce_max([time.perf_counter() - t0], world, "cuda")[0]
    field_bytes = 4 * 8 * sites
    e2e = {"value": whole_job_mlups(sites, e2e_steps, world, t_e2e), "unit": "MLUPS", "steps": e2e_steps,
           "h2d_bytes_per_step": field_bytes / e2e_steps, "d2h_bytes_per_step": field_bytes / e2e_steps,
           "call": "lbm_run_host (pinned host rho,u,T in -> init -> K steps -> host rho,u,T out)"}
    lat.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_kind = measured_peak()
    # Dominant kernel: the step kernel.  Algorithmic bytes per launch = 592 B/site/step x sites x
    # the steps one launch advances (1: step_kernel_site, 2: step2s_kernel, which keeps the intermediate lattice
    # in shared memory, so its DRAM traffic -- `traffic`, from ncu -- is about half its algorithmic bytes and
    # `frac` can exceed 1: DESIGN.md section 6).  Launch duration = CUDA-event time of the K steps / launches.
    # Launches of the STEP kernel in the timed region: with the two-step kernel K // 2 fused launches (+ one single step if
    # K is odd); `step_launches` (all kernels the library launched while stepping) can hold one more, the refresh of the
    # wrap columns after a warm-up that ended on a single step (~30 us).  The roofline is that of the dominant kernel:
    # an even K gives whole fused launches; their duration is the stepping time over their number.
    n_step_kernels = (args.steps // 2 + args.steps % 2) if fused else args.steps
    if args.variant in (1, 2):
        n_step_kernels = args.steps
    # tiny lattices: ONE cooperative launch of step_persistent_kernel runs all K steps (the handle counted one launch)
    persistent = not fused and args.variant in (None, 0) and step_launches == 1 and args.steps > 1
    if persistent:
        n_step_kernels = 1
    spl = args.steps / max(n_step_kernels, 1)
    launch_ms = t_steps / max(n_step_kernels, 1) * 1e3
    alg_bytes = BYTES_PER_SITE * sites * spl
    achieved = alg_bytes / (launch_ms * 1e-3) / 1e9
    # what the kernel cannot avoid moving through DRAM per launch, whatever its fused depth: one read and one write
    # of the lattice (the intermediate lattice of the two-step kernel lives in shared memory only)
    compulsory = BYTES_PER_SITE * sites
    own_gbs = compulsory / (launch_ms * 1e-3) / 1e9
    whole = abs(spl - round(spl)) < 1e-9
    traffic, traffic_source = ncu_traffic(cfg.name, int(round(spl)), strip_w, zchunk) if whole and args.wall_kind == 0 else (None, None)
    rate = sites * spl / (launch_ms * 1e-3)                        # site-steps per second of the kernel
    roofline = {"bound": "hbm",
                "kernel": "step_persistent_kernel (all K steps in one cooperative launch, grid barrier between steps; L2-resident)" if persistent
                else "step2s_kernel (two fused propagate+bc+collide steps per launch)" if spl > 1.5
                else "step_kernel_site (fused propagate+bc+collide)",
                "frac_of_compulsory_dram": own_gbs / peak,
                "achieved": achieved, "peak": peak,
                "peak_kind": f"{peak_kind} copy bandwidth (MEASURED_PEAKS.json hbm_gbs)",
                "unit": "GB/s", "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / 8000.0,
                "bytes_per_site_step": BYTES_PER_SITE, "steps_per_launch": spl, "launches": n_step_kernels, "all_launches_while_stepping": step_launches,
                "launch_plan": {"fused": fused, "strip_width": strip_w, "rows_per_chunk": zchunk},
                "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": launch_ms,
                "note": ("`achieved`/`frac` count the ALGORITHMIC 592 B per site and step (SURVEY 8(d)). With steps_per_launch"
                         " = 2 the intermediate lattice never reaches DRAM, so the kernel moves about half of that and frac can"
                         " exceed 1 (temporal blocking, not skipped work: every launch is checked against the oracle in"
                         " tests/). `own_dram_roof` is the fraction against the traffic this kernel cannot avoid.")
                if spl > 1.5 else "one step per launch: algorithmic bytes = compulsory DRAM traffic",
                "own_dram_roof": {"compulsory_bytes_per_launch": compulsory, "compulsory_gbs": own_gbs,
                                  "frac_of_own_dram_roof": own_gbs / peak,
                                  "roof_mlups": peak * 1e9 / (BYTES_PER_SITE / spl) / 1e6},
                "traffic": traffic, "traffic_source": traffic_source,
                "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum per launch from the named ncu capture of this"
                                " workload and launch plan; not measured in this run (null if no capture matches)",
                # the other candidate roof (north_star): FP64, with the flops counted from the oracle and, for
                # comparison, the flops the kernel really issues.  Peak = the vector-FP64 rate a DFMA-chain probe
                # reaches on this GPU in this process.
                "fp64": {"peak_tflops": fp64_peak, "peak_kind": "measured: lbm_fp64_peak (8 DFMA chains/thread, all SMs)",
                         "flops_per_site_step_oracle": FLOPS_PER_SITE_ORACLE,
                         "roof_mlups_oracle_count": fp64_peak * 1e12 / FLOPS_PER_SITE_ORACLE / 1e6,
                         "flops_per_site_step_kernel": FLOPS_PER_SITE,
                         "roof_mlups_kernel_count": fp64_peak * 1e12 / FLOPS_PER_SITE / 1e6,
                         "achieved_tflops_kernel_count": FLOPS_PER_SITE * rate / 1e12,
                         "frac_kernel_count": FLOPS_PER_SITE * rate / 1e12 / fp64_peak},
                "binding_roof": {"hbm_mlups": peak * 1e9 / BYTES_PER_SITE / 1e6,
                                 "fp64_mlups_oracle_count": fp64_peak * 1e12 / FLOPS_PER_SITE_ORACLE / 1e6,
                                 "which": "hbm" if peak * 1e9 / BYTES_PER_SITE < fp64_peak * 1e12 / FLOPS_PER_SITE_ORACLE else "fp64",
                                 "kernel_mlups": rate / 1e6}}
    cpu = None
    if not args.no_cpu_baseline:
        v, cores, sample = oracle_sample_rate(cfg, args.cpu_budget)
        v1, _, sample1 = oracle_sample_rate(cfg, min(args.cpu_budget, 6.0), threads=1)
        cpu = {"value": v, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample,
               "single_thread": {"value": v1, "unit": "MLUPS", "cores": 1, "sample": sample1},
               "named_samples": oracle_named_samples()}
    print(json.dumps({
        "metric": "MLUPS (FP64)", "value": value, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_total / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "Lx": cfg.Lx, "Lz": cfg.Lz, "tau": cfg.tau, "g": cfg.g,
                   "parallelism": "replicas only" if world > 1 else "single GPU, whole lattice resident",
                   "l2": "inputs larger than L2 (2 x 37 planes, %.1f GB)" % (2 * 37 * 8 * sites / 1e9),
                   "variant": args.variant, "wall_kind": args.wall_kind, "widths_calls_in_timed_region": 1,
                   "L_u": widths[0], "L_d": widths[1]},
        "sustained": sustained,
        "roofline": roofline, "roofline_a6": a6, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
    }))
    if world > 1:
        dist.destroy_process_group()


def run_slabs(args):
    """--slabs under torchrun (N > 1): ONE lattice (the N = 1 workload) cut into z-slabs, one per rank, ghost rows
    exchanged over NCCL point-to-point calls (SlabRing: 6 whole rows per pair of steps for the two-step kernel; 26
    population-rows per step, hidden behind the interior rows, for an odd step -- SURVEY 8(f)4; PAPER.md:110,
    116-118).  Strong scaling: value = sites x steps / max-over-ranks time.  Not the default N > 1 mode
    (north_star fixes one GPU: the default is independent replicas); unmeasured on hardware in this run (one GPU per
    call), verified on one GPU by tests/test_gpu_variants.py (slabs on one device, bit-identical to the whole lattice)."""
    import torch
    import torch.distributed as dist

    import __graft_entry__ as entry
    from paper_1405_1253_b200.slab_ring import SlabRing

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if world < 2:
        raise SystemExit("bench.py --slabs needs torchrun with N > 1 ranks")
    # --backend gloo: the ranks may share GPUs (messages staged through pinned host memory): runs the whole schedule on
    # a one-GPU box; the number it prints is a smoke value, not a scaling measurement
    local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    if args.backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    else:
        dist.init_process_group(args.backend)
    red_dev = "cuda" if args.backend == "nccl" else "cpu"
    if rank == 0:
        entry.build()
    dist.barrier()
    cfg = si.rt_config(args.config)
    ring = SlabRing(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, rank, world, wall_kind=args.wall_kind, T_wall=(cfg.T_d, cfg.T_u))
    ring.slab.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize(); dist.barrier(); torch.cuda.synchronize()

    ring.step(args.warmup)
    barrier()
    sampler = ClockSampler(local); sampler.start()
    l0 = ring.slab.kernel_launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream); ring.step(args.steps); e1.record(stream)
    barrier()
    clocks = sampler.finish()
    t = reduce_max([e0.elapsed_time(e1) * 1e-3], world, red_dev)[0]
    part = ring.slab.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u, want_tbar=False)
    w = torch.tensor([part[0], part[1]], dtype=torch.float64, device=red_dev)
    dist.all_reduce(w)                                           # the widths of eq. 12 are sums over rows
    launches = ring.slab.kernel_launches - l0
    if rank == 0:
        sites = cfg.Lx * cfg.Lz
        print(json.dumps({
            "metric": "MLUPS (FP64)", "value": sites * args.steps / t / 1e6, "unit": "MLUPS", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "Lx": cfg.Lx, "Lz": cfg.Lz, "tau": cfg.tau, "g": cfg.g,
                       "parallelism": f"{world} z-slabs; pairs of steps with the two-step kernel (6 whole ghost rows per open "
                                      "side and pair), an odd step with the one-step kernel (26 population-rows); interior rows first, "
                                      "the exchange behind them",
                       "backend": args.backend, "wall_kind": args.wall_kind,
                       "message2_bytes": 6 * 37 * (cfg.Lx + 16) * 8, "message_bytes": 26 * cfg.Lx * 8,
                       "L_u": float(w[0]), "L_d": float(w[1])},
            "gpu_launches": launches, "clocks": clocks}))
    ring.close()
    dist.destroy_process_group()


def run_slabs_local(args):
    """--slabs-local K: the N = 1 workload cut into K z-slabs that all live on THIS device, ghost rows exchanged every
    step by device-to-device copies on a second stream while the interior rows run (the machinery of --slabs without the
    network): measures what packing, unpacking and the interior/edge split cost against the whole lattice stepped with
    the same one-step kernel.  Prints one JSON line; not the driver's contract line."""
    import torch

    import __graft_entry__ as entry
    import paper_1405_1253_b200 as pkg
    from paper_1405_1253_b200.slab_ring import partition
    entry.build()
    torch.cuda.set_device(0)
    cfg = si.rt_config(args.config)
    if args.lx and args.lz:
        cfg = si.scaled(cfg, args.lx, args.lz)
    main = torch.cuda.current_stream()
    xs = torch.cuda.Stream()
    K = args.slabs_local

    def timed(fn):
        fn(args.warmup)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(main); fn(args.steps); e1.record(main)
        torch.cuda.synchronize()
        return cfg.Lx * cfg.Lz * args.steps / (e0.elapsed_time(e1) * 1e-3) / 1e6

    whole = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    whole.set_variant(1)
    whole.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    mlups_whole = timed(whole.step)
    whole.close()
    del whole
    torch.cuda.empty_cache()
    slabs = [pkg.Slab(cfg.Lx, cfg.Lz, z0, nz, cfg.tau, cfg.g) for z0, nz in partition(cfg.Lz, K)]
    for s in slabs:
        s.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    up, dn, below, above = ([s.new_message() for s in slabs] for _ in range(4))

    def step_slabs(n):
        for _ in range(n):
            xs.wait_stream(main)
            with torch.cuda.stream(xs):
                for i, s in enumerate(slabs):
                    if s.open_above: s.pack(1, up[i], stream=xs)
                    if s.open_below: s.pack(0, dn[i], stream=xs)
            for s in slabs:
                s.step_part(s.INTERIOR, stream=main)
            with torch.cuda.stream(xs):
                for i, s in enumerate(slabs):
                    if s.open_below: below[i].copy_(up[i - 1], non_blocking=True); s.unpack(0, below[i], stream=xs)
                    if s.open_above: above[i].copy_(dn[i + 1], non_blocking=True); s.unpack(1, above[i], stream=xs)
            main.wait_stream(xs)
            for s in slabs:
                s.step_part(s.EDGES, stream=main)

    mlups_slabs = timed(step_slabs)

    # the same slabs with the two-step kernel: 6 whole ghost rows per open side and pair of steps, interior rows first
    up2, dn2, below2, above2 = ([s.new_message(True) for s in slabs] for _ in range(4))

    def step_slabs_fused(n):
        for _ in range(n // 2):
            xs.wait_stream(main)
            for i, s in enumerate(slabs):
                if s.open_above: s.pack2(1, up2[i], stream=xs)
                if s.open_below: s.pack2(0, dn2[i], stream=xs)
            main.wait_stream(xs)
            for s in slabs:
                s.step2_part(s.INTERIOR, stream=main)
            with torch.cuda.stream(xs):
                for i, s in enumerate(slabs):
                    if s.open_below: below2[i].copy_(up2[i - 1], non_blocking=True); s.unpack2(0, below2[i], stream=xs)
                    if s.open_above: above2[i].copy_(dn2[i + 1], non_blocking=True); s.unpack2(1, above2[i], stream=xs)
            main.wait_stream(xs)
            for s in slabs:
                s.step2_part(s.EDGES, stream=main)

    mlups_fused = timed(step_slabs_fused)
    mlups_whole2 = None
    if torch.cuda.mem_get_info()[0] > 2.2 * pkg.buffer_bytes(cfg.Lx, cfg.Lz):      # room for the whole lattice beside the slabs
        whole2 = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
        whole2.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
        mlups_whole2 = timed(whole2.step)
        whole2.close()
    print(json.dumps({"slabs_local": K, "workload": cfg.name, "Lx": cfg.Lx, "Lz": cfg.Lz, "steps": args.steps,
                      "mlups_whole_lattice_one_step_kernel": mlups_whole, "mlups_slabs": mlups_slabs,
                      "mlups_whole_lattice_default_plan": mlups_whole2, "mlups_slabs_two_step_kernel": mlups_fused,
                      "message2_bytes": 6 * 37 * (cfg.Lx + 16) * 8,
                      "ratio": mlups_slabs / mlups_whole, "message_bytes": 26 * cfg.Lx * 8,
                      "launches_per_step": sum(2 * (s.open_above + s.open_below) + 1 + (s.open_above + s.open_below) for s in slabs)}))
    for s in slabs:
        s.close()


def run_sweep(args):
    """--sweep: BASELINE.json configs[4] -- steady-state throughput from 256x512 to 8192x16384, populations at
    the equilibrium of i.i.d. rho, T, u fields; 200 timed steps per size (after 10 warm-up), one JSON line per
    (size, variant) with MLUPS, algorithmic GB/s and the moments kernel's rate.  Not the driver's contract line."""
    import torch

    import __graft_entry__ as entry
    import paper_1405_1253_b200 as pkg
    entry.build()
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    peak, _ = measured_peak()
    variants = [int(v) for v in args.sweep_variants.split(",")]
    sizes = [tuple(int(x) for x in sz.split("x")) for sz in args.sweep_sizes.split(",")] if args.sweep_sizes \
        else si.SWEEP_SIZES
    for Lx, Lz in sizes:
        sites = Lx * Lz
        fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
        lat = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G, inplace=args.inplace)
        for v in variants:
            lat.set_variant(v)
            if args.zchunk:
                lat.set_zchunk(args.zchunk)
            lat.init_equilibrium(*fields)
            lat.step(args.warmup)
            torch.cuda.synchronize()
            e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
            e0.record(stream); lat.step(args.steps); e1.record(stream)
            lat.moments(*fields); e2.record(stream)            # overwrites the input fields: re-drawn per size
            torch.cuda.synchronize()
            t = e0.elapsed_time(e1) * 1e-3 / args.steps
            tm = e1.elapsed_time(e2) * 1e-3
            tot = lat.totals()
            print(json.dumps({"sweep": f"{Lx}x{Lz}", "variant": v, "inplace": args.inplace, "plan": lat.plan(), "zchunk": args.zchunk, "mlups": sites / t / 1e6, "us_per_step": t * 1e6,
                              "gbs": BYTES_PER_SITE * sites / t / 1e9, "frac_of_measured_peak": BYTES_PER_SITE * sites / t / 1e9 / peak,
                              "resident": "L2" if 2 * 37 * 8 * sites < 126e6 else "HBM",
                              "moments_gbs": 328 * sites / tm / 1e9, "mass": tot[0]}), flush=True)
            fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
        lat.close()
        del fields, lat
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="RT config 1..4 of BASELINE.json (default 4: 4096x8192)")
    ap.add_argument("--lx", type=int, default=0)
    ap.add_argument("--lz", type=int, default=0)
    ap.add_argument("--variant", type=int, default=None, help="step-kernel variant (default: library default)")
    ap.add_argument("--wall-kind", type=int, default=0, choices=[0, 1], help="0 bounce-back walls (default), 1 isothermal no-slip walls")
    ap.add_argument("--zchunk", type=int, default=0, help="rows per block of the two-step kernel (multiple of 3)")
    ap.add_argument("--e2e-steps", type=int, default=0)
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle time for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sustain", type=float, default=3.0,
                    help="seconds of the extra sustained-throughput leg after the timed region (0 = skip)")
    ap.add_argument("--sweep", action="store_true", help="config 5: throughput sweep over lattice sizes")
    ap.add_argument("--sweep-variants", default="0")
    ap.add_argument("--inplace", action="store_true", help="sweep with ONE lattice copy (in-place streaming)")
    ap.add_argument("--slabs", action="store_true", help="N > 1: one lattice cut into z-slabs over the ranks (strong scaling)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"], help="--slabs transport (gloo: ranks may share a GPU)")
    ap.add_argument("--slabs-local", type=int, default=0, help="K z-slabs on this one device (cost of the slab machinery)")
    ap.add_argument("--sweep-sizes", default="", help="e.g. 256x512,4096x8192 (default: all of config 5)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.sweep:
        run_sweep(args)
    elif args.slabs:
        run_slabs(args)
    elif args.slabs_local:
        run_slabs_local(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
