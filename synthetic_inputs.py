"""Seeded synthetic workloads shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no velocity set, no equilibrium, no moments):
it only names the five BASELINE.json configurations and draws the random per-site fields of
config 5.  Both the CPU oracle (oracle/) and the CUDA library (paper_1405_1253_b200/) receive
these values as plain inputs; neither imports the other.

The inputs are synthetic stand-ins for the paper's Rayleigh-Taylor runs (Table II,
/root/reference PAPER.md:139-144: 2400x6144 tank, T within +-2.5 % of 1, g = 1.5e-5, white-noise
interface); the recipe is stated in DESIGN.md "Input recipe".
"""
from __future__ import annotations

from dataclasses import dataclass, asdict

import numpy as np

DEFAULT_SEED = 12345

PERT_NONE, PERT_MODES, PERT_WHITE = 0, 1, 2


@dataclass(frozen=True)
class RTConfig:
    """One Rayleigh-Taylor workload: lattice, model parameters and lbm_init_rt arguments."""
    name: str
    Lx: int
    Lz: int
    tau: float
    g: float
    T_d: float
    T_m: float
    T_u: float
    rho_m: float
    delta: float
    smooth_w: float
    pert_kind: int
    n_modes: int
    amp_lo: float
    amp_hi: float
    steps: int

    def rt_args(self) -> dict:
        d = asdict(self)
        for k in ("name", "Lx", "Lz", "tau", "g", "steps"):
            d.pop(k)
        return d


def rt_config(idx: int) -> RTConfig:
    """BASELINE.json configs[0..3] (idx 1..4).  idx 4 is the one the headline metric is quoted on."""
    if idx == 1:  # oracle-scale double front, 4 modes of amplitude 1 site
        return RTConfig("rt_double_64x128", 64, 128, 0.8, 1e-4, 1.05, 1.00, 0.95, 1.0, 128 / 4, 2.5,
                        PERT_MODES, 4, 1.0, 1.0, 100)
    if idx == 2:  # 16 modes, amplitudes uniform in [0, 2] sites
        return RTConfig("rt_double_512x1024", 512, 1024, 0.8, 1e-4, 1.05, 1.00, 0.95, 1.0, 1024 / 4, 2.5,
                        PERT_MODES, 16, 0.0, 2.0, 5000)
    if idx == 3:  # white noise +-1 site
        return RTConfig("rt_double_2048x4096", 2048, 4096, 0.7, 5e-5, 1.05, 1.00, 0.95, 1.0, 4096 / 4, 2.5,
                        PERT_WHITE, 0, 0.0, 1.0, 20000)
    if idx == 4:  # classic single front; T_m is the virtual middle temperature
        return RTConfig("rt_single_4096x8192", 4096, 8192, 0.7, 5e-5, 1.02, 1.00, 0.98, 1.0, 0.0, 2.5,
                        PERT_WHITE, 0, 0.0, 1.0, 10000)
    raise ValueError(f"no RT config {idx}")


def scaled(cfg: RTConfig, Lx: int, Lz: int, name: str | None = None) -> RTConfig:
    """Same physics on another lattice (delta keeps its fraction of Lz)."""
    d = asdict(cfg)
    d.update(Lx=Lx, Lz=Lz, delta=cfg.delta * Lz / cfg.Lz, name=name or f"{cfg.name}@{Lx}x{Lz}")
    return RTConfig(**d)


# config 5: throughput sweep, Lx x Lz
SWEEP_SIZES = [(256, 512), (512, 512), (512, 1024), (1024, 1024), (1024, 2048), (2048, 2048), (2048, 4096),
               (4096, 4096), (4096, 8192), (8192, 8192), (8192, 16384)]
SWEEP_TAU, SWEEP_G = 0.8, 1e-4

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64_uniform(seed: int, first: int, count: int) -> np.ndarray:
    """U_n = (n-th output of the SplitMix64 stream seeded with `seed`) >> 11) * 2^-53, n = first..first+count-1.

    SplitMix64 is counter-based (its n-th output is a hash of seed + (n+1)*gamma), so the stream is
    evaluated here in one vectorised pass.
    """
    with np.errstate(over="ignore"):
        n = np.arange(first + 1, first + count + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + n * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def sweep_fields(Lx: int, Lz: int, seed: int = DEFAULT_SEED, rows: slice | None = None):
    """Config-5 kinetic fields rho = 1+-0.01, T = 1+-0.01, u_x, u_z = +-0.01, i.i.d. uniform per site.

    Site s = k*Lx + i consumes draws 4s..4s+3 in the order rho, T, u_x, u_z.  `rows` restricts the
    result to a row range without drawing the rest (used to sample large lattices).
    Returns (rho, ux, uz, T), each [rows][Lx] float64.
    """
    k0, k1, _ = (rows or slice(0, Lz)).indices(Lz)
    n = (k1 - k0) * Lx
    u = splitmix64_uniform(seed, 4 * k0 * Lx, 4 * n).reshape(k1 - k0, Lx, 4)
    rho = 1.0 + 0.01 * (2.0 * u[..., 0] - 1.0)
    T = 1.0 + 0.01 * (2.0 * u[..., 1] - 1.0)
    ux = 0.01 * (2.0 * u[..., 2] - 1.0)
    uz = 0.01 * (2.0 * u[..., 3] - 1.0)
    return (np.ascontiguousarray(rho), np.ascontiguousarray(ux), np.ascontiguousarray(uz),
            np.ascontiguousarray(T))


def _splitmix64_uniform_torch(seed: int, first: int, count: int, device):
    """Same stream as splitmix64_uniform, evaluated with torch int64 arithmetic (wraps mod 2^64) on `device`."""
    import torch

    def s64(v):  # two's-complement view of a uint64 constant
        v &= 0xFFFFFFFFFFFFFFFF
        return v - (1 << 64) if v >= (1 << 63) else v

    def lsr(z, n):  # logical shift right on int64
        return (z >> n) & ((1 << (64 - n)) - 1)

    n = torch.arange(first + 1, first + count + 1, dtype=torch.int64, device=device)
    z = n * s64(0x9E3779B97F4A7C15) + s64(seed)
    z = (z ^ lsr(z, 30)) * s64(0xBF58476D1CE4E5B9)
    z = (z ^ lsr(z, 27)) * s64(0x94D049BB133111EB)
    z = z ^ lsr(z, 31)
    return lsr(z, 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def sweep_fields_torch(Lx: int, Lz: int, seed: int = DEFAULT_SEED, device="cuda", chunk_rows: int = 1024):
    """sweep_fields() produced directly on `device` (bit-identical values), in row chunks to bound memory."""
    import torch
    out = [torch.empty((Lz, Lx), dtype=torch.float64, device=device) for _ in range(4)]
    for k0 in range(0, Lz, chunk_rows):
        k1 = min(Lz, k0 + chunk_rows)
        u = _splitmix64_uniform_torch(seed, 4 * k0 * Lx, 4 * (k1 - k0) * Lx, device).reshape(k1 - k0, Lx, 4)
        out[0][k0:k1] = 1.0 + 0.01 * (2.0 * u[..., 0] - 1.0)      # rho
        out[3][k0:k1] = 1.0 + 0.01 * (2.0 * u[..., 1] - 1.0)      # T
        out[1][k0:k1] = 0.01 * (2.0 * u[..., 2] - 1.0)            # u_x
        out[2][k0:k1] = 0.01 * (2.0 * u[..., 3] - 1.0)            # u_z
    return tuple(out)
