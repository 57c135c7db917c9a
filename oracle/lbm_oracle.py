"""ctypes loader for the CPU oracle (oracle/lbm_oracle.c) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It holds no arithmetic of the method: every function below only marshals
numpy arrays into the plain-C oracle, which is written from PAPER.md (see the header of
lbm_oracle.c for citations and for what pins each function).

Arrays: populations are dense float64 ``[37][Lz][Lx]`` (x fastest), fields ``[Lz][Lx]``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.c")
_LIB = os.path.join(_HERE, "liblbm_oracle.so")
NPOP = 37

_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no fast-math). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_tables.argtypes = [_ip, _ip, _dp, C.POINTER(C.c_double)]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_max_threads.restype = C.c_int
        L.orc_feq.argtypes = [C.c_double] * 4 + [_dp]
        L.orc_site_moments.argtypes = [_dp, _dp]
        L.orc_propagate.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_int, C.c_int]
        L.orc_collide.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double]
        L.orc_step.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int]
        L.orc_bc_isothermal.argtypes = [_dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_step_walls.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double,
                                     C.c_double]
        L.orc_moments.argtypes = [_dp, C.c_int, C.c_int, C.c_double] + [C.c_void_p] * 4
        L.orc_totals.argtypes = [_dp, C.c_int, C.c_int, _dp]
        L.orc_mixing_widths.argtypes = (
            [_dp, C.c_int, C.c_int] + [C.c_double] * 4 + [C.POINTER(C.c_double)] * 2 + [C.c_void_p]
        )
        L.orc_init_equilibrium.argtypes = [_dp, C.c_int, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_interfaces.argtypes = [C.c_uint64, C.c_int, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double, _dp, _dp]
        L.orc_rt_profile.argtypes = [C.c_int, C.c_int] + [C.c_double] * 7 + [_dp, _dp, _dp, _dp]
        L.orc_init_rt.argtypes = (
            [_dp, C.c_int, C.c_int, C.c_double, C.c_uint64]
            + [C.c_double] * 6
            + [C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        )
        L.orc_profiles.argtypes = [_dp, C.c_int, C.c_int, C.c_double] + [C.c_void_p] * 4
        L.orc_growth_rate.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, _dp]
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def tables():
    """(ex[37], ez[37], w[37], r) of the D2Q37 set in canonical order."""
    ex = np.zeros(NPOP, np.int32)
    ez = np.zeros(NPOP, np.int32)
    w = np.zeros(NPOP, np.float64)
    r = C.c_double()
    lib().orc_tables(ex, ez, w, C.byref(r))
    return ex, ez, w, r.value


def feq(rho: float, ux: float, uz: float, T: float) -> np.ndarray:
    out = np.zeros(NPOP)
    lib().orc_feq(rho, ux, uz, T, out)
    return out


def site_moments(fl: np.ndarray):
    out = np.zeros(4)
    lib().orc_site_moments(np.ascontiguousarray(fl, np.float64), out)
    return tuple(out)


def propagate(f: np.ndarray, periodic_z: bool = False, direction: int = 1) -> np.ndarray:
    _, Lz, Lx = f.shape
    out = np.empty_like(f)
    lib().orc_propagate(f, out, Lx, Lz, int(periodic_z), int(direction))
    return out


def collide(fs: np.ndarray, tau: float, g: float) -> np.ndarray:
    _, Lz, Lx = fs.shape
    out = np.empty_like(fs)
    lib().orc_collide(fs, out, Lx, Lz, tau, g)
    return out


def step(f: np.ndarray, tau: float, g: float, nsteps: int = 1, periodic_z: bool = False, wall_kind: int = 0,
         T_bot: float = 1.0, T_top: float = 1.0) -> np.ndarray:
    """Returns the state after nsteps x (propagate, bc, collide); the input is not modified.
    wall_kind 1 = isothermal no-slip walls at T_bot / T_top (orc_step_walls)."""
    _, Lz, Lx = f.shape
    cur = np.array(f, dtype=np.float64, order="C", copy=True)
    tmp = np.empty_like(cur)
    if wall_kind == 0:
        lib().orc_step(cur, tmp, Lx, Lz, tau, g, int(nsteps), int(periodic_z))
    else:
        assert not periodic_z
        lib().orc_step_walls(cur, tmp, Lx, Lz, tau, g, int(nsteps), int(wall_kind), T_bot, T_top)
    return cur


def bc_isothermal(fs: np.ndarray, g: float, T_bot: float, T_top: float) -> np.ndarray:
    """The wall adjustment of reading 19 applied to post-propagate populations (returns a copy)."""
    _, Lz, Lx = fs.shape
    out = np.array(fs, dtype=np.float64, order="C", copy=True)
    lib().orc_bc_isothermal(out, Lx, Lz, g, T_bot, T_top)
    return out


def moments(f: np.ndarray, g: float):
    """Hydrodynamic rho, u_x^(H), u_z^(H), T^(H) of the stored state, each [Lz][Lx]."""
    _, Lz, Lx = f.shape
    outs = [np.empty((Lz, Lx)) for _ in range(4)]
    lib().orc_moments(f, Lx, Lz, g, *[o.ctypes.data for o in outs])
    return tuple(outs)


def totals(f: np.ndarray) -> np.ndarray:
    _, Lz, Lx = f.shape
    out = np.zeros(4)
    lib().orc_totals(f, Lx, Lz, out)
    return out


def mixing_widths(f: np.ndarray, g: float, T_d: float, T_m: float, T_u: float):
    """(L_u, L_d, Tbar[Lz]) per eq. 12 on the x-averaged T^(H)."""
    _, Lz, Lx = f.shape
    lu, ld = C.c_double(), C.c_double()
    tbar = np.empty(Lz)
    lib().orc_mixing_widths(f, Lx, Lz, g, T_d, T_m, T_u, C.byref(lu), C.byref(ld), tbar.ctypes.data)
    return lu.value, ld.value, tbar


def init_equilibrium(rho, ux, uz, T) -> np.ndarray:
    Lz, Lx = rho.shape
    f = np.empty((NPOP, Lz, Lx))
    a = [np.ascontiguousarray(x, np.float64) for x in (rho, ux, uz, T)]
    lib().orc_init_equilibrium(f, Lx, Lz, *a)
    return f


def interfaces(seed: int, Lx: int, delta: float, pert_kind: int, n_modes: int, amp_lo: float, amp_hi: float):
    h_lo, h_hi = np.empty(Lx), np.empty(Lx)
    lib().orc_interfaces(seed, Lx, delta, pert_kind, n_modes, amp_lo, amp_hi, h_lo, h_hi)
    return h_lo, h_hi


def rt_profile(Lx, Lz, g, T_d, T_m, T_u, rho_m, delta, w, h_lo, h_hi):
    rho0, T0 = np.empty((Lz, Lx)), np.empty((Lz, Lx))
    lib().orc_rt_profile(Lx, Lz, g, T_d, T_m, T_u, rho_m, delta, w,
                         np.ascontiguousarray(h_lo, np.float64), np.ascontiguousarray(h_hi, np.float64), rho0, T0)
    return rho0, T0


def init_rt(Lx, Lz, g, seed, T_d, T_m, T_u, rho_m=1.0, delta=0.0, smooth_w=2.5, pert_kind=0, n_modes=0,
            amp_lo=0.0, amp_hi=0.0, return_fields=False):
    f = np.empty((NPOP, Lz, Lx))
    rho0 = np.empty((Lz, Lx)) if return_fields else None
    T0 = np.empty((Lz, Lx)) if return_fields else None
    lib().orc_init_rt(f, Lx, Lz, g, seed, T_d, T_m, T_u, rho_m, delta, smooth_w, pert_kind, n_modes, amp_lo,
                      amp_hi, rho0.ctypes.data if return_fields else None, T0.ctypes.data if return_fields else None)
    return (f, rho0, T0) if return_fields else f


def profiles(f: np.ndarray, g: float):
    """(Tbar, Trms, Ekbar, Ekrms), each [Lz]: x-means and x-fluctuations of T^(H) and E_k = rho |u^(H)|^2 / 2."""
    _, Lz, Lx = f.shape
    outs = [np.empty(Lz) for _ in range(4)]
    lib().orc_profiles(f, Lx, Lz, g, *[o.ctypes.data for o in outs])
    return tuple(outs)


def growth_rate(t, L, g: float, At: float) -> np.ndarray:
    """alpha(t_j) = (dL/dt)^2 / (4 g At L), eq. 11 / 14."""
    t = np.ascontiguousarray(t, np.float64)
    L = np.ascontiguousarray(L, np.float64)
    out = np.empty(len(t))
    lib().orc_growth_rate(len(t), t, L, g, At, out)
    return out
