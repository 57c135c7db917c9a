"""Thin ctypes binding of liblbm_b200.so (include/lbm.h): argument marshalling only.

PyTorch supplies device memory and streams; every arithmetic step runs in the CUDA kernels of csrc/.
There is no CPU fallback: importing works without a GPU (so the CPU test tier can check the exported
symbols), but any compute call without the library or a device raises.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblbm_b200.so")
NPOP = 37
NOALLOC_MAX_ROWS = 16384   # LBM_NOALLOC_MAX_ROWS of include/lbm.h

# every symbol include/lbm.h declares
SYMBOLS = [
    "lbm_buffer_bytes", "lbm_create", "lbm_destroy", "lbm_init_rt", "lbm_init_equilibrium",
    "lbm_set_populations", "lbm_get_populations", "lbm_set_populations_host", "lbm_get_populations_host",
    "lbm_step", "lbm_moments", "lbm_mixing_widths", "lbm_profiles", "lbm_growth_rate", "lbm_totals", "lbm_run_host", "lbm_steps_done",
    "lbm_layout", "lbm_kernel_launches", "lbm_fp64_peak", "lbm_set_variant", "lbm_set_zchunk", "lbm_get_plan", "lbm_tables", "lbm_last_error",
    "lbm_diagnostics", "lbm_rt_scales", "lbm_slab_buffer_bytes", "lbm_create_slab", "lbm_slab_info", "lbm_slab_pack",
    "lbm_slab_unpack", "lbm_slab_step", "lbm_get_window", "lbm_slab_pack2", "lbm_slab_unpack2", "lbm_slab_step2",
    "lbm_diagnostics_noalloc", "lbm_kinetic_moments", "lbm_slab_step2_part",
]


class LbmError(RuntimeError):
    pass


class lbm_params(C.Structure):
    _fields_ = [("tau", C.c_double), ("g", C.c_double), ("wall_kind", C.c_int), ("pop_buf0", C.c_void_p),
                ("pop_buf1", C.c_void_p), ("buf_bytes", C.c_size_t), ("T_wall_bottom", C.c_double),
                ("T_wall_top", C.c_double)]


class lbm_rt_init(C.Structure):
    _fields_ = [("T_d", C.c_double), ("T_m", C.c_double), ("T_u", C.c_double), ("rho_m", C.c_double),
                ("delta", C.c_double), ("smooth_w", C.c_double), ("pert_kind", C.c_int), ("n_modes", C.c_int),
                ("amp_lo", C.c_double), ("amp_hi", C.c_double)]


_lib = None


def load():
    """Loads the shared library; raises LbmError if it has not been built (run __graft_entry__.build())."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise LbmError(f"{LIB_PATH} is missing: build it with `python -c 'import __graft_entry__ as g; g.build()'`"
                       " (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    L.lbm_last_error.restype = C.c_char_p
    L.lbm_buffer_bytes.restype = C.c_size_t
    L.lbm_buffer_bytes.argtypes = [C.c_int, C.c_int]
    L.lbm_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.POINTER(lbm_params)]
    L.lbm_destroy.argtypes = [vp]
    L.lbm_init_rt.argtypes = [vp, C.c_uint64, C.POINTER(lbm_rt_init), vp]
    L.lbm_init_equilibrium.argtypes = [vp, vp, vp, vp, vp, vp]
    for name in ("lbm_set_populations", "lbm_get_populations", "lbm_set_populations_host", "lbm_get_populations_host"):
        getattr(L, name).argtypes = [vp, vp, vp]
    L.lbm_step.argtypes = [vp, C.c_int, vp]
    L.lbm_moments.argtypes = [vp, vp, vp, vp, vp, vp]
    L.lbm_kinetic_moments.argtypes = [vp, vp, vp, vp, vp, vp]
    L.lbm_mixing_widths.argtypes = [vp, C.c_double, C.c_double, C.c_double, dp, dp, vp, vp]
    L.lbm_profiles.argtypes = [vp, vp, vp, vp, vp, vp]
    L.lbm_growth_rate.argtypes = [C.c_int, vp, vp, C.c_double, C.c_double, vp]
    L.lbm_totals.argtypes = [vp, dp, vp]
    L.lbm_run_host.argtypes = [vp, vp, vp, vp, vp, C.c_int, vp, vp, vp, vp, vp]
    L.lbm_steps_done.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.lbm_layout.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_longlong)]
    L.lbm_kernel_launches.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.lbm_fp64_peak.argtypes = [dp, C.c_int, vp]
    L.lbm_set_variant.argtypes = [vp, C.c_int]
    L.lbm_set_zchunk.argtypes = [vp, C.c_int]
    L.lbm_get_plan.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.lbm_tables.argtypes = [C.POINTER(C.c_int), C.POINTER(C.c_int), dp, dp]
    L.lbm_diagnostics.argtypes = [vp, C.c_double, C.c_double, C.c_double, vp, vp, vp, vp, vp, vp, vp]
    L.lbm_rt_scales.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, dp, dp]
    L.lbm_slab_buffer_bytes.restype = C.c_size_t
    L.lbm_slab_buffer_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int]
    L.lbm_create_slab.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(lbm_params)]
    L.lbm_slab_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int),
                                C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    L.lbm_slab_pack2.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_slab_unpack2.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_slab_step2.argtypes = [vp, vp]
    L.lbm_slab_step2_part.argtypes = [vp, C.c_int, vp]
    L.lbm_slab_pack.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_slab_unpack.argtypes = [vp, C.c_int, vp, vp]
    L.lbm_slab_step.argtypes = [vp, C.c_int, vp]
    L.lbm_get_window.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp]
    L.lbm_diagnostics_noalloc.argtypes = [vp, C.c_size_t, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                          vp, vp, vp]
    for name in SYMBOLS:
        if name not in ("lbm_buffer_bytes", "lbm_slab_buffer_bytes", "lbm_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def check(rc: int) -> None:
    if rc != 0:
        raise LbmError(f"lbm error {rc}: {load().lbm_last_error().decode()}")
