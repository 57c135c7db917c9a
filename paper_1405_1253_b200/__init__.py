"""paper_1405_1253_b200 -- B200-native thermal D2Q37 Lattice-Boltzmann step (arxiv/paper_1405_1253).

`Lattice` mirrors the C ABI of include/lbm.h call for call (lbm_create / lbm_init_rt / lbm_step /
lbm_moments / ...).  It only marshals arguments: device memory and streams come from PyTorch, every
step of the path runs in the hand-written CUDA kernels of csrc/ (liblbm_b200.so).  No CPU fallback.
"""
from __future__ import annotations

import ctypes as C

from . import binding
from .binding import LbmError, NPOP, lbm_params, lbm_rt_init

__all__ = ["Lattice", "LbmError", "NPOP", "buffer_bytes", "tables", "growth_rate"]


def buffer_bytes(Lx: int, Lz: int) -> int:
    return int(binding.load().lbm_buffer_bytes(Lx, Lz))


def tables():
    """(e_x[37], e_z[37], w[37], r) as the CUDA library uses them."""
    ex, ez, w, r = (C.c_int * NPOP)(), (C.c_int * NPOP)(), (C.c_double * NPOP)(), C.c_double()
    binding.check(binding.load().lbm_tables(ex, ez, w, C.byref(r)))
    return list(ex), list(ez), list(w), r.value


def growth_rate(t, L, g: float, At: float):
    """alpha(t_j) of eq. 11 / 14 from a logged mixing length (lbm_growth_rate; host-only)."""
    import numpy as np
    t = np.ascontiguousarray(t, np.float64)
    L = np.ascontiguousarray(L, np.float64)
    out = np.empty(len(t))
    binding.check(binding.load().lbm_growth_rate(len(t), t.ctypes.data, L.ctypes.data, g, At, out.ctypes.data))
    return out


def fp64_peak(iters: int = 0, stream=None) -> float:
    """Vector-FP64 rate of this GPU in TFLOP/s from a DFMA-chain probe (lbm_fp64_peak; measurement aid)."""
    out = C.c_double(0.0)
    binding.check(binding.load().lbm_fp64_peak(C.byref(out), int(iters), _stream_ptr(stream)))
    return out.value


def _stream_ptr(stream):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class Lattice:
    """One Lx x Lz lattice resident on the current CUDA device (lbm_create)."""

    def __init__(self, Lx: int, Lz: int, tau: float, g: float, wall_kind: int = 0, device="cuda"):
        import torch
        self._lib = binding.load()
        if not torch.cuda.is_available():
            raise LbmError("no CUDA device: the lattice update has no CPU fallback")
        self.Lx, self.Lz, self.tau, self.g = int(Lx), int(Lz), float(tau), float(g)
        self.device = torch.device(device)
        nbytes = buffer_bytes(Lx, Lz)
        if nbytes == 0:
            raise LbmError(f"invalid lattice {Lx} x {Lz}")
        # the two lattice copies (prv / nxt): torch owns the memory, the library only uses it
        self._bufs = [torch.empty(nbytes // 8, dtype=torch.float64, device=self.device) for _ in range(2)]
        p = lbm_params(tau, g, wall_kind, self._bufs[0].data_ptr(), self._bufs[1].data_ptr(), nbytes)
        h = C.c_void_p()
        binding.check(self._lib.lbm_create(C.byref(h), Lx, Lz, C.byref(p)))
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.lbm_destroy(self._h)
            self._h = None
            self._bufs = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- initial states
    def init_rt(self, seed: int, T_d, T_m, T_u, rho_m=1.0, delta=0.0, smooth_w=2.5, pert_kind=0, n_modes=0,
                amp_lo=0.0, amp_hi=0.0, stream=None):
        ic = lbm_rt_init(T_d, T_m, T_u, rho_m, delta, smooth_w, pert_kind, n_modes, amp_lo, amp_hi)
        binding.check(self._lib.lbm_init_rt(self._h, C.c_uint64(seed), C.byref(ic), _stream_ptr(stream)))

    def init_equilibrium(self, rho, ux, uz, T, stream=None):
        self._check_fields(rho, ux, uz, T)
        binding.check(self._lib.lbm_init_equilibrium(self._h, _dptr(rho), _dptr(ux), _dptr(uz), _dptr(T),
                                                     _stream_ptr(stream)))

    # ---- populations, canonical dense [37][Lz][Lx]
    def set_populations(self, f, stream=None):
        self._check_pops(f)
        fn = self._lib.lbm_set_populations if f.is_cuda else self._lib.lbm_set_populations_host
        binding.check(fn(self._h, _dptr(f), _stream_ptr(stream)))

    def get_populations(self, out=None, host=False, stream=None):
        import torch
        if out is None:
            out = torch.empty((NPOP, self.Lz, self.Lx), dtype=torch.float64, device="cpu" if host else self.device)
        self._check_pops(out)
        fn = self._lib.lbm_get_populations if out.is_cuda else self._lib.lbm_get_populations_host
        binding.check(fn(self._h, _dptr(out), _stream_ptr(stream)))
        return out

    # ---- the hot path
    def step(self, n: int = 1, stream=None):
        binding.check(self._lib.lbm_step(self._h, int(n), _stream_ptr(stream)))

    # ---- diagnostics
    def moments(self, rho=None, ux=None, uz=None, T=None, stream=None, alloc=True):
        import torch
        if alloc and rho is None and ux is None and uz is None and T is None:
            rho, ux, uz, T = (torch.empty((self.Lz, self.Lx), dtype=torch.float64, device=self.device) for _ in range(4))
        self._check_fields(*[x for x in (rho, ux, uz, T) if x is not None])
        binding.check(self._lib.lbm_moments(self._h, _dptr(rho), _dptr(ux), _dptr(uz), _dptr(T), _stream_ptr(stream)))
        return rho, ux, uz, T

    def mixing_widths(self, T_d, T_m, T_u, want_tbar=True, stream=None):
        import numpy as np
        lu, ld = C.c_double(), C.c_double()
        tbar = np.empty(self.Lz) if want_tbar else None
        binding.check(self._lib.lbm_mixing_widths(self._h, T_d, T_m, T_u, C.byref(lu), C.byref(ld),
                                                  tbar.ctypes.data if want_tbar else None, _stream_ptr(stream)))
        return lu.value, ld.value, tbar

    def profiles(self, stream=None):
        """(Tbar, Trms, Ekbar, Ekrms), host numpy arrays [Lz] (lbm_profiles)."""
        import numpy as np
        outs = [np.empty(self.Lz) for _ in range(4)]
        binding.check(self._lib.lbm_profiles(self._h, *[o.ctypes.data for o in outs], _stream_ptr(stream)))
        return tuple(outs)

    def totals(self, stream=None):
        import numpy as np
        out = (C.c_double * 4)()
        binding.check(self._lib.lbm_totals(self._h, out, _stream_ptr(stream)))
        return np.array(list(out))

    def run_host(self, rho, ux, uz, T, n, outs=None, stream=None):
        """lbm_run_host: HOST (ideally pinned) kinetic fields in, n steps, HOST hydrodynamic fields out."""
        import torch
        ins = (rho, ux, uz, T)
        for x in ins:
            if x.is_cuda or x.dtype != torch.float64 or not x.is_contiguous() or tuple(x.shape) != (self.Lz, self.Lx):
                raise LbmError("run_host wants contiguous float64 host tensors [Lz][Lx]")
        if outs is None:
            outs = tuple(torch.empty((self.Lz, self.Lx), dtype=torch.float64).pin_memory() for _ in range(4))
        binding.check(self._lib.lbm_run_host(self._h, *[_dptr(x) for x in ins], int(n), *[_dptr(x) for x in outs],
                                             _stream_ptr(stream)))
        return outs

    # ---- introspection
    @property
    def steps_done(self) -> int:
        v = C.c_longlong()
        binding.check(self._lib.lbm_steps_done(self._h, C.byref(v)))
        return v.value

    @property
    def kernel_launches(self) -> int:
        v = C.c_longlong()
        binding.check(self._lib.lbm_kernel_launches(self._h, C.byref(v)))
        return v.value

    def layout(self):
        p, s = C.c_int(), C.c_longlong()
        binding.check(self._lib.lbm_layout(self._h, C.byref(p), C.byref(s)))
        return p.value, s.value

    def set_variant(self, variant: int):
        binding.check(self._lib.lbm_set_variant(self._h, int(variant)))

    def set_zchunk(self, rows: int):
        binding.check(self._lib.lbm_set_zchunk(self._h, int(rows)))

    # ---- argument checks (marshalling only)
    def _check_fields(self, *fields):
        import torch
        for x in fields:
            if not x.is_cuda or x.dtype != torch.float64 or not x.is_contiguous() or x.numel() != self.Lx * self.Lz:
                raise LbmError("fields must be contiguous float64 CUDA tensors [Lz][Lx]")

    def _check_pops(self, f):
        import torch
        if f.dtype != torch.float64 or not f.is_contiguous() or f.numel() != NPOP * self.Lx * self.Lz:
            raise LbmError("populations must be a contiguous float64 tensor [37][Lz][Lx]")
