"""paper_1405_1253_b200 -- B200-native thermal D2Q37 Lattice-Boltzmann step (arxiv/paper_1405_1253).

`Lattice` mirrors the C ABI of include/lbm.h call for call (lbm_create / lbm_init_rt / lbm_step /
lbm_moments / ...).  It only marshals arguments: device memory and streams come from PyTorch, every
step of the path runs in the hand-written CUDA kernels of csrc/ (liblbm_b200.so).  No CPU fallback.
"""
from __future__ import annotations

import ctypes as C

from . import binding
from .binding import LbmError, NPOP, lbm_params, lbm_rt_init

__all__ = ["Lattice", "Slab", "LbmError", "NPOP", "buffer_bytes", "slab_buffer_bytes", "tables", "growth_rate",
           "rt_scales", "fp64_peak", "diagnostics_noalloc"]


def buffer_bytes(Lx: int, Lz: int) -> int:
    return int(binding.load().lbm_buffer_bytes(Lx, Lz))


def slab_buffer_bytes(Lx: int, Lz_global: int, z0: int, nz: int) -> int:
    return int(binding.load().lbm_slab_buffer_bytes(Lx, Lz_global, z0, nz))


def rt_scales(Lx: float, g: float, T_d: float, T_u: float):
    """(At, tau_RT) of a Rayleigh-Taylor run (lbm_rt_scales: Table II / PAPER.md:126 arithmetic, in the library)."""
    at, tr = C.c_double(), C.c_double()
    binding.check(binding.load().lbm_rt_scales(Lx, g, T_d, T_u, C.byref(at), C.byref(tr)))
    return at.value, tr.value


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


def _stream_ptr(stream, device=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream(device)
    return C.c_void_p(s.cuda_stream)


def diagnostics_noalloc(pop_buf, Lx: int, Lz: int, g: float, T_d: float, T_m: float, T_u: float, result6, Tbar=None,
                        stream=None):
    """lbm_diagnostics_noalloc: mixing widths, lattice totals and Tbar of a lattice copy, for callers that must not
    allocate device memory (their memory comes from a pool that cudaMalloc would bypass, or they run inside another
    code's time loop, which a cudaMalloc would stall).  Nothing is allocated here either: `pop_buf` is the float64 CUDA
    tensor that holds the lattice copy (what lbm_create was given), `result6` a float64 CUDA tensor of 6 entries
    (L_u, L_d, sum f, sum c_x f, sum c_z f, sum |c|^2 f) and `Tbar` an optional one of Lz entries, all owned by the
    caller.  The scratch is a 1 MiB static array inside the library, shared by every call on that GPU: Lz may be at
    most binding.NOALLOC_MAX_ROWS, and calls that can overlap on the GPU (different streams) race.  Asynchronous."""
    import torch
    for t, n, name in ((result6, 6, "result6"), (Tbar, Lz, "Tbar")):
        if t is not None and (not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() < n
                              or t.device != pop_buf.device):
            raise LbmError(f"{name} must be a contiguous float64 CUDA tensor of at least {n} entries on the lattice's device")
    with torch.cuda.device(pop_buf.device):
        binding.check(binding.load().lbm_diagnostics_noalloc(
            _dptr(pop_buf), pop_buf.numel() * pop_buf.element_size(), int(Lx), int(Lz), float(g), float(T_d), float(T_m),
            float(T_u), _dptr(result6), _dptr(Tbar), _stream_ptr(stream, pop_buf.device)))


def _on_device(method):
    """Runs a Lattice method with the lattice's device current (lbm_create binds the handle to the current device,
    and every lbm_* call checks it)."""
    import functools

    @functools.wraps(method)
    def wrapper(self, *args, **kwargs):
        import torch
        with torch.cuda.device(self.device):
            return method(self, *args, **kwargs)
    return wrapper


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


class Lattice:
    """One Lx x Lz lattice resident on a CUDA device (lbm_create).  wall_kind 1: isothermal no-slip walls at
    T_wall = (bottom, top).  inplace = True: one lattice copy instead of two (in-place streaming)."""

    def __init__(self, Lx: int, Lz: int, tau: float, g: float, wall_kind: int = 0, T_wall=(1.0, 1.0),
                 inplace: bool = False, device="cuda", _slab=None):
        import torch
        self._lib = binding.load()
        if not torch.cuda.is_available():
            raise LbmError("no CUDA device: the lattice update has no CPU fallback")
        self.Lx, self.Lz, self.tau, self.g = int(Lx), int(Lz), float(tau), float(g)
        self.device = torch.device(device)
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        nbytes = buffer_bytes(Lx, Lz) if _slab is None else slab_buffer_bytes(Lx, *_slab)
        if nbytes == 0:
            raise LbmError(f"invalid lattice {Lx} x {Lz}" + (f" / slab {_slab}" if _slab else ""))
        # the lattice copies (prv / nxt, or the one copy of the in-place path): torch owns the memory
        self._bufs = [torch.empty(nbytes // 8, dtype=torch.float64, device=self.device) for _ in range(1 if inplace else 2)]
        p = lbm_params(tau, g, wall_kind, self._bufs[0].data_ptr(), None if inplace else self._bufs[1].data_ptr(), nbytes,
                       float(T_wall[0]), float(T_wall[1]))
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            if _slab is None:
                binding.check(self._lib.lbm_create(C.byref(h), Lx, Lz, C.byref(p)))
            else:
                binding.check(self._lib.lbm_create_slab(C.byref(h), Lx, *_slab, C.byref(p)))
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
    @_on_device
    def init_rt(self, seed: int, T_d, T_m, T_u, rho_m=1.0, delta=0.0, smooth_w=2.5, pert_kind=0, n_modes=0,
                amp_lo=0.0, amp_hi=0.0, stream=None):
        ic = lbm_rt_init(T_d, T_m, T_u, rho_m, delta, smooth_w, pert_kind, n_modes, amp_lo, amp_hi)
        binding.check(self._lib.lbm_init_rt(self._h, C.c_uint64(seed), C.byref(ic), _stream_ptr(stream, self.device)))

    @_on_device
    def init_equilibrium(self, rho, ux, uz, T, stream=None):
        self._check_fields(rho, ux, uz, T)
        binding.check(self._lib.lbm_init_equilibrium(self._h, _dptr(rho), _dptr(ux), _dptr(uz), _dptr(T),
                                                     _stream_ptr(stream, self.device)))

    # ---- populations, canonical dense [37][Lz][Lx]
    @_on_device
    def set_populations(self, f, stream=None):
        self._check_pops(f)
        fn = self._lib.lbm_set_populations if f.is_cuda else self._lib.lbm_set_populations_host
        binding.check(fn(self._h, _dptr(f), _stream_ptr(stream, self.device)))

    @_on_device
    def get_populations(self, out=None, host=False, stream=None):
        import torch
        if out is None:
            out = torch.empty((NPOP, self.Lz, self.Lx), dtype=torch.float64, device="cpu" if host else self.device)
        self._check_pops(out)
        fn = self._lib.lbm_get_populations if out.is_cuda else self._lib.lbm_get_populations_host
        binding.check(fn(self._h, _dptr(out), _stream_ptr(stream, self.device)))
        return out

    @_on_device
    def get_window(self, k0: int, nk: int, i0: int, ni: int, stream=None):
        """Dense [37][nk][ni] populations of rows k0.., columns i0.. (mod Lx) (lbm_get_window)."""
        import torch
        out = torch.empty((NPOP, nk, ni), dtype=torch.float64, device=self.device)
        binding.check(self._lib.lbm_get_window(self._h, int(k0), int(nk), int(i0), int(ni), _dptr(out),
                                               _stream_ptr(stream, self.device)))
        return out

    # ---- the hot path
    @_on_device
    def step(self, n: int = 1, stream=None):
        binding.check(self._lib.lbm_step(self._h, int(n), _stream_ptr(stream, self.device)))

    # ---- diagnostics
    @_on_device
    def moments(self, rho=None, ux=None, uz=None, T=None, stream=None, alloc=True):
        import torch
        if alloc and rho is None and ux is None and uz is None and T is None:
            rho, ux, uz, T = (torch.empty((self.Lz, self.Lx), dtype=torch.float64, device=self.device) for _ in range(4))
        self._check_fields(*[x for x in (rho, ux, uz, T) if x is not None])
        binding.check(self._lib.lbm_moments(self._h, _dptr(rho), _dptr(ux), _dptr(uz), _dptr(T), _stream_ptr(stream, self.device)))
        return rho, ux, uz, T

    @_on_device
    def kinetic_moments(self, stream=None):
        """(rho, ux, uz, T) of eq. 7 without the half-force shift (lbm_kinetic_moments): the inputs of
        init_equilibrium / run_host.  New device tensors [Lz][Lx]."""
        import torch
        out = tuple(torch.empty((self.Lz, self.Lx), dtype=torch.float64, device=self.device) for _ in range(4))
        binding.check(self._lib.lbm_kinetic_moments(self._h, *[_dptr(x) for x in out], _stream_ptr(stream, self.device)))
        return out

    @_on_device
    def mixing_widths(self, T_d, T_m, T_u, want_tbar=True, stream=None):
        import numpy as np
        lu, ld = C.c_double(), C.c_double()
        tbar = np.empty(self.Lz) if want_tbar else None
        binding.check(self._lib.lbm_mixing_widths(self._h, T_d, T_m, T_u, C.byref(lu), C.byref(ld),
                                                  tbar.ctypes.data if want_tbar else None, _stream_ptr(stream, self.device)))
        return lu.value, ld.value, tbar

    @_on_device
    def profiles(self, stream=None):
        """(Tbar, Trms, Ekbar, Ekrms), host numpy arrays [Lz] (lbm_profiles)."""
        import numpy as np
        outs = [np.empty(self.Lz) for _ in range(4)]
        binding.check(self._lib.lbm_profiles(self._h, *[o.ctypes.data for o in outs], _stream_ptr(stream, self.device)))
        return tuple(outs)

    @_on_device
    def diagnostics(self, T_d=0.0, T_m=0.0, T_u=0.0, widths=True, totals=True, profiles=True, rms=True, stream=None):
        """lbm_diagnostics: widths (L_u, L_d), lattice totals and row profiles in one pass over the lattice.
        Returns a dict with the requested entries."""
        import numpy as np
        w, t = (C.c_double * 2)(), (C.c_double * 4)()
        rows = [np.empty(self.Lz) if profiles and (rms or j % 2 == 0) else None for j in range(4)]
        binding.check(self._lib.lbm_diagnostics(
            self._h, T_d, T_m, T_u, w if widths else None, t if totals else None,
            *[r.ctypes.data if r is not None else None for r in rows], _stream_ptr(stream, self.device)))
        out = {}
        if widths:
            out["L_u"], out["L_d"] = w[0], w[1]
        if totals:
            out["totals"] = np.array(list(t))
        if profiles:
            out["Tbar"], out["Trms"], out["Ekbar"], out["Ekrms"] = rows
        return out

    @_on_device
    def totals(self, stream=None):
        import numpy as np
        out = (C.c_double * 4)()
        binding.check(self._lib.lbm_totals(self._h, out, _stream_ptr(stream, self.device)))
        return np.array(list(out))

    @_on_device
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
                                             _stream_ptr(stream, self.device)))
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

    def plan(self):
        """(fused, strip_width, zchunk) of lbm_get_plan: how lbm_step launches on this lattice."""
        f, w, z = C.c_int(), C.c_int(), C.c_int()
        binding.check(self._lib.lbm_get_plan(self._h, C.byref(f), C.byref(w), C.byref(z)))
        return bool(f.value), w.value, z.value

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


class Slab(Lattice):
    """Rows [z0, z0 + nz) of an Lx x Lz_global lattice with ghost rows towards its neighbours (lbm_create_slab).
    Dense arrays cover the slab's own rows ([nz][Lx], [37][nz][Lx]).  One step = pack -> step(INTERIOR) ->
    (the caller moves the messages) -> unpack -> step(EDGES); `exchange_and_step` does it for slabs on one device."""
    INTERIOR, EDGES = 0, 1

    def __init__(self, Lx: int, Lz_global: int, z0: int, nz: int, tau: float, g: float, wall_kind: int = 0,
                 T_wall=(1.0, 1.0), device="cuda"):
        super().__init__(Lx, nz, tau, g, wall_kind=wall_kind, T_wall=T_wall, device=device, _slab=(Lz_global, z0, nz))
        self.Lz_global, self.z0, self.nz = int(Lz_global), int(z0), int(nz)
        z, n, lo, hi, m, m2 = C.c_int(), C.c_int(), C.c_int(), C.c_int(), C.c_size_t(), C.c_size_t()
        binding.check(self._lib.lbm_slab_info(self._h, C.byref(z), C.byref(n), C.byref(lo), C.byref(hi), C.byref(m),
                                              C.byref(m2)))
        self.open_below, self.open_above = bool(lo.value), bool(hi.value)
        self.message_doubles, self.message2_doubles = int(m.value), int(m2.value)

    def new_message(self, two_steps: bool = False):
        """A device buffer for one message of pack / unpack (two_steps: of pack2 / unpack2)."""
        import torch
        return torch.empty(self.message2_doubles if two_steps else self.message_doubles, dtype=torch.float64,
                           device=self.device)

    @_on_device
    def pack2(self, side: int, msg, stream=None):
        binding.check(self._lib.lbm_slab_pack2(self._h, int(side), _dptr(msg), _stream_ptr(stream, self.device)))

    @_on_device
    def unpack2(self, side: int, msg, stream=None):
        binding.check(self._lib.lbm_slab_unpack2(self._h, int(side), _dptr(msg), _stream_ptr(stream, self.device)))

    @_on_device
    def step2(self, stream=None):
        """Two time steps of the slab's own rows with the two-step kernel (after pack2 / transport / unpack2)."""
        binding.check(self._lib.lbm_slab_step2(self._h, _stream_ptr(stream, self.device)))

    @_on_device
    def step2_part(self, part: int, stream=None):
        """The two steps of step2 in two launches groups: INTERIOR (reads no ghost row; after pack2, while the messages
        travel) and EDGES (after unpack2) -- lbm_slab_step2_part."""
        binding.check(self._lib.lbm_slab_step2_part(self._h, int(part), _stream_ptr(stream, self.device)))

    @_on_device
    def pack(self, side: int, msg, stream=None):
        binding.check(self._lib.lbm_slab_pack(self._h, int(side), _dptr(msg), _stream_ptr(stream, self.device)))

    @_on_device
    def unpack(self, side: int, msg, stream=None):
        binding.check(self._lib.lbm_slab_unpack(self._h, int(side), _dptr(msg), _stream_ptr(stream, self.device)))

    @_on_device
    def step_part(self, part: int, stream=None):
        binding.check(self._lib.lbm_slab_step(self._h, int(part), _stream_ptr(stream, self.device)))

    def step(self, n: int = 1, stream=None):
        raise LbmError("a slab is stepped with pack / step_part / unpack (its ghost rows are exchanged every step)")
