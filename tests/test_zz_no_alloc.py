"""lbm_diagnostics_noalloc: the diagnostics pass for callers that cannot allocate device memory.

Some users of this library get their GPU memory from a pool they do not own (a framework's caching allocator, a fixed
carve-out of a shared GPU) or are called from inside another code's time loop.  A cudaMalloc there bypasses the pool
and stalls every stream of the device, so they can use neither lbm_create (it allocates the handle's scratch) nor
lbm_diagnostics.  The entry point tested here takes the raw lattice copy and keeps its scratch in a static 1 MiB
device array inside the library, at most LBM_NOALLOC_MAX_ROWS = 16384 lattice rows.

What is checked: its widths, totals and Tbar equal those of the existing handle path (lbm_diagnostics) on two calls in
a row that share the static array -- a tall lattice first, then a shorter one that reuses the bottom of the array
while the rest still holds the first call's rows, then the tall one again -- and that an oversized lattice is refused.
The existing path is itself compared with the CPU oracle in test_gpu_parity.py.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests.  It passes alone in a fresh process and after the other GPU tests.
"""
import ctypes as C

import numpy as np
import pytest

import synthetic_inputs as si

REL_TOL = 1e-12      # the bound test_gpu_parity.py puts on lattice totals; the same kernels run, so 0 is expected


def _existing_path(pkg, cfg, Lx, Lz, nsteps):
    """A lattice stepped `nsteps` (even: the current copy is buffer 0 again) and its lbm_diagnostics results."""
    lat = pkg.Lattice(Lx, Lz, cfg.tau, cfg.g)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    lat.step(nsteps)
    want = lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u, widths=True, totals=True, profiles=True, rms=False)
    return lat, want


def _no_alloc_path(pkg, torch, lat, cfg, result6, tbar):
    result6.fill_(float("nan"))
    tbar.fill_(float("nan"))
    pkg.diagnostics_noalloc(lat._bufs[0], lat.Lx, lat.Lz, cfg.g, cfg.T_d, cfg.T_m, cfg.T_u, result6, tbar)
    torch.cuda.synchronize()
    return result6.cpu().numpy(), tbar[: lat.Lz].cpu().numpy()


def _assert_same(got6, got_tbar, want, what):
    want6 = np.array([want["L_u"], want["L_d"], *want["totals"]])
    assert np.all(np.isfinite(got6)) and np.all(np.isfinite(got_tbar)), what
    scale = np.maximum(np.abs(want6), 1.0)
    assert np.max(np.abs(got6 - want6) / scale) <= REL_TOL, (what, got6, want6)
    assert np.max(np.abs(got_tbar - want["Tbar"]) / np.abs(want["Tbar"])) <= REL_TOL, what
    assert want6[0] > 0.0 and want6[1] > 0.0 and want6[2] > 0.0, (what, want6)    # a real front, not an all-zero match


@pytest.mark.gpu
def test_no_alloc_diagnostics_match_the_handle_path_on_consecutive_calls():
    import torch

    import paper_1405_1253_b200 as pkg

    cfg = si.rt_config(1)
    tall, want_tall = _existing_path(pkg, cfg, 300, 200, 4)
    short, want_short = _existing_path(pkg, cfg, 64, 128, 6)
    # outputs belong to the caller; allocated here, once, before the calls under test
    result6 = torch.empty(6, dtype=torch.float64, device="cuda")
    tbar = torch.empty(200, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    for lat, want, what in ((tall, want_tall, "first call, 300x200"), (short, want_short, "second call, 64x128"),
                            (tall, want_tall, "third call, 300x200 again")):
        got6, got_tbar = _no_alloc_path(pkg, torch, lat, cfg, result6, tbar)
        _assert_same(got6, got_tbar, want, what)
    tall.close()
    short.close()


def test_no_alloc_refuses_lattices_beyond_its_static_array():
    """Argument checks run before any device work, so this needs no GPU."""
    import __graft_entry__ as g
    g.build()
    from paper_1405_1253_b200 import binding
    lib = binding.load()
    too_tall = binding.NOALLOC_MAX_ROWS + 1
    rc = lib.lbm_diagnostics_noalloc(C.c_void_p(256), C.c_size_t(1 << 50), 64, too_tall, 1e-4, 1.0, 0.9, 0.8,
                                     C.c_void_p(512), None, None)
    assert rc == -1
    msg = lib.lbm_last_error().decode()
    assert "LBM_NOALLOC_MAX_ROWS" in msg and str(binding.NOALLOC_MAX_ROWS) in msg
    header = open(g.ROOT + "/include/lbm.h").read()
    assert f"#define LBM_NOALLOC_MAX_ROWS {binding.NOALLOC_MAX_ROWS}" in header
    # null buffer, undersized buffer, misaligned buffer: refused the same way
    assert lib.lbm_diagnostics_noalloc(None, C.c_size_t(1 << 50), 64, 128, 1e-4, 1.0, 0.9, 0.8, C.c_void_p(512), None, None) == -1
    assert lib.lbm_diagnostics_noalloc(C.c_void_p(256), C.c_size_t(64), 64, 128, 1e-4, 1.0, 0.9, 0.8, C.c_void_p(512), None, None) == -1
    assert lib.lbm_diagnostics_noalloc(C.c_void_p(264), C.c_size_t(1 << 50), 64, 128, 1e-4, 1.0, 0.9, 0.8, C.c_void_p(512), None, None) == -1
