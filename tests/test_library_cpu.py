"""CPU tier for the CUDA library: it builds, exports every symbol of include/lbm.h, its host-side logic
(argument checks, buffer sizes, tables) behaves, and the product path has no CPU fallback.
No compute call is made here (there is no GPU)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as g
    g.build()
    from paper_1405_1253_b200 import binding
    return binding.load()


def test_library_exports_every_declared_symbol(lib):
    from paper_1405_1253_b200 import binding
    header = open(os.path.join(ROOT, "include", "lbm.h")).read()
    declared = set(re.findall(r"\b(lbm_[a-z0-9_]+)\s*\(", header))
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_buffer_bytes_and_layout_rules(lib):
    assert lib.lbm_buffer_bytes(6, 128) == 0 and lib.lbm_buffer_bytes(64, 5) == 0
    for Lx, Lz in [(64, 128), (100, 37), (4096, 8192)]:
        b = lib.lbm_buffer_bytes(Lx, Lz)
        pitch = (Lx + 15) // 16 * 16
        assert b >= 37 * pitch * Lz * 8 and b % 128 == 0
        plane = b // 37
        assert plane % 128 == 0                       # plane bases stay on 128-byte lines
        assert (plane // 128) % 2 == 1 or Lx % 32     # ... and off power-of-two strides


def test_tables_match_paper_constants(lib):
    """The library's own tables satisfy the same paper pins as the oracle's (M = 37, r ~ 1.1969,
    PAPER.md:75, 100) and the Gaussian moment conditions -- checked independently of the oracle."""
    import paper_1405_1253_b200 as pkg
    ex, ez, w, r = pkg.tables()
    ex, ez, w = np.array(ex), np.array(ez), np.array(w)
    assert len(ex) == 37 and int(r * 1e4) == 11969
    assert np.all(ex[::-1] == -ex) and np.all(ez[::-1] == -ez) and abs(w.sum() - 1) < 1e-15
    for a, b, want in [(2, 0, 1), (4, 0, 3), (2, 2, 1), (6, 0, 15), (4, 2, 3), (8, 0, 105), (6, 2, 15), (4, 4, 9)]:
        assert abs(np.sum(w * (r * ex) ** a * (r * ez) ** b) - want) < 1e-12 * want


def test_create_rejects_bad_arguments_before_touching_a_device(lib):
    from paper_1405_1253_b200.binding import lbm_params
    h = C.c_void_p()
    good = dict(tau=0.8, g=1e-4, wall_kind=0, pop_buf0=256, pop_buf1=512, buf_bytes=1 << 40)
    for bad in [dict(tau=0.5), dict(g=-1.0), dict(wall_kind=3), dict(pop_buf0=0), dict(pop_buf1=256),
                dict(pop_buf0=264), dict(buf_bytes=16)]:
        p = lbm_params(**{**good, **bad})
        assert lib.lbm_create(C.byref(h), 64, 128, C.byref(p)) == -1, bad
        assert h.value is None and lib.lbm_last_error()
    p = lbm_params(**good)
    assert lib.lbm_create(C.byref(h), 3, 128, C.byref(p)) == -1
    assert lib.lbm_create(C.byref(h), 64, 128, None) == -1
    assert lib.lbm_step(None, 1, None) == -1 and lib.lbm_destroy(None) == 0


def test_no_cpu_fallback_and_no_oracle_on_the_product_path():
    """The package never imports oracle/ and refuses to run without a device."""
    import torch
    import paper_1405_1253_b200 as pkg
    pkgdir = os.path.dirname(pkg.__file__)
    for dirpath, _, files in os.walk(pkgdir):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "lbm_oracle" not in src, fn
    if not torch.cuda.is_available():
        with pytest.raises(pkg.LbmError):
            pkg.Lattice(64, 128, 0.8, 1e-4)


def test_synthetic_inputs_are_reproducible_and_sliceable():
    import synthetic_inputs as si
    full = si.sweep_fields(32, 24, seed=5)
    part = si.sweep_fields(32, 24, seed=5, rows=slice(7, 12))
    for a, b in zip(full, part):
        assert np.array_equal(a[7:12], b)
    rho, ux, uz, T = full
    assert abs(rho.mean() - 1) < 2e-3 and np.all(np.abs(rho - 1) <= 0.01) and np.all(np.abs(ux) <= 0.01)
    assert np.all(np.abs(T - 1) <= 0.01) and np.all(np.abs(uz) <= 0.01)
    cfg = si.rt_config(4)
    assert (cfg.Lx, cfg.Lz, cfg.delta, cfg.pert_kind) == (4096, 8192, 0.0, si.PERT_WHITE)
    assert si.scaled(si.rt_config(2), 128, 256).delta == 64


def test_growth_rate_host_function_matches_oracle_and_closed_form(lib, orc):
    """lbm_growth_rate is host-only post-processing (eq. 11 / 14), so it is checked here without a GPU."""
    import paper_1405_1253_b200 as pkg
    rng = np.random.default_rng(8)
    t = np.cumsum(rng.uniform(50, 150, 30))
    L = 0.05 * 1.5e-5 * 0.025 * t ** 2 * (1 + 0.1 * np.sin(t / 300))
    a, b = pkg.growth_rate(t, L, 1.5e-5, 0.025), orc.growth_rate(t, L, 1.5e-5, 0.025)
    assert np.max(np.abs(a - b)) <= 1e-15 * np.max(np.abs(b))
    tq = np.arange(1, 20) * 100.0
    assert np.max(np.abs(pkg.growth_rate(tq, 0.04 * 1e-4 * 0.05 * tq ** 2, 1e-4, 0.05)[1:-1] / 0.04 - 1)) < 1e-12
    with pytest.raises(pkg.LbmError):
        pkg.growth_rate(tq[::-1].copy(), tq, 1e-4, 0.05)      # times must increase
    with pytest.raises(pkg.LbmError):
        pkg.growth_rate(tq, tq, 0.0, 0.05)


def test_two_step_kernel_releases_buffers_only_after_consuming_them(lib):
    """Guards the fix of the hand-off race of lbm_step2s.cuh (profiles/r1_two_step.md, section 4) against compiler
    scheduling: in the SASS of step2s_kernel every gather of 37 populations from shared memory (a run of LDS) must be
    followed by the moment sums (>= 60 DADD, which cannot issue before the loaded values have returned) BEFORE the
    next mbarrier arrive (SYNCS.ARRIVE) that releases the buffer.  First line of defence is the proxy fence in the
    kernel (FENCE.VIEW.ASYNC.S must be present too).  Skipped where cuobjdump is not installed (fails on a GPU box)."""
    import shutil
    import subprocess
    from paper_1405_1253_b200 import binding
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        import torch
        assert not torch.cuda.is_available(), "cuobjdump is missing on a GPU box: the hand-off guard cannot be checked"
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    ops, inside = [], False
    for line in sass.splitlines():
        if "Function :" in line:
            inside = "step2s_kernel" in line
        elif inside and "/*" in line and "*/" in line:
            body = line.split("*/", 1)[1].strip()
            tok = body.split()
            if not tok:
                continue
            op = tok[1] if tok[0].startswith("@") and len(tok) > 1 else tok[0]
            ops.append(op.rstrip(";"))
    assert ops, "step2s_kernel not found in the library"
    gathers = 0
    i = 0
    while i < len(ops):
        if ops[i].startswith("LDS"):
            j, n_lds = i, 0
            while j < len(ops) and not ops[j].startswith(("DADD", "SYNCS")):   # the run of loads (with address arithmetic)
                n_lds += ops[j].startswith("LDS")
                j += 1
            if n_lds >= 30:
                gathers += 1
                k, n_dadd = j, 0
                while k < len(ops) and not ops[k].startswith("SYNCS.ARRIVE"):
                    n_dadd += ops[k].startswith("DADD")
                    k += 1
                assert k < len(ops), "no release after a gather"
                assert n_dadd >= 60, f"buffer released after only {n_dadd} DADD following a gather of {n_lds} LDS"
            i = j
        i += 1
    assert gathers >= 2, f"expected the producers' and the consumers' gathers, found {gathers}"
    assert any(o.startswith("FENCE.VIEW.ASYNC") for o in ops), "the stage reads are not fenced into the async proxy"


def test_slab_buffer_bytes_refuses_what_create_slab_refuses(lib):
    """the size query and lbm_create_slab agree on the smallest slab (6 own rows)."""
    for nz in (3, 4, 5):
        assert lib.lbm_slab_buffer_bytes(64, 128, 10, nz) == 0
    assert lib.lbm_slab_buffer_bytes(64, 128, 10, 6) > 0
