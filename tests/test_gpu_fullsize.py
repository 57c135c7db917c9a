"""Full-size GPU checks in the launch configuration bench.py times (4096x8192, default variant) and at the
largest config-5 lattice (8192x16384, element offsets beyond 2^32): sampled windows are recomputed by the
oracle one by one (the domain of dependence of a site after n steps is a (6n+1)^2 window), plus properties
that hold at any size."""
import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu
NSTEPS = 3
M = 3 * NSTEPS      # rows/columns near a window edge that see outside the window


@pytest.fixture(scope="module")
def pkg():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    if torch.cuda.get_device_properties(0).total_memory < 150e9:
        pytest.skip("needs a 180 GB device")
    import __graft_entry__ as g
    g.build()
    import paper_1405_1253_b200 as p
    return p


def _window(dense, r0, r1, cols):
    return dense[:, r0:r1][:, :, cols].contiguous().cpu().numpy()


def _check_windows(orc, before, after, Lx, Lz, tau, g, tol):
    """before/after: dense device populations [37][Lz][Lx] at step 0 and step NSTEPS."""
    import torch
    W = 40
    worst = 0.0
    cases = [  # (first row, first column, kind)
        (0, Lx - 17, "bottom"),                 # bottom wall, straddles the periodic seam
        (Lz - W, Lx // 2 + 5, "top"),           # top wall
        (Lz // 2 - W // 2, 3, "bulk"),          # the interface region
        (Lz - W - 1000, Lx - 23, "bulk"),       # far rows, seam
    ]
    for r0, c0, kind in cases:
        cols = (torch.arange(c0, c0 + W, device=before.device) % Lx)
        w0 = _window(before, r0, r0 + W, cols)
        w1 = _window(after, r0, r0 + W, cols)
        ref = orc.step(w0, tau, g, nsteps=NSTEPS, periodic_z=(kind == "bulk"))
        rows = slice(0, W - M) if kind == "bottom" else slice(M, W) if kind == "top" else slice(M, W - M)
        a, b = w1[:, rows, M:W - M], ref[:, rows, M:W - M]
        worst = max(worst, float(np.max(np.abs(a - b) / np.abs(b))))
    assert worst < tol, worst
    return worst


def test_config4_fullsize_sampled_windows_and_conservation(pkg, orc):
    """BASELINE.json configs[3] exactly as bench.py launches it."""
    cfg = si.rt_config(4)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    t0 = lat.totals()
    before = lat.get_populations()
    lat.step(NSTEPS)
    after = lat.get_populations()
    _check_windows(orc, before, after, cfg.Lx, cfg.Lz, cfg.tau, cfg.g, 1e-13)
    del before, after
    lat.step(50 - NSTEPS)
    t1 = lat.totals()
    assert abs(t1[0] / t0[0] - 1) < 1e-13                     # mass
    assert abs(t1[1]) < 1e-9 * t0[0]                          # no net x momentum appears
    lu, ld, tbar = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    assert np.all(np.isfinite(tbar)) and abs(tbar[0] - cfg.T_d) < 1e-3 and abs(tbar[-1] - cfg.T_u) < 1e-3
    assert 2.0 < lu < 12.0 and 2.0 < ld < 12.0 and abs(lu - ld) < 0.5   # tanh front of w = 2.5, diffusing
    lat.close()


def test_largest_sweep_lattice_offsets_beyond_32_bits(pkg, orc):
    """8192x16384 (79.5 GB of populations): init_equilibrium + 3 steps, windows checked from the oracle's own
    equilibrium of the same seeded fields."""
    import torch
    Lx, Lz = si.SWEEP_SIZES[-1]
    fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
    lat = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G)
    lat.init_equilibrium(*fields)
    before = lat.get_populations()
    # init parity on a far window (plane 36 sits 4.8e9 doubles into the buffer)
    r0, c0, W = Lz - 64, Lx - 64, 48
    host = si.sweep_fields(Lx, Lz, si.DEFAULT_SEED, rows=slice(r0, r0 + W))
    ref0 = orc.init_equilibrium(*[np.ascontiguousarray(x[:, c0:c0 + W]) for x in host])
    got0 = _window(before, r0, r0 + W, torch.arange(c0, c0 + W, device="cuda"))
    assert float(np.max(np.abs(got0 - ref0) / ref0)) < 1e-13
    del fields
    lat.step(NSTEPS)
    after = lat.get_populations()
    _check_windows(orc, before, after, Lx, Lz, si.SWEEP_TAU, si.SWEEP_G, 1e-13)
    lat.close()


@pytest.mark.gpu
def test_two_step_kernel_back_to_back_launches_stay_bitwise_equal(pkg):
    """Regression for a shared-memory hand-off race of the two-step kernel that only showed with many launches back
    to back on a lattice of >= 1024 x 2048 (a stage buffer released before its loads had completed was overwritten
    by the next TMA load when the source rows were L2-resident; about one block in 1e5): 200 steps in one call,
    default (two-step) kernel against the one-step kernel, every population of every site, bit for bit."""
    import torch
    Lx, Lz = 1024, 2048
    fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
    a, b = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G), pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G)
    a.set_variant(1)
    l0 = b.kernel_launches
    for lat in (a, b):
        lat.init_equilibrium(*fields)
        lat.step(200)
    assert b.kernel_launches - l0 == 1 + 100          # init + 100 two-step launches: the default path is the fused one
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()
