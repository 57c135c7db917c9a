"""Full-size GPU checks in the launch configuration bench.py times (4096x8192, default variant) and at the
largest config-5 lattice (8192x16384, element offsets beyond 2^32): sampled windows are recomputed by the
oracle one by one (the domain of dependence of a site after n steps is a (6n+1)^2 window), plus properties
that hold at any size."""
import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu
NSTEPS = 7          # three fused launches of the two-step kernel and one single step
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


def _check_windows(orc, before, after, Lx, Lz, tau, g, tol, plan=None, walls=None):
    """before/after: dense device populations [37][Lz][Lx] at step 0 and step NSTEPS.  With `plan` = (fused, strip
    width w, rows per chunk ZC) of the launch, extra windows straddle a chunk boundary (rows around c ZC, where one
    block hands over to the next: ring wrap, warm-up rows) and a strip boundary (columns around s w)."""
    import torch
    W = 40 + 2 * M
    worst = 0.0
    cases = [  # (first row, first column, kind)
        (0, Lx - W // 2 - 1, "bottom"),         # bottom wall, straddles the periodic seam
        (Lz - W, Lx // 2 + 5, "top"),           # top wall
        (Lz // 2 - W // 2, 3, "bulk"),          # the interface region
        (Lz - W - 1000, Lx - W // 2 - 3, "bulk"),   # far rows, seam
    ]
    if plan is not None and plan[0]:
        _, w, zc = plan
        nchunks, nstrips = (Lz + zc - 1) // zc, (Lx + w - 1) // w
        assert nstrips >= 3
        sx = (nstrips // 2) * w                  # a strip boundary in the middle of the lattice
        cases.append((Lz // 3, sx - W // 2, "bulk"))                     # a strip boundary
        if nchunks >= 2:
            cases += [
                (zc - W // 2, sx - W // 2, "bulk"),                          # first chunk boundary x strip boundary
                ((nchunks // 2) * zc - W // 2, sx - W // 2 + 11, "bulk"),    # a middle chunk boundary
                ((nchunks - 1) * zc - W // 2, Lx - W // 2, "bulk"),          # last chunk boundary on the seam
            ]
    for r0, c0, kind in cases:
        cols = (torch.arange(c0, c0 + W, device=before.device) % Lx)
        w0 = _window(before, r0, r0 + W, cols)
        w1 = _window(after, r0, r0 + W, cols)
        if walls is not None and kind != "bulk":   # wall_kind 1: `walls` = (T_bottom, T_top); bulk rows do not see the wall rule
            ref = orc.step(w0, tau, g, nsteps=NSTEPS, wall_kind=1, T_bot=walls[0], T_top=walls[1])
        else:
            ref = orc.step(w0, tau, g, nsteps=NSTEPS, periodic_z=(kind == "bulk"))
        rows = slice(0, W - M) if kind == "bottom" else slice(M, W) if kind == "top" else slice(M, W - M)
        a, b = w1[:, rows, M:W - M], ref[:, rows, M:W - M]
        worst = max(worst, float(np.max(np.abs(a - b) / np.abs(b))))
    assert worst < tol, worst
    return worst


def _check_row_slabs_after_n_steps(orc, lat, cfg, n, centres, tol, walls=None, h=24):
    """The north_star criterion at full size: `lat` (initialised, at step 0) is stepped n times; for each (kind, row)
    of `centres` the oracle steps a full-width slab (exact periodic x) of h rows plus 3n rows of halo -- the domain of
    dependence of a row after n steps -- and the h rows are compared population by population.  Bulk slabs are closed
    periodically in z (the wrong closure stays within the halo); wall slabs have the real wall on one side."""
    halo = 3 * n
    spans = []
    for kind, centre in centres:
        if kind == "bulk":
            spans.append((centre - h // 2 - halo, centre + h // 2 + halo, slice(halo, halo + h)))
        elif kind == "bottom":
            spans.append((0, h + halo, slice(0, h)))
        else:
            spans.append((cfg.Lz - h - halo, cfg.Lz, slice(halo, halo + h)))
    assert all(0 <= r0 and r1 <= cfg.Lz for r0, r1, _ in spans), spans
    before = [lat.get_window(r0, r1 - r0, 0, cfg.Lx).cpu().numpy() for r0, r1, _ in spans]
    lat.step(n)
    worst = 0.0
    for (kind, _), (r0, r1, rows), w0 in zip(centres, spans, before):
        w1 = lat.get_window(r0, r1 - r0, 0, cfg.Lx).cpu().numpy()
        if walls is not None and kind != "bulk":
            ref = orc.step(w0, cfg.tau, cfg.g, nsteps=n, wall_kind=1, T_bot=walls[0], T_top=walls[1])
        else:
            ref = orc.step(w0, cfg.tau, cfg.g, nsteps=n, periodic_z=(kind == "bulk"))
        worst = max(worst, float(np.max(np.abs(w1[:, rows] - ref[:, rows]) / np.abs(ref[:, rows]))))
        del w1, ref
    assert worst < tol, worst
    return worst


def test_config4_100_steps_slabs_against_oracle(pkg, orc):
    """the headline lattice (BASELINE.json configs[3], 4096x8192) in the launch bench.py times, after
    100 steps -- the north_star criterion, 1e-11 per population -- on full-width row slabs at the interface, at both
    walls and across a chunk boundary of the launch plan; lattice totals to 1e-12."""
    cfg = si.rt_config(4)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    fused, w, zc = lat.plan()
    assert fused and zc < cfg.Lz
    nchunks = (cfg.Lz + zc - 1) // zc
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    t0 = lat.totals()
    centres = [("bulk", cfg.Lz // 2), ("bottom", 0), ("top", cfg.Lz), ("bulk", (nchunks // 4) * zc)]
    _check_row_slabs_after_n_steps(orc, lat, cfg, 100, centres, 1e-11)
    t1 = lat.totals()
    assert abs(t1[0] / t0[0] - 1) < 1e-12                    # mass
    lat.close()


def test_isothermal_walls_at_size_with_the_automatic_plan(pkg, orc):
    """wall_kind 1 runs its own instances of the step kernels.  2048x4096 (config 3), automatic plan,
    100 steps: both wall slabs against the oracle's isothermal-wall step and the lower interface, 1e-11.
    4096x8192 (config 4): 7-step windows on both walls, the seam, strip and chunk boundaries, 1e-13."""
    cfg = si.rt_config(3)
    walls = (cfg.T_d, cfg.T_u)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, wall_kind=1, T_wall=walls)
    assert lat.plan()[0]
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    _check_row_slabs_after_n_steps(orc, lat, cfg, 100, [("bottom", 0), ("top", cfg.Lz), ("bulk", int(cfg.Lz / 2 - cfg.delta / 2))],
                                   1e-11, walls=walls)
    lat.close()
    cfg = si.rt_config(4)
    walls = (cfg.T_d + 0.01, cfg.T_u - 0.01)                 # walls that differ from the fluid next to them
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, wall_kind=1, T_wall=walls)
    plan = lat.plan()
    assert plan[0] and plan[2] < cfg.Lz
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    before = lat.get_populations()
    lat.step(NSTEPS)
    after = lat.get_populations()
    _check_windows(orc, before, after, cfg.Lx, cfg.Lz, cfg.tau, cfg.g, 1e-13, plan, walls=walls)
    lat.close()


def test_two_slabs_of_config3_isothermal_walls_fused_path_equal_the_whole_lattice(pkg):
    """config 3 with wall_kind 1 as two z-slabs stepped with the two-step kernel (pack2 / unpack2 /
    step2), 50 steps, against the whole lattice with the automatic plan: bit-identical."""
    import torch
    from test_gpu_variants import _run_slabs_fused
    cfg = si.rt_config(3)
    kw = dict(wall_kind=1, T_wall=(cfg.T_d, cfg.T_u))
    whole = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, **kw)
    assert whole.plan()[0]
    whole.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    whole.step(50)
    ref = whole.get_populations()
    whole.close()
    slabs = [pkg.Slab(cfg.Lx, cfg.Lz, z0, nz, cfg.tau, cfg.g, **kw) for z0, nz in ((0, 2048), (2048, 2048))]
    for s in slabs:
        s.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    _run_slabs_fused(pkg, slabs, 25)
    for s, rows in zip(slabs, (slice(0, 2048), slice(2048, 4096))):
        assert torch.equal(s.get_populations(), ref[:, rows])
        s.close()


def test_config4_fullsize_sampled_windows_and_conservation(pkg, orc):
    """BASELINE.json configs[3] exactly as bench.py launches it."""
    cfg = si.rt_config(4)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    plan = lat.plan()
    assert plan[0] and plan[2] < cfg.Lz                      # the bench's launch: the two-step kernel, several chunks
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    t0 = lat.totals()
    before = lat.get_populations()
    lat.step(NSTEPS)
    after = lat.get_populations()
    _check_windows(orc, before, after, cfg.Lx, cfg.Lz, cfg.tau, cfg.g, 1e-13, plan)
    del before, after
    lat.step(50 - NSTEPS)
    t1 = lat.totals()
    assert abs(t1[0] / t0[0] - 1) < 1e-13                     # mass
    assert abs(t1[1]) < 1e-9 * t0[0]                          # no net x momentum appears
    lu, ld, tbar = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    assert np.all(np.isfinite(tbar)) and abs(tbar[0] - cfg.T_d) < 1e-3 and abs(tbar[-1] - cfg.T_u) < 1e-3
    assert 2.0 < lu < 12.0 and 2.0 < ld < 12.0 and abs(lu - ld) < 0.5   # tanh front of w = 2.5, diffusing
    # row profiles at this width (the rows' T and E_k kept in 64 KB of shared memory between the two passes): rows
    # around the front against the oracle's profiles of the same rows
    prof = lat.profiles()
    r0 = cfg.Lz // 2 - 4
    want = orc.profiles(lat.get_window(r0, 8, 0, cfg.Lx).cpu().numpy(), cfg.g)
    for a, b, tol in zip(prof, want, (1e-12, 1e-11, 1e-15, 1e-14)):
        assert np.max(np.abs(a[r0:r0 + 8] - b)) < tol, (np.max(np.abs(a[r0:r0 + 8] - b)), tol)
    assert want[1].max() > 1e-6
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
    plan = lat.plan()
    lat.step(NSTEPS)
    after = lat.get_populations()
    _check_windows(orc, before, after, Lx, Lz, si.SWEEP_TAU, si.SWEEP_G, 1e-13, plan)
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
    assert b.kernel_launches - l0 == 1 + 1 + 100      # init + wrap-column refresh + 100 two-step launches: the default path is the fused one
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


def test_config3_100_steps_slabs_against_oracle(pkg, orc):
    """BASELINE.json configs[2]: 2048x4096 double front, white-noise interfaces, tau = 0.7, the automatic launch plan,
    100 steps (the north_star criterion).  The domain of dependence of a row after n steps is +-3n rows, so the
    oracle steps full-width slabs (exact periodic x, seam included) of h + 2 x 300 rows and the central h rows are
    compared population by population: one slab per interface, one on the bottom wall, one on the top wall."""
    cfg = si.rt_config(3)
    n, h = 100, 24
    halo = 3 * n
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    assert lat.plan()[0]
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    before = lat.get_populations()
    lat.step(n)
    after = lat.get_populations()
    lat.close()
    lo_if, hi_if = int(cfg.Lz / 2 - cfg.delta / 2), int(cfg.Lz / 2 + cfg.delta / 2)
    worst = 0.0
    for kind, centre in (("bulk", lo_if), ("bulk", hi_if), ("bottom", 0), ("top", cfg.Lz)):
        if kind == "bulk":
            r0, r1 = centre - h // 2 - halo, centre + h // 2 + halo
            rows = slice(halo, halo + h)
        elif kind == "bottom":
            r0, r1 = 0, h + halo
            rows = slice(0, h)
        else:
            r0, r1 = cfg.Lz - h - halo, cfg.Lz
            rows = slice(halo, halo + h)
        w0 = before[:, r0:r1].contiguous().cpu().numpy()
        w1 = after[:, r0:r1].contiguous().cpu().numpy()
        # bulk slabs: periodic in z (the contamination from the wrong closure stays within `halo` rows of the edges);
        # wall slabs: the real wall on one side, a spurious wall on the other, `halo` rows away from the rows compared
        ref = orc.step(w0, cfg.tau, cfg.g, nsteps=n, periodic_z=(kind == "bulk"))
        a, b = w1[:, rows], ref[:, rows]
        worst = max(worst, float(np.max(np.abs(a - b) / np.abs(b))))
        del w0, w1, ref
    assert worst < 1e-11, worst


def test_two_step_kernel_bitwise_at_the_large_lattice_plan(pkg):
    """The two-step kernel in the launch plan of the large lattices (a few long chunks per strip, whole waves) against
    the one-step kernel, 50 steps at 2048x4096, every population of every site, bit for bit."""
    import torch
    Lx, Lz = 2048, 4096
    fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
    a, b = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G), pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G)
    a.set_variant(1)
    fused, w, zc = b.plan()
    assert fused and zc >= 128
    for lat in (a, b):
        lat.init_equilibrium(*fields)
        lat.step(50)
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


def test_inplace_16384x16384_one_copy_windows_against_oracle(pkg, orc):
    """16384 x 16384 (80 GB for ONE lattice copy; two would not leave room for anything else on a 180 GB
    device) with in-place streaming: equilibrium of the seeded config-5 fields, NSTEPS steps (ending in the shifted
    layout, NSTEPS is odd), windows through lbm_get_window against the oracle's own equilibrium + steps: walls, seam,
    bulk, element offsets beyond 2^33."""
    import torch
    Lx = Lz = 16384
    lat = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G, inplace=True)
    fields = si.sweep_fields_torch(Lx, Lz, si.DEFAULT_SEED, "cuda")
    lat.init_equilibrium(*fields)
    del fields
    torch.cuda.empty_cache()
    W = 40 + 2 * M
    cases = [(0, Lx - W // 2 - 1, "bottom"), (Lz - W, Lx // 2 + 5, "top"), (Lz // 2 - 7, 3, "bulk"), (Lz - W - 1000, Lx - W // 2 - 3, "bulk")]
    before = [lat.get_window(r0, W, c0, W).cpu().numpy() for r0, c0, _ in cases]
    # the oracle's own equilibrium of the same seeded fields on the first window
    r0, c0, _ = cases[2]
    host = si.sweep_fields(Lx, Lz, si.DEFAULT_SEED, rows=slice(r0, r0 + W))
    ref0 = orc.init_equilibrium(*[np.ascontiguousarray(x[:, c0:c0 + W]) for x in host])
    assert float(np.max(np.abs(before[2] - ref0) / ref0)) < 1e-13
    lat.step(NSTEPS)
    assert NSTEPS % 2 == 1
    worst = 0.0
    for (r0, c0, kind), w0 in zip(cases, before):
        w1 = lat.get_window(r0, W, c0, W).cpu().numpy()
        ref = orc.step(w0, si.SWEEP_TAU, si.SWEEP_G, nsteps=NSTEPS, periodic_z=(kind == "bulk"))
        rows = slice(0, W - M) if kind == "bottom" else slice(M, W) if kind == "top" else slice(M, W - M)
        a, b = w1[:, rows, M:W - M], ref[:, rows, M:W - M]
        worst = max(worst, float(np.max(np.abs(a - b) / np.abs(b))))
    assert worst < 1e-13, worst
    t = lat.totals()
    assert abs(t[0] / (Lx * Lz) - 1) < 1e-3                   # rho = 1 +- 0.01 per site
    lat.close()


def test_two_slabs_of_config3_equal_the_whole_lattice_after_100_steps(pkg):
    """SURVEY 8(f)4 on one device: the 2048x4096 lattice of config 3 as two z-slabs, ghost rows exchanged every step by
    device-to-device copies on a second stream while the interior rows run, against the whole lattice stepped with the
    default plan (two-step kernel): bit-identical after 100 steps."""
    import torch
    from test_gpu_variants import _run_slabs
    cfg = si.rt_config(3)
    whole = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    assert whole.plan()[0]
    whole.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    whole.step(100)
    ref = whole.get_populations()
    whole.close()
    slabs = [pkg.Slab(cfg.Lx, cfg.Lz, z0, nz, cfg.tau, cfg.g) for z0, nz in ((0, 2048), (2048, 2048))]
    for s in slabs:
        s.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    _run_slabs(pkg, slabs, 100)
    for s, rows in zip(slabs, (slice(0, 2048), slice(2048, 4096))):
        assert torch.equal(s.get_populations(), ref[:, rows])
        s.close()
