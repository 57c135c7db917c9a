"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (north_star): max relative error per population <= 1e-11 after 100 steps,
conserved totals to 1e-12 relative.  Run on the B200 box: pytest -m gpu."""
import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu

POP_RTOL = 1e-11
TOT_RTOL = 1e-12


@pytest.fixture(scope="module")
def pkg():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import __graft_entry__ as g
    g.build()
    import paper_1405_1253_b200 as p
    return p


def _rel(a, b):
    return float(np.max(np.abs(a - b) / np.abs(b)))


def _oracle_rt(orc, cfg, seed, nsteps):
    f0 = orc.init_rt(cfg.Lx, cfg.Lz, cfg.g, seed, **cfg.rt_args())
    return f0, orc.step(f0, cfg.tau, cfg.g, nsteps=nsteps)


def test_tables_agree_with_oracle(pkg, orc):
    ex, ez, w, r = pkg.tables()
    oex, oez, ow, orr = orc.tables()
    assert list(oex) == ex and list(oez) == ez
    assert np.max(np.abs(np.array(w) / ow - 1)) < 4e-16 and abs(r / orr - 1) < 4e-16


def test_config1_init_matches_oracle(pkg, orc):
    cfg = si.rt_config(1)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    got = lat.get_populations(host=True).numpy()
    ref = orc.init_rt(cfg.Lx, cfg.Lz, cfg.g, si.DEFAULT_SEED, **cfg.rt_args())
    assert _rel(got, ref) < 1e-13        # exp/tanh/log1p differ by an ulp or two between libm and CUDA
    lat.close()


@pytest.mark.parametrize("variant", [0, 1, 2, 3])
def test_config1_100_steps_population_parity(pkg, orc, variant):
    """BASELINE.json configs[0]: 64x128 double-front RT, 100 steps, every population of every site."""
    cfg = si.rt_config(1)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    lat.set_variant(variant)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    lat.step(cfg.steps)
    assert lat.steps_done == 100
    got = lat.get_populations(host=True).numpy()
    _, ref = _oracle_rt(orc, cfg, si.DEFAULT_SEED, cfg.steps)
    assert _rel(got, ref) < POP_RTOL
    tg, tr = lat.totals(), orc.totals(ref)
    assert abs(tg[0] / tr[0] - 1) < TOT_RTOL and abs(tg[3] / tr[3] - 1) < TOT_RTOL
    assert abs(tg[1] - tr[1]) < TOT_RTOL * tr[0] and abs(tg[2] - tr[2]) < TOT_RTOL * tr[0]
    lat.close()


def test_config2_100_steps_population_parity_automatic_plan(pkg, orc):
    """BASELINE.json configs[1] in full: 512x1024 double-front RT, 16 modes, seed 12345, the AUTOMATIC launch plan
    (the two-step kernel with many short chunks at this size), 100 steps: every population of every site, the
    lattice totals and the mixing widths L_u, L_d against the oracle."""
    cfg = si.rt_config(2)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    fused, w, zc = lat.plan()
    assert fused and w < cfg.Lx and zc < cfg.Lz              # several strips and several chunks per strip
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    lat.step(100)
    got = lat.get_populations(host=True).numpy()
    _, ref = _oracle_rt(orc, cfg, si.DEFAULT_SEED, 100)
    assert _rel(got, ref) < POP_RTOL
    tg, tr = lat.totals(), orc.totals(ref)
    assert abs(tg[0] / tr[0] - 1) < TOT_RTOL and abs(tg[3] / tr[3] - 1) < TOT_RTOL
    assert abs(tg[1] - tr[1]) < TOT_RTOL * tr[0] and abs(tg[2] - tr[2]) < TOT_RTOL * tr[0]
    lu, ld, tbar = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    olu, old, otbar = orc.mixing_widths(ref, cfg.g, cfg.T_d, cfg.T_m, cfg.T_u)
    assert np.max(np.abs(tbar - otbar)) < 1e-13 and abs(lu - olu) < 1e-10 and abs(ld - old) < 1e-10
    lat.close()


@pytest.mark.parametrize("variant", [0, 3])
@pytest.mark.parametrize("Lx,Lz,steps", [(7, 6, 5), (33, 9, 12), (130, 70, 20), (257, 40, 10), (520, 18, 7)])
def test_ragged_and_tiny_lattices_from_identical_populations(pkg, orc, Lx, Lz, steps, variant):
    """Same starting populations on both sides (uploaded), odd sizes: minimum lattice, ragged block tails,
    lattices where every row is a wall row, several blocks per row -- with the automatic kernel choice (one step
    per launch at these sizes) and with the two-step kernel forced (strips narrower than 56 columns, odd widths,
    an odd last step)."""
    rng = np.random.default_rng(Lx * 1000 + Lz)
    rho = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx)); T = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx))
    ux = 0.03 * rng.uniform(-1, 1, (Lz, Lx)); uz = 0.03 * rng.uniform(-1, 1, (Lz, Lx))
    f0 = orc.init_equilibrium(rho, ux, uz, T) * (1 + 0.01 * rng.uniform(-1, 1, (37, Lz, Lx)))
    import torch
    lat = pkg.Lattice(Lx, Lz, 0.63, 2e-4)
    lat.set_variant(variant)
    lat.set_populations(torch.from_numpy(f0))                 # host path
    assert np.array_equal(lat.get_populations(host=True).numpy(), f0)   # layout round trip is bit exact
    lat.step(steps)
    got = lat.get_populations().cpu().numpy()                 # device path
    ref = orc.step(f0, 0.63, 2e-4, nsteps=steps)
    assert _rel(got, ref) < POP_RTOL
    lat.close()


def test_single_step_walls_and_wrap_exact_structure(pkg, orc):
    """One step from a state where every (l, i, k) value is distinct: any wrong source index (wrap,
    wall mirror, opposite population) changes the result at O(1), far above rounding."""
    Lx, Lz = 19, 11
    l, k, i = np.meshgrid(np.arange(37), np.arange(Lz), np.arange(Lx), indexing="ij")
    f0 = orc.feq(1.0, 0.0, 0.0, 1.0)[:, None, None] * (1 + 0.3 * np.sin(1.0 + 0.7 * l + 1.3 * k + 2.1 * i))
    import torch
    lat = pkg.Lattice(Lx, Lz, 0.9, 1e-3)
    lat.set_populations(torch.from_numpy(f0).cuda())
    lat.step(1)
    got = lat.get_populations(host=True).numpy()
    assert _rel(got, orc.step(f0, 0.9, 1e-3, nsteps=1)) < 1e-13
    lat.close()


def test_init_equilibrium_moments_and_widths(pkg, orc):
    import torch
    Lx, Lz, g = 96, 80, 1e-4
    rho, ux, uz, T = si.sweep_fields(Lx, Lz, seed=3)
    z = np.arange(Lz)[:, None]
    T = T + 0.05 * np.tanh((z - 40) / 6.0) * -1.0            # a front so that the widths are not trivial
    lat = pkg.Lattice(Lx, Lz, 0.8, g)
    lat.init_equilibrium(*[torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (rho, ux, uz, T)])
    f0 = orc.init_equilibrium(rho, ux, uz, T)
    assert _rel(lat.get_populations(host=True).numpy(), f0) < 1e-13
    lat.step(3)
    ref = orc.step(f0, 0.8, g, nsteps=3)
    m = [x.cpu().numpy() for x in lat.moments()]
    mo = orc.moments(ref, g)
    assert np.max(np.abs(m[0] - mo[0])) < 1e-13 and np.max(np.abs(m[3] - mo[3])) < 1e-13
    assert np.max(np.abs(m[1] - mo[1])) < 1e-14 and np.max(np.abs(m[2] - mo[2])) < 1e-14
    # kinetic moments (eq. 7, no half-force shift) = the oracle's moments at g = 0; fed back through
    # init_equilibrium they reproduce themselves (what bench.py's end-to-end leg relies on)
    km = lat.kinetic_moments()
    ko = orc.moments(ref, 0.0)
    for a, b in zip(km, ko):
        assert np.max(np.abs(a.cpu().numpy() - b)) < 1e-13
    again = pkg.Lattice(Lx, Lz, 0.8, g)
    again.init_equilibrium(*km)
    for a, b in zip(again.kinetic_moments(), km):
        assert float((a - b).abs().max()) < 1e-13
    again.close()
    lu, ld, tbar = lat.mixing_widths(1.05, 1.0, 0.95)
    olu, old, otbar = orc.mixing_widths(ref, g, 1.05, 1.0, 0.95)
    assert np.max(np.abs(tbar - otbar)) < 1e-13 and abs(lu - olu) < 1e-10 and abs(ld - old) < 1e-10
    assert lu > 1 and ld > 1
    # only-T request leaves the other outputs untouched (null pointers are skipped)
    Tonly = torch.empty((Lz, Lx), dtype=torch.float64, device="cuda")
    lat.moments(T=Tonly, alloc=False)
    assert np.array_equal(Tonly.cpu().numpy(), m[3])
    lat.close()


def test_conservation_and_invariants_on_gpu(pkg):
    """Properties that hold at any size, on the CUDA path alone: mass and (without gravity) energy are
    conserved by walls + collision to rounding -- momentum is not, rigid walls absorb it -- and
    x-translation invariance is bit exact."""
    import torch
    Lx, Lz = 160, 96
    rho, ux, uz, T = [torch.from_numpy(x).cuda() for x in si.sweep_fields(Lx, Lz, seed=11)]
    lat = pkg.Lattice(Lx, Lz, 0.7, 0.0)
    lat.init_equilibrium(rho, ux, uz, T)
    t0 = lat.totals(); lat.step(50); t1 = lat.totals()
    assert abs(t1[0] / t0[0] - 1) < 1e-13 and abs(t1[3] / t0[3] - 1) < 1e-13
    a = lat.get_populations()
    lat2 = pkg.Lattice(Lx, Lz, 0.7, 0.0)
    lat2.init_equilibrium(*[torch.roll(x, 37, dims=1).contiguous() for x in (rho, ux, uz, T)])
    lat2.step(50)
    assert torch.equal(torch.roll(a, 37, dims=2), lat2.get_populations())
    lat.close(); lat2.close()


def test_run_host_end_to_end(pkg, orc):
    import torch
    Lx, Lz, g = 64, 48, 1e-4
    fields = si.sweep_fields(Lx, Lz, seed=2)
    lat = pkg.Lattice(Lx, Lz, 0.8, g)
    ins = [torch.from_numpy(x).pin_memory() for x in fields]
    outs = lat.run_host(*ins, n=4)
    ref = orc.moments(orc.step(orc.init_equilibrium(*fields), 0.8, g, nsteps=4), g)
    for o, r_ in zip(outs, ref):
        assert np.max(np.abs(o.numpy() - r_)) < 1e-13
    lat.close()


def test_section4_profiles_match_oracle(pkg, orc):
    """Fluctuation profiles of Fig. 8-9 (lbm_profiles) on an evolved RT state, row by row."""
    cfg = si.scaled(si.rt_config(2), 200, 96)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, 2e-3)       # strong gravity so that the half-step shifts matter
    lat.init_rt(5, **cfg.rt_args())
    lat.step(30)
    ref = orc.step(orc.init_rt(cfg.Lx, cfg.Lz, 2e-3, 5, **cfg.rt_args()), cfg.tau, 2e-3, nsteps=30)
    got, want = lat.profiles(), orc.profiles(ref, 2e-3)
    for a, b, tol in zip(got, want, (1e-13, 1e-12, 1e-16, 1e-15)):
        assert np.max(np.abs(a - b)) < tol
    assert want[1].max() > 1e-4 and want[3].max() > 1e-9      # the profiles are not trivially zero
    assert np.max(np.abs(got[0] - lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)[2])) < 1e-14
    lat.close()


def test_step_is_cuda_graph_capturable(pkg):
    """lbm_step only enqueues kernels on the given stream, so an even number of steps can be captured in a
    CUDA graph and replayed (the ping-pong returns to the same buffers)."""
    import torch
    Lx, Lz = 96, 64
    fields = [torch.from_numpy(x).cuda() for x in si.sweep_fields(Lx, Lz, seed=4)]
    a, b = pkg.Lattice(Lx, Lz, 0.8, 1e-4), pkg.Lattice(Lx, Lz, 0.8, 1e-4)
    a.init_equilibrium(*fields); b.init_equilibrium(*fields)
    a.step(10)                                            # 2 warm-up + 4 replays x 2; capture itself runs nothing
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        b.step(2, stream=s)                                   # warm-up outside capture
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            b.step(2, stream=s)
        for _ in range(4):
            graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


@pytest.mark.parametrize("Lx,Lz,zchunk,n", [(7, 6, 3, 4), (33, 9, 3, 5), (64, 128, 192, 6), (130, 70, 9, 7),
                                            (257, 40, 15, 4), (520, 18, 126, 2), (70, 64, 12, 10), (191, 37, 21, 3),
                                            (130, 70, 7, 4), (200, 50, 10, 6), (128, 31, 5, 2), (64, 20, 3, 2), (100, 12, 4, 4),
                                            (57, 6, 4, 2), (113, 7, 3, 6)])
@pytest.mark.parametrize("fused_variant", [3])
def test_two_step_kernel_is_bitwise_equal_to_single_steps(pkg, orc, Lx, Lz, zchunk, n, fused_variant):
    """Variant 3 fuses two time steps per launch through shared memory (lbm_step2s.cuh: TMA loader, producer and
    consumer warps, per-population ring depths, ghost rows).  It uses the same
    collide arithmetic, so the result must be bit-identical to n single steps (odd n: last step unfused) --
    for ragged strips, chunks that do not divide Lz, lattices made only of wall rows -- and within the oracle
    tolerance."""
    import torch
    rng = np.random.default_rng(Lx * 31 + Lz)
    rho = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx)); T = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx))
    ux = 0.03 * rng.uniform(-1, 1, (Lz, Lx)); uz = 0.03 * rng.uniform(-1, 1, (Lz, Lx))
    f0 = orc.init_equilibrium(rho, ux, uz, T) * (1 + 0.01 * rng.uniform(-1, 1, (37, Lz, Lx)))
    a, b = pkg.Lattice(Lx, Lz, 0.66, 3e-4), pkg.Lattice(Lx, Lz, 0.66, 3e-4)
    a.set_variant(1); b.set_variant(fused_variant); b.set_zchunk(zchunk)
    for lat in (a, b):
        lat.set_populations(torch.from_numpy(f0).cuda())
        lat.step(n)
    fa, fb = a.get_populations(), b.get_populations()
    assert b.steps_done == n and torch.equal(fa, fb)
    for bad in (1, 2, -3):                      # chunks must be at least as tall as the wall zone
        with pytest.raises(pkg.LbmError):
            b.set_zchunk(bad)
    assert _rel(fb.cpu().numpy(), orc.step(f0, 0.66, 3e-4, nsteps=n)) < POP_RTOL
    a.close(); b.close()


def test_fp64_peak_probe_is_plausible(pkg):
    """lbm_fp64_peak (DFMA chains on all SMs) backs the FP64 side of the roofline in bench.py: B200 is specified
    at 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s; anything far off means a broken probe or a throttled GPU."""
    v = max(pkg.fp64_peak() for _ in range(3))
    assert 15.0 < v < 45.0, v


@pytest.mark.parametrize("tau,g", [(0.51, 0.0), (2.0, 1e-3), (0.8, 0.0)])
def test_two_step_kernel_parameter_extremes_against_oracle(pkg, orc, tau, g):
    """Relaxation close to the stability limit, over-relaxation, no gravity: 30 steps of the two-step kernel on a
    lattice with a ragged strip (300 = 5 x 56 + 20) and chunk tail, every population against the oracle."""
    import torch
    Lx, Lz = 300, 100
    rng = np.random.default_rng(77)
    rho = 1 + 0.02 * rng.uniform(-1, 1, (Lz, Lx)); T = 1 + 0.02 * rng.uniform(-1, 1, (Lz, Lx))
    ux = 0.01 * rng.uniform(-1, 1, (Lz, Lx)); uz = 0.01 * rng.uniform(-1, 1, (Lz, Lx))
    f0 = orc.init_equilibrium(rho, ux, uz, T)
    lat = pkg.Lattice(Lx, Lz, tau, g)
    lat.set_variant(3); lat.set_zchunk(28)
    lat.set_populations(torch.from_numpy(f0).cuda())
    lat.step(30)
    got = lat.get_populations(host=True).numpy()
    ref = orc.step(f0, tau, g, nsteps=30)
    assert _rel(got, ref) < POP_RTOL
    tg, tr = lat.totals(), orc.totals(ref)
    assert abs(tg[0] / tr[0] - 1) < TOT_RTOL and abs(tg[3] / tr[3] - 1) < TOT_RTOL
    lat.close()
