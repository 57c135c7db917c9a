"""GPU parity for the SURVEY 8(f) rows: isothermal no-slip walls (wall_kind 1, reading 19), in-place streaming with
one lattice copy, z-slabs with exchanged ghost rows -- each against the CPU oracle element by element (1e-11) and,
where the arithmetic is the same, bit for bit against the two-copy whole-lattice path.  Run on the B200 box."""
import numpy as np
import pytest

import synthetic_inputs as si

pytestmark = pytest.mark.gpu
POP_RTOL = 1e-11


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


def _random_state(orc, Lx, Lz, seed):
    rng = np.random.default_rng(seed)
    rho = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx)); T = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx))
    ux = 0.03 * rng.uniform(-1, 1, (Lz, Lx)); uz = 0.03 * rng.uniform(-1, 1, (Lz, Lx))
    return orc.init_equilibrium(rho, ux, uz, T) * (1 + 0.01 * rng.uniform(-1, 1, (37, Lz, Lx)))


# ------------------------------------------------------------------------------------------ isothermal walls
@pytest.mark.parametrize("variant", [0, 1, 2, 3])
def test_isothermal_walls_config1_100_steps(pkg, orc, variant):
    """BASELINE.json configs[0] with wall_kind 1 (walls at T_d below, T_u above): 100 steps, all populations."""
    cfg = si.rt_config(1)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, wall_kind=1, T_wall=(cfg.T_d, cfg.T_u))
    lat.set_variant(variant)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    lat.step(100)
    got = lat.get_populations(host=True).numpy()
    f0 = orc.init_rt(cfg.Lx, cfg.Lz, cfg.g, si.DEFAULT_SEED, **cfg.rt_args())
    ref = orc.step(f0, cfg.tau, cfg.g, nsteps=100, wall_kind=1, T_bot=cfg.T_d, T_top=cfg.T_u)
    assert _rel(got, ref) < POP_RTOL
    assert _rel(got, orc.step(f0, cfg.tau, cfg.g, nsteps=100)) > 1e-6        # and it is not the bounce-back result
    _, ux, uz, T = [x.cpu().numpy() for x in lat.moments()]
    assert np.abs(uz[:3]).max() < 1e-15 and np.abs(T[:3] - cfg.T_d).max() < 1e-14 and np.abs(T[-3:] - cfg.T_u).max() < 1e-14
    tg, tr = lat.totals(), orc.totals(ref)
    assert abs(tg[0] / tr[0] - 1) < 1e-12 and abs(tg[3] / tr[3] - 1) < 1e-12
    lat.close()


@pytest.mark.parametrize("Lx,Lz,zchunk,n", [(7, 6, 3, 4), (33, 9, 3, 5), (130, 70, 9, 7), (257, 40, 15, 4), (300, 100, 28, 12)])
def test_isothermal_walls_two_step_kernel_ragged(pkg, orc, Lx, Lz, zchunk, n):
    """wall_kind 1 in the two-step kernel (producer wall rows of the first step, consumer wall rows of the second):
    lattices made only of wall rows, ragged strips, chunk tails; bitwise equal to the one-step kernel, and within
    the oracle tolerance."""
    import torch
    f0 = _random_state(orc, Lx, Lz, Lx * 7 + Lz)
    a = pkg.Lattice(Lx, Lz, 0.66, 3e-4, wall_kind=1, T_wall=(1.03, 0.96))
    b = pkg.Lattice(Lx, Lz, 0.66, 3e-4, wall_kind=1, T_wall=(1.03, 0.96))
    a.set_variant(1); b.set_variant(3); b.set_zchunk(zchunk)
    for lat in (a, b):
        lat.set_populations(torch.from_numpy(f0).cuda())
        lat.step(n)
    assert torch.equal(a.get_populations(), b.get_populations())
    ref = orc.step(f0, 0.66, 3e-4, nsteps=n, wall_kind=1, T_bot=1.03, T_top=0.96)
    assert _rel(b.get_populations(host=True).numpy(), ref) < POP_RTOL
    a.close(); b.close()


# ------------------------------------------------------------------------------------------ in-place streaming
@pytest.mark.parametrize("wall_kind", [0, 1])
@pytest.mark.parametrize("Lx,Lz", [(7, 6), (33, 9), (130, 70), (257, 40)])
def test_inplace_streaming_matches_oracle_after_every_step(pkg, orc, Lx, Lz, wall_kind):
    """One lattice copy: after an odd number of steps the store is in the shifted layout, after an even number in
    the ordinary one; lbm_get_populations, lbm_moments and the row diagnostics read either.  Every step 1..6 against
    the oracle, and bit for bit against the two-copy path."""
    import torch
    f0 = _random_state(orc, Lx, Lz, Lx + 13 * Lz)
    kw = dict(wall_kind=wall_kind, T_wall=(1.02, 0.97))
    one, two = pkg.Lattice(Lx, Lz, 0.7, 2e-4, inplace=True, **kw), pkg.Lattice(Lx, Lz, 0.7, 2e-4, **kw)
    two.set_variant(1)
    for lat in (one, two):
        lat.set_populations(torch.from_numpy(f0).cuda())
    ref = f0
    for n in range(1, 7):
        one.step(1); two.step(1)
        ref = orc.step(ref, 0.7, 2e-4, nsteps=1, wall_kind=wall_kind, T_bot=1.02, T_top=0.97)
        got = one.get_populations()
        assert torch.equal(got, two.get_populations()), n
        assert _rel(got.cpu().numpy(), ref) < POP_RTOL
        assert np.array_equal(one.get_populations(host=True).numpy(), got.cpu().numpy())     # plane-by-plane host path
        for x, y in zip(one.moments(), two.moments()):
            assert torch.equal(x, y)
        assert np.array_equal(one.totals(), two.totals())
    with pytest.raises(pkg.LbmError):
        one.set_variant(3); one.step(2)                      # the two-step kernel needs two copies
    one.close(); two.close()


def test_inplace_streaming_config1_100_steps_and_host_upload(pkg, orc):
    cfg = si.rt_config(1)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g, inplace=True)
    lat.init_rt(si.DEFAULT_SEED, **cfg.rt_args())
    lat.step(99)                                              # ends in the shifted layout
    f0 = orc.init_rt(cfg.Lx, cfg.Lz, cfg.g, si.DEFAULT_SEED, **cfg.rt_args())
    assert _rel(lat.get_populations(host=True).numpy(), orc.step(f0, cfg.tau, cfg.g, nsteps=99)) < POP_RTOL
    lu, ld, tbar = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    olu, old, otbar = orc.mixing_widths(orc.step(f0, cfg.tau, cfg.g, nsteps=99), cfg.g, cfg.T_d, cfg.T_m, cfg.T_u)
    assert np.max(np.abs(tbar - otbar)) < 1e-13 and abs(lu - olu) < 1e-10 and abs(ld - old) < 1e-10
    import torch
    lat.set_populations(torch.from_numpy(f0))                 # host upload resets to the ordinary layout
    lat.step(2)
    assert _rel(lat.get_populations(host=True).numpy(), orc.step(f0, cfg.tau, cfg.g, nsteps=2)) < POP_RTOL
    lat.close()


# ------------------------------------------------------------------------------------------ z-slabs
def _run_slabs(pkg, slabs, nsteps, exchange_stream=None):
    """Steps slabs that live on one device: messages are packed on the exchange stream, copied device to device and
    unpacked there while the interior rows run on the main stream (the exchange hides behind the
    bulk), then the edge rows."""
    import torch
    main = torch.cuda.current_stream()
    xs = exchange_stream or torch.cuda.Stream()
    up = [s.new_message() for s in slabs]      # message of slab i to the slab above
    dn = [s.new_message() for s in slabs]
    from_below = [s.new_message() for s in slabs]   # receive buffers
    from_above = [s.new_message() for s in slabs]
    for _ in range(nsteps):
        xs.wait_stream(main)
        with torch.cuda.stream(xs):
            for i, s in enumerate(slabs):
                if s.open_above: s.pack(1, up[i], stream=xs)
                if s.open_below: s.pack(0, dn[i], stream=xs)
        for s in slabs:
            s.step_part(pkg.Slab.INTERIOR, stream=main)
        with torch.cuda.stream(xs):
            for i, s in enumerate(slabs):                     # "transport": device-to-device copies (cudaMemcpyAsync)
                if s.open_below: from_below[i].copy_(up[i - 1], non_blocking=True); s.unpack(0, from_below[i], stream=xs)
                if s.open_above: from_above[i].copy_(dn[i + 1], non_blocking=True); s.unpack(1, from_above[i], stream=xs)
        main.wait_stream(xs)
        for s in slabs:
            s.step_part(pkg.Slab.EDGES, stream=main)
    torch.cuda.synchronize()


@pytest.mark.parametrize("wall_kind", [0, 1])
@pytest.mark.parametrize("Lx,Lz,cuts,n", [(64, 128, (0, 50, 128), 100), (130, 70, (0, 6, 30, 64, 70), 25), (33, 40, (0, 17, 40), 9)])
def test_slabs_with_exchanged_ghost_rows_equal_the_whole_lattice(pkg, orc, Lx, Lz, cuts, n, wall_kind):
    """The lattice cut into z-slabs (down to the minimum of 6 rows), 26 population-rows exchanged per open side and
    step: bit-identical to the whole-lattice run, and within the oracle tolerance."""
    import torch
    f0 = _random_state(orc, Lx, Lz, 5 * Lx + Lz)
    kw = dict(wall_kind=wall_kind, T_wall=(1.02, 0.97))
    whole = pkg.Lattice(Lx, Lz, 0.75, 2e-4, **kw)
    whole.set_variant(1)
    whole.set_populations(torch.from_numpy(f0).cuda())
    whole.step(n)
    slabs = [pkg.Slab(Lx, Lz, z0, z1 - z0, 0.75, 2e-4, **kw) for z0, z1 in zip(cuts[:-1], cuts[1:])]
    for s in slabs:
        s.set_populations(torch.from_numpy(np.ascontiguousarray(f0[:, s.z0:s.z0 + s.nz])).cuda())
    _run_slabs(pkg, slabs, n)
    got = torch.cat([s.get_populations() for s in slabs], dim=1)
    assert torch.equal(got, whole.get_populations())
    ref = orc.step(f0, 0.75, 2e-4, nsteps=n, wall_kind=wall_kind, T_bot=1.02, T_top=0.97)
    assert _rel(got.cpu().numpy(), ref) < POP_RTOL
    assert abs(sum(s.totals()[0] for s in slabs) / whole.totals()[0] - 1) < 1e-14       # partial sums add up
    with pytest.raises(pkg.LbmError):
        slabs[0].pack(0, slabs[0].new_message())                                          # side 0 of the bottom slab is a wall
    with pytest.raises(pkg.LbmError):
        slabs[0].step_part(pkg.Slab.EDGES)                                                # interior first
    for s in slabs:
        s.close()
    whole.close()


def _run_slabs_fused(pkg, slabs, npairs, parts=False):
    """Pairs of steps with the two-step kernel: whole 6-row messages, device-to-device copies.  parts = False: one
    stream, lbm_slab_step2 after the exchange; parts = True: interior rows on the main stream while the messages are
    copied and unpacked on a second stream, then the edge rows (lbm_slab_step2_part)."""
    import torch
    up, dn, below, above = ([s.new_message(True) for s in slabs] for _ in range(4))
    main = torch.cuda.current_stream()
    xs = torch.cuda.Stream() if parts else main
    for _ in range(npairs):
        xs.wait_stream(main)
        for i, s in enumerate(slabs):
            if s.open_above: s.pack2(1, up[i], stream=xs)
            if s.open_below: s.pack2(0, dn[i], stream=xs)
        if parts:
            main.wait_stream(xs)
            for s in slabs:
                s.step2_part(pkg.Slab.INTERIOR, stream=main)
        with torch.cuda.stream(xs):
            for i, s in enumerate(slabs):
                if s.open_below: below[i].copy_(up[i - 1], non_blocking=True); s.unpack2(0, below[i], stream=xs)
                if s.open_above: above[i].copy_(dn[i + 1], non_blocking=True); s.unpack2(1, above[i], stream=xs)
        main.wait_stream(xs)
        for s in slabs:
            if parts: s.step2_part(pkg.Slab.EDGES, stream=main)
            else: s.step2(stream=main)
    torch.cuda.synchronize()


@pytest.mark.parametrize("parts", [False, True])
@pytest.mark.parametrize("wall_kind", [0, 1])
@pytest.mark.parametrize("Lx,Lz,cuts,n", [(64, 128, (0, 50, 128), 21), (130, 70, (0, 6, 30, 64, 70), 11), (33, 40, (0, 17, 40), 9),
                                          (600, 300, (0, 100, 207, 300), 14)])
def test_slabs_with_the_two_step_kernel_equal_the_whole_lattice(pkg, orc, Lx, Lz, cuts, n, wall_kind, parts):
    """z-slabs stepped two steps at a time (lbm_slab_pack2 / unpack2 / step2: 6 whole ghost rows with wrap columns), an
    odd last step with the one-step slab path: bit-identical to the whole lattice, within the oracle tolerance; slabs
    down to 6 rows, several strips, both wall kinds."""
    import torch
    f0 = _random_state(orc, Lx, Lz, 3 * Lx + 7 * Lz)
    kw = dict(wall_kind=wall_kind, T_wall=(1.02, 0.97))
    whole = pkg.Lattice(Lx, Lz, 0.75, 2e-4, **kw)
    whole.set_variant(1)
    whole.set_populations(torch.from_numpy(f0).cuda())
    whole.step(n)
    slabs = [pkg.Slab(Lx, Lz, z0, z1 - z0, 0.75, 2e-4, **kw) for z0, z1 in zip(cuts[:-1], cuts[1:])]
    for s in slabs:
        s.set_populations(torch.from_numpy(np.ascontiguousarray(f0[:, s.z0:s.z0 + s.nz])).cuda())
    _run_slabs_fused(pkg, slabs, n // 2, parts=parts)
    _run_slabs(pkg, slabs, n % 2)
    got = torch.cat([s.get_populations() for s in slabs], dim=1)
    assert torch.equal(got, whole.get_populations())
    ref = orc.step(f0, 0.75, 2e-4, nsteps=n, wall_kind=wall_kind, T_bot=1.02, T_top=0.97)
    assert _rel(got.cpu().numpy(), ref) < POP_RTOL
    for s in slabs:
        s.close()
    whole.close()


def test_slabs_rt_config_init_and_widths(pkg, orc):
    """lbm_init_rt on slabs uses global heights and fills the ghost rows; the mixing widths are partial sums."""
    cfg = si.scaled(si.rt_config(2), 128, 256)
    whole = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    whole.set_variant(1)
    whole.init_rt(7, **cfg.rt_args())
    slabs = [pkg.Slab(cfg.Lx, cfg.Lz, z0, nz, cfg.tau, cfg.g) for z0, nz in ((0, 100), (100, 60), (160, 96))]
    for s in slabs:
        s.init_rt(7, **cfg.rt_args())
    import torch
    assert torch.equal(torch.cat([s.get_populations() for s in slabs], dim=1), whole.get_populations())
    whole.step(40)
    _run_slabs(pkg, slabs, 40)
    assert torch.equal(torch.cat([s.get_populations() for s in slabs], dim=1), whole.get_populations())
    lu, ld, tbar = whole.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    parts = [s.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u) for s in slabs]
    assert abs(sum(p[0] for p in parts) - lu) < 1e-12 and abs(sum(p[1] for p in parts) - ld) < 1e-12
    assert np.array_equal(np.concatenate([p[2] for p in parts]), tbar)
    for s in slabs:
        s.close()
    whole.close()


# ------------------------------------------------------------------------------------------ boundary behaviour
def test_fused_diagnostics_equal_the_single_calls_and_null_moments_are_rejected(pkg):
    cfg = si.scaled(si.rt_config(2), 200, 96)
    lat = pkg.Lattice(cfg.Lx, cfg.Lz, cfg.tau, cfg.g)
    lat.init_rt(5, **cfg.rt_args())
    lat.step(20)
    d = lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u)
    lu, ld, tbar = lat.mixing_widths(cfg.T_d, cfg.T_m, cfg.T_u)
    prof = lat.profiles()
    assert d["L_u"] == lu and d["L_d"] == ld and np.array_equal(d["totals"], lat.totals())
    for key, want in zip(("Tbar", "Trms", "Ekbar", "Ekrms"), prof):
        assert np.array_equal(d[key], want)
    assert np.array_equal(tbar, prof[0])
    l0 = lat.kernel_launches
    lat.diagnostics(cfg.T_d, cfg.T_m, cfg.T_u)
    assert lat.kernel_launches - l0 == 2                      # one pass over the lattice + one small block
    with pytest.raises(pkg.LbmError):
        lat.moments(alloc=False)                              # all four outputs null
    at, tau_rt = pkg.rt_scales(cfg.Lx, cfg.g, cfg.T_d, cfg.T_u)
    assert abs(at - (cfg.T_d - cfg.T_u) / (cfg.T_d + cfg.T_u)) < 1e-16 and abs(tau_rt - (cfg.Lx / (cfg.g * at)) ** 0.5) < 1e-9
    lat.close()


def test_graph_capture_of_the_two_step_kernel_and_odd_launch_counts(pkg):
    """lbm_step under stream capture on a lattice that takes the fused path (tensor maps as __grid_constant__
    kernel arguments, the shared-memory opt-in): 4 steps = 2 launches are captured and replayed; 2 steps = 1 launch
    would leave the other copy current and are rejected, as are 3 one-step launches."""
    import torch
    Lx, Lz = 512, 1024
    fields = [x for x in si.sweep_fields_torch(Lx, Lz, 4, "cuda")]
    a, b = pkg.Lattice(Lx, Lz, 0.8, 1e-4), pkg.Lattice(Lx, Lz, 0.8, 1e-4)
    assert b.plan()[0]
    a.init_equilibrium(*fields); b.init_equilibrium(*fields)
    a.step(4 + 3 * 4)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        b.step(4, stream=s)                                   # warm-up outside capture
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            b.step(4, stream=s)
            with pytest.raises(pkg.LbmError):
                b.step(2, stream=s)                           # one fused launch: odd
        for _ in range(3):
            graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


def test_a_captured_fused_step_can_be_replayed_after_the_lattice_is_reinitialised(pkg):
    """a graph captured while the wrap columns of the current copy were valid must still refresh them at
    replay, because lbm_init_* / lbm_set_populations between replays rewrite the lattice without its periodic images."""
    import torch
    Lx, Lz = 512, 1024
    f1 = si.sweep_fields_torch(Lx, Lz, 4, "cuda")
    f2 = si.sweep_fields_torch(Lx, Lz, 5, "cuda")
    a, b = pkg.Lattice(Lx, Lz, 0.8, 1e-4), pkg.Lattice(Lx, Lz, 0.8, 1e-4)
    assert b.plan()[0]
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        b.init_equilibrium(*f1, stream=s)
        b.step(4, stream=s)                                   # leaves wrap_ok set for the current copy
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            b.step(4, stream=s)
        b.init_equilibrium(*f2, stream=s)                     # new contents, stale wrap columns
        graph.replay()
    torch.cuda.synchronize()
    a.init_equilibrium(*f2)
    a.step(4)
    assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


def test_boundary_refusals_from_the_round2_review(pkg):
    """ADVICE r2 / VERDICT r2 7(d): host copies of a slab whose step is half done are refused (they stage through the
    copy that already holds the interior rows); forcing the two-step kernel on a one-copy handle is an argument error."""
    import ctypes as C
    import torch
    sl = pkg.Slab(64, 128, 32, 40, 0.8, 1e-4)
    sl.init_equilibrium(*[x[32:72].contiguous() for x in si.sweep_fields_torch(64, 128, 3, "cuda")])
    before = sl.get_populations(host=True)
    sl.step_part(pkg.Slab.INTERIOR)
    with pytest.raises(pkg.LbmError):
        sl.get_populations(host=True)
    with pytest.raises(pkg.LbmError):
        sl.set_populations(before)
    sl.step_part(pkg.Slab.EDGES)
    sl.get_populations(host=True)                                # whole steps: fine again
    sl.close()
    lat = pkg.Lattice(64, 128, 0.8, 1e-4, inplace=True)
    lat.set_variant(3)
    assert lat._lib.lbm_step(lat._h, 2, C.c_void_p(torch.cuda.current_stream().cuda_stream)) == -1
    lat.close()


def test_persistent_kernel_barrier_counter_crosses_the_32_bit_wrap(pkg):
    """the grid barrier of the persistent kernel counts arrivals in 32 bits.  The counter now starts every
    launch at 0xFFFFFFFF, so the very first barrier crosses the wrap; 200 steps in one launch against 200 launched
    steps, bit for bit, on both block sizes of that kernel (64x128 -> 64-thread blocks, 150x200 -> 128)."""
    import torch
    for Lx, Lz in ((64, 128), (150, 200)):
        fields = si.sweep_fields_torch(Lx, Lz, 11, "cuda")
        a, b = pkg.Lattice(Lx, Lz, 0.8, 1e-4), pkg.Lattice(Lx, Lz, 0.8, 1e-4)
        a.set_variant(1)
        a.init_equilibrium(*fields); b.init_equilibrium(*fields)
        n0 = b.kernel_launches
        a.step(200); b.step(200)
        assert b.kernel_launches - n0 == 1                       # the persistent path really ran
        assert torch.equal(a.get_populations(), b.get_populations())
        a.close(); b.close()


def test_two_step_kernel_soak_on_an_l2_resident_lattice(pkg):
    """the stage hand-off (generic-proxy reads, then the TMA unit rewrites the buffer) is most exposed when
    the source rows come from L2 and the boxes land fast: 256x512 (both copies L2-resident), two-step kernel forced,
    3000 steps in batches, compared bit for bit with the one-step kernel after every batch."""
    import torch
    Lx, Lz = 256, 512
    fields = si.sweep_fields_torch(Lx, Lz, 9, "cuda")
    a, b = pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G), pkg.Lattice(Lx, Lz, si.SWEEP_TAU, si.SWEEP_G)
    a.set_variant(1); b.set_variant(3)
    assert b.plan()[0]
    for lat in (a, b):
        lat.init_equilibrium(*fields)
    for _ in range(6):
        a.step(500); b.step(500)
        assert torch.equal(a.get_populations(), b.get_populations())
    a.close(); b.close()


def test_a_handle_rejects_calls_from_another_device(pkg):
    """a handle belongs to the device that was current in lbm_create (the shared-memory opt-in, the tensor
    maps and the scratch live there); with another device current every device call is refused.  Needs two GPUs."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    lat0 = pkg.Lattice(512, 1024, 0.8, 1e-4, device="cuda:0")
    lat1 = pkg.Lattice(512, 1024, 0.8, 1e-4, device="cuda:1")
    cfg = si.rt_config(2)
    for lat in (lat0, lat1):
        lat.init_rt(1, **cfg.rt_args())
        lat.step(4)                                           # the fused path on both devices
    assert torch.equal(lat0.get_populations().cpu(), lat1.get_populations().cpu())
    import ctypes as C
    with torch.cuda.device(0):                                # the raw call, bypassing the binding's device guard
        rc = lat1._lib.lbm_step(lat1._h, 2, C.c_void_p(0))
    assert rc == -1
    lat0.close(); lat1.close()
