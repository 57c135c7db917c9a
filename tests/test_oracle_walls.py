"""Pins for the oracle's isothermal no-slip wall rule, wall_kind = 1 (reading 19; PAPER.md:114 says only
that step bc "adjusts population values at sites with coordinates z = 0, 1, 2 and z = Lz-3, Lz-2, Lz-1" for "rigid
boundary conditions").  The rule is a reading; what pins it is what the words fix (three rows, the wall state imposed,
nothing else touched) and the physics the rule must reproduce: mass conservation, a rest fixed point, the location of
the no-slip planes, steady conduction with the bulk conductivity, a smaller hydrostatic wall layer than reading 9.
CPU only."""
import numpy as np
import pytest


def _perturbed_state(orc, rng, Lx, Lz):
    rho = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx)); T = 1 + 0.05 * rng.uniform(-1, 1, (Lz, Lx))
    ux = 0.03 * rng.uniform(-1, 1, (Lz, Lx)); uz = 0.03 * rng.uniform(-1, 1, (Lz, Lx))
    return orc.init_equilibrium(rho, ux, uz, T) * (1 + 0.01 * rng.uniform(-1, 1, (37, Lz, Lx)))


def test_bc_adjusts_exactly_the_three_rows_per_wall_and_imposes_the_wall_state(orc):
    """only rows 0..2 and Lz-3..Lz-1 change; on them the kinetic moments become (rho*, -g_vec/2,
    T_wall - g^2/8) -- the state PAPER.md:94 maps to u^(H) = 0, T^(H) = T_wall -- with the density and the
    non-equilibrium part of every population untouched (recomputed here in numpy from the oracle's f_eq)."""
    rng = np.random.default_rng(41)
    Lx, Lz, g, Tb, Tt = 7, 11, 2e-3, 1.04, 0.93
    fs = orc.propagate(_perturbed_state(orc, rng, Lx, Lz))
    out = orc.bc_isothermal(fs, g, Tb, Tt)
    assert np.array_equal(out[:, 3:-3], fs[:, 3:-3])
    for k in (0, 1, 2, Lz - 3, Lz - 2, Lz - 1):
        Tw = Tb if k < 3 else Tt
        for i in range(Lx):
            rho, ux, uz, T = orc.site_moments(fs[:, k, i])
            r2, ux2, uz2, T2 = orc.site_moments(out[:, k, i])
            assert abs(r2 - rho) < 2e-15 * rho and abs(ux2) < 1e-15 and abs(uz2 - 0.5 * g) < 1e-15
            assert abs(T2 - (Tw - g * g / 8)) < 2e-15
            neq_before = fs[:, k, i] - orc.feq(rho, ux, uz, T)
            neq_after = out[:, k, i] - orc.feq(rho, 0.0, 0.5 * g, Tw - g * g / 8)
            assert np.max(np.abs(neq_before - neq_after)) < 1e-16


def test_after_a_step_the_wall_rows_are_at_rest_at_the_wall_temperature_and_mass_is_conserved(orc):
    rng = np.random.default_rng(42)
    Lx, Lz, g, Tb, Tt = 12, 20, 1e-3, 1.05, 0.95
    f0 = _perturbed_state(orc, rng, Lx, Lz)
    f1 = orc.step(f0, 0.8, g, 1, wall_kind=1, T_bot=Tb, T_top=Tt)
    _, ux, uz, T = orc.moments(f1, g)                       # hydrodynamic fields of the stored state
    for rows, Tw in ((slice(0, 3), Tb), (slice(Lz - 3, Lz), Tt)):
        assert np.abs(ux[rows]).max() < 1e-15 and np.abs(uz[rows]).max() < 1e-15
        assert np.abs(T[rows] - Tw).max() < 4e-15
    assert np.abs(uz[3:-3]).max() > 1e-3                    # ... and only those rows
    f50 = orc.step(f0, 0.8, g, 50, wall_kind=1, T_bot=Tb, T_top=Tt)
    assert abs(f50.sum() / f0.sum() - 1) < 1e-14            # the equilibrium shift keeps the density of every site
    # with wall_kind 0 the same start gives different wall rows: the branch really is a different rule
    assert np.abs(orc.moments(orc.step(f0, 0.8, g, 1), g)[3][:3] - Tb).max() > 1e-3


def test_rest_state_at_the_wall_temperature_is_a_fixed_point(orc):
    Lx, Lz = 6, 14
    one, zero = np.ones((Lz, Lx)), np.zeros((Lz, Lx))
    f = orc.init_equilibrium(1.3 * one, zero, zero, 0.97 * one)
    f5 = orc.step(f, 0.8, 0.0, 5, wall_kind=1, T_bot=0.97, T_top=0.97)
    assert np.max(np.abs(f5 - f)) < 2e-15
    # a wall at another temperature is not a fixed point: the wall temperature really enters
    f5b = orc.step(f, 0.8, 0.0, 5, wall_kind=1, T_bot=1.0, T_top=0.97)
    assert np.max(np.abs(f5b - f)) > 1e-4


@pytest.mark.parametrize("Lz,nsteps", [(32, 800), (48, 1800)])
def test_no_slip_planes_sit_at_the_innermost_imposed_rows(orc, Lz, nsteps):
    """Slowest shear mode between the walls: u_x decays at nu (pi / H)^2 with nu = (tau - 1/2) T / r^2 (pinned in
    test_oracle_dynamics) and H the distance between the no-slip planes.  Velocity is imposed on rows 0..2 and
    Lz-3..Lz-1, so H is the distance between rows 2 and Lz-3, Lz - 5, to within half a site (measured: Lz - 5.3) --
    against H = Lz for the bounce-back rule of reading 9 (half a site outside rows 0 and Lz-1)."""
    Lx, tau = 4, 0.8
    _, _, _, r = orc.tables()
    k = np.arange(Lz)
    ux = 1e-3 * np.sin(np.pi * (k - 2) / (Lz - 5.0)).clip(0)[:, None] * np.ones((Lz, Lx))
    one, zero = np.ones((Lz, Lx)), np.zeros((Lz, Lx))
    f = orc.init_equilibrium(one, ux, zero, one)
    f = orc.step(f, tau, 0.0, nsteps // 2, wall_kind=1)
    a0 = orc.moments(f, 0.0)[1][Lz // 2, 0]
    f = orc.step(f, tau, 0.0, nsteps // 2, wall_kind=1)
    a1 = orc.moments(f, 0.0)[1][Lz // 2, 0]
    rate = np.log(a0 / a1) / (nsteps // 2)
    H = np.pi / np.sqrt(rate / ((tau - 0.5) / r ** 2))
    assert abs(H - (Lz - 5)) < 0.5, H


def test_steady_conduction_is_linear_and_carries_the_bulk_heat_flux(orc):
    """Walls at different temperatures, no gravity.  In the steady state the pressure is uniform, so the conductivity
    k = rho c_p kappa = c_p (tau - 1/2) p / r^2 (c_p = D/2 + 1 = 2; kappa = nu by Pr = 1, pinned in
    test_oracle_dynamics) is uniform and T(z) is linear away from the walls' kinetic layers; the energy that the wall
    adjustment injects per step at the bottom rows leaves at the top rows and equals k |dT/dz|."""
    Lx, Lz, tau, Tb, Tt = 4, 32, 0.9, 1.03, 0.97
    _, _, _, r = orc.tables()
    k = np.arange(Lz)
    T0 = (Tb + (Tt - Tb) * (k - 2) / (Lz - 5.0)).clip(Tt, Tb)[:, None] * np.ones((Lz, Lx))
    zero = np.zeros((Lz, Lx))
    f = orc.init_equilibrium(1.0 / T0, zero, zero, T0)
    f = orc.step(f, tau, 0.0, 4000, wall_kind=1, T_bot=Tb, T_top=Tt)
    rho, _, uz, T = orc.moments(f, 0.0)
    assert np.max(np.abs(orc.moments(orc.step(f, tau, 0.0, 200, wall_kind=1, T_bot=Tb, T_top=Tt), 0.0)[3] - T)) < 1e-10
    Tz = T[:, 0]
    assert np.abs(Tz[:3] - Tb).max() < 1e-14 and np.abs(Tz[-3:] - Tt).max() < 1e-14
    bulk = slice(10, Lz - 10)
    slope = np.polyfit(k[bulk], Tz[bulk], 1)[0]
    assert np.abs(np.diff(Tz[bulk], 2)).max() < 2e-3 * abs(slope)          # linear
    assert 0.95 < slope / ((Tt - Tb) / (Lz - 5.0)) <= 1.0                 # a small temperature jump at the walls
    # energy balance of the wall adjustment, per column and step
    fs = orc.propagate(f)
    adj = orc.bc_isothermal(fs, 0.0, Tb, Tt)

    def energy(pops):       # rho (T + |u|^2 / 2) = (1/2) sum |c|^2 f per site, D = 2
        m = np.array([orc.site_moments(pops[:, kk, 0]) for kk in range(Lz)])
        return m[:, 0] * (m[:, 3] + 0.5 * (m[:, 1] ** 2 + m[:, 2] ** 2))
    dE = energy(adj) - energy(fs)
    q_in, q_out = dE[:3].sum(), -dE[-3:].sum()
    p = float((rho * T)[bulk].mean())
    q_bulk = 2.0 * (tau - 0.5) * p / r ** 2 * abs(slope)
    assert abs(q_in / q_out - 1) < 1e-8
    assert abs(q_in / q_bulk - 1) < 5e-3, (q_in, q_bulk)


def test_hydrostatic_wall_layer_is_smaller_than_with_bounce_back(orc):
    """Single-temperature hydrostatic column (eq. 1): reading 9's bounce-back leaves a steady kinetic layer of
    ~0.05 g on the wall rows; with the wall state imposed the three rows are exactly at rest and the layer next to
    them stays below 0.01 g."""
    Lx, Lz, g, tau = 4, 96, 1e-4, 0.8
    f = orc.init_rt(Lx, Lz, g, 1, 1.0, 1.0, 1.0)
    uz0 = orc.moments(orc.step(f, tau, g, 100), g)[2]
    uz1 = orc.moments(orc.step(f, tau, g, 100, wall_kind=1, T_bot=1.0, T_top=1.0), g)[2]
    assert np.abs(uz0).max() > 0.03 * g
    assert np.abs(uz1[:3]).max() < 1e-15 and np.abs(uz1).max() < 0.01 * g
