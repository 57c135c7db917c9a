"""Pins for the oracle's section-IV observables: fluctuation profiles (Fig. 8-9) and growth rate (eq. 11, 14)."""
import math

import numpy as np


def test_fluctuation_profiles_closed_form(orc):
    """Rows modulated by a cosine: T = Tm_k + A_k cos(phi), E_k = E0_k (1 + a_k cos(phi)), so the x-rms values
    are |A_k|/sqrt2 and E0_k |a_k|/sqrt2 exactly, including the half-step shifts of
    PAPER.md:94 (fields are given as hydrodynamic values and converted to the stored kinetic ones)."""
    Lx, Lz, g = 48, 9, 2e-3
    k = np.arange(Lz)[:, None]
    phi = 2 * math.pi * 3 * np.arange(Lx)[None, :] / Lx
    Tm, A = 1.0 + 0.01 * k, 0.002 * (k + 1)
    E0, a = 1e-4 * (1 + k), 0.1 + 0.05 * k
    rho = 1.0 + 0.03 * np.sin(phi + k)
    T_h = Tm + A * np.cos(phi)
    Ek = E0 * (1 + a * np.cos(phi))
    speed = np.sqrt(2 * Ek / rho)
    ang = 0.7 + 0.3 * k + 0.0 * phi
    ux_h, uz_h = speed * np.cos(ang), speed * np.sin(ang)
    f = orc.init_equilibrium(rho, ux_h, uz_h - g / 2, T_h - g * g / 8)      # stored kinetic fields (reading 8)
    Tbar, Trms, Ekbar, Ekrms = orc.profiles(f, g)
    assert np.max(np.abs(Tbar - Tm[:, 0])) < 1e-14 and np.max(np.abs(Trms - A[:, 0] / math.sqrt(2))) < 1e-14
    assert np.max(np.abs(Ekbar - E0[:, 0])) < 1e-16 and np.max(np.abs(Ekrms - (E0 * a)[:, 0] / math.sqrt(2))) < 1e-16
    # consistent with the Tbar of the mixing-width routine
    assert np.max(np.abs(orc.mixing_widths(f, g, 1.05, 1.0, 0.95)[2] - Tbar)) < 1e-15


def test_growth_rate_recovers_alpha_on_the_quadratic_law(orc):
    """L = alpha g At t^2 (eq. 10): the centred difference of t^2 is exact, so alpha comes back
    to rounding at interior points; eq. 14: alpha_tot = (alpha_u At_u + alpha_d At_d)/At."""
    g, Tu, Tm, Td = 1.5e-5, 0.975, 1.0, 1.025                 # Table II
    At, At_u, At_d = (Td - Tu) / (Td + Tu), (Tm - Tu) / (Tm + Tu), (Td - Tm) / (Td + Tm)
    t = np.arange(1, 40) * 250.0
    alpha = 0.04
    L = alpha * g * At * t ** 2
    got = orc.growth_rate(t, L, g, At)
    assert np.max(np.abs(got[1:-1] / alpha - 1)) < 1e-12
    # one-sided ends: the two-point difference of t^2 is t_a + t_b, so alpha is off by a known factor
    assert abs(got[0] / (alpha * (t[0] + t[1]) ** 2 / (4 * t[0] ** 2)) - 1) < 1e-12
    assert abs(got[-1] / (alpha * (t[-1] + t[-2]) ** 2 / (4 * t[-1] ** 2)) - 1) < 1e-12
    au, ad = 0.03, 0.05
    Ltot = au * g * At_u * t ** 2 + ad * g * At_d * t ** 2
    tot = orc.growth_rate(t, Ltot, g, At)
    assert np.max(np.abs(tot[1:-1] - (au * At_u + ad * At_d) / At)) < 1e-12
    # non-uniform sampling and zero length
    t2 = np.array([0.0, 10.0, 30.0, 35.0])
    assert orc.growth_rate(t2, 2.0 * t2, 1.0, 0.5)[0] == 0.0
    assert abs(orc.growth_rate(t2, 2.0 * t2, 1.0, 0.5)[2] - 4.0 / (4 * 0.5 * 60.0)) < 1e-15
