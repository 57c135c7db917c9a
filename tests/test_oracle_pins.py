"""Pins for the CPU oracle: each test checks oracle/lbm_oracle.c against something the paper or the
mathematics fixes (never against the CUDA path, never against a retyped copy of its own formula).
All CPU, run with -m "not gpu".  Citations are PAPER.md lines."""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import hermite_e as He

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


# ----------------------------------------------------------------------------- velocity set / quadrature
def test_velocity_set_matches_paper(orc):
    gold = _golden("paper_constants.txt")
    ex, ez, w, r = orc.tables()
    assert len(ex) == int(gold["M"]) == 37
    assert len({(a, b) for a, b in zip(ex, ez)}) == 37
    assert max(np.abs(ex).max(), np.abs(ez).max()) == int(gold["H_x"])
    assert math.floor(r * 1e4) / 1e4 == gold["r"]                 # PAPER.md:100 (4 decimals, truncated)
    # canonical order: ascending e_z then e_x; opposite of l is 36 - l
    assert (ex[0], ez[0]) == (-1, -3) and (ex[18], ez[18]) == (0, 0) and (ex[36], ez[36]) == (1, 3)
    assert np.all(ex[::-1] == -ex) and np.all(ez[::-1] == -ez)
    keys = [(int(b), int(a)) for a, b in zip(ex, ez)]
    assert keys == sorted(keys)
    assert np.all(w > 0) and abs(w.sum() - 1.0) < 1e-15
    # weights depend on |e|^2 only (isotropy of the shells)
    for e2 in set(ex * ex + ez * ez):
        assert np.ptp(w[ex * ex + ez * ez == e2]) == 0.0


def test_quadrature_reproduces_gaussian_moments_to_degree_9(orc):
    """sum_l w_l c_x^a c_z^b = G_a G_b for EVERY a + b <= 9 (G_n = (n-1)!! for even n, 0 for odd):
    the degree of precision that M = 37 buys and that the 4th-order equilibrium needs."""
    ex, ez, w, r = orc.tables()
    cx, cz = r * ex, r * ez
    G = lambda n: 0.0 if n % 2 else float(np.prod(np.arange(n - 1, 0, -2))) if n else 1.0
    for a in range(10):
        for b in range(10 - a):
            got = float(np.sum(w * cx ** a * cz ** b))
            assert abs(got - G(a) * G(b)) < 2e-13 * max(1.0, G(a) * G(b)), (a, b, got)
    # and it is NOT exact at degree 10 -- guards against a trivially over-determined check
    assert abs(float(np.sum(w * cx ** 10)) - 945.0) > 1.0


# ----------------------------------------------------------------------------- equilibrium
def _rand_state(rng):
    return rng.uniform(0.5, 2.0), rng.uniform(-0.2, 0.2), rng.uniform(-0.2, 0.2), rng.uniform(0.8, 1.2)


def test_feq_moment_closure_eq7(orc):
    """eq. 7: the moments of f_eq(rho,u,T) are rho, u, T."""
    rng = np.random.default_rng(1)
    ex, ez, w, r = orc.tables()
    for _ in range(200):
        rho, ux, uz, T = _rand_state(rng)
        f = orc.feq(rho, ux, uz, T)
        assert abs(f.sum() - rho) < 4e-15 * rho
        assert abs((r * ex * f).sum() / rho - ux) < 4e-15
        assert abs((r * ez * f).sum() / rho - uz) < 4e-15
        e = (((r * ex - ux) ** 2 + (r * ez - uz) ** 2) * f).sum() / (2 * rho)
        assert abs(e - T) < 6e-15
        m = orc.site_moments(f)
        assert np.allclose(m, (rho, ux, uz, T), rtol=0, atol=6e-15)


def test_feq_higher_moments_of_maxwellian(orc):
    """Closed forms of a Maxwellian N(u, T) in D = 2: pressure tensor rho T delta, zero central heat
    flux, full third raw moment, and the 4th central trace D(D+2) rho T^2 (which an expansion
    truncated at 3rd order gets wrong)."""
    rng = np.random.default_rng(2)
    ex, ez, w, r = orc.tables()
    for _ in range(100):
        rho, ux, uz, T = _rand_state(rng)
        f = orc.feq(rho, ux, uz, T)
        dx, dz = r * ex - ux, r * ez - uz
        assert abs((dx * dx * f).sum() - rho * T) < 2e-14
        assert abs((dz * dz * f).sum() - rho * T) < 2e-14
        assert abs((dx * dz * f).sum()) < 2e-14
        d2 = dx * dx + dz * dz
        assert abs((d2 * dx * f).sum()) < 5e-14 and abs((d2 * dz * f).sum()) < 5e-14
        assert abs((d2 * d2 * f).sum() - 8.0 * rho * T * T) < 2e-13
        cx, cz = r * ex, r * ez
        assert abs((cx ** 3 * f).sum() - rho * (ux ** 3 + 3 * T * ux)) < 5e-14
        assert abs((cx * cx * cz * f).sum() - rho * (ux * ux * uz + T * uz)) < 5e-14


def test_feq_is_hermite_projection_of_continuous_maxwellian(orc):
    """Definition written out with library routines only: f_eq_l = w_l sum_{m+n<=4} a_mn He_m(c_lx)
    He_n(c_lz) / (m! n!), a_mn = rho E[He_m(X)] E[He_n(Z)], X ~ N(u_x, T), Z ~ N(u_z, T), the
    expectations taken by 40-point Gauss-Hermite quadrature of the CONTINUOUS Maxwellian
    (Hermite expansion of the local Maxwellian)."""
    rng = np.random.default_rng(3)
    ex, ez, w, r = orc.tables()
    y, wy = He.hermegauss(40)
    wy = wy / math.sqrt(2 * math.pi)
    unit = lambda n: np.eye(n + 1)[n]
    for _ in range(50):
        rho, ux, uz, T = _rand_state(rng)
        ax = [np.sum(wy * He.hermeval(ux + math.sqrt(T) * y, unit(n))) for n in range(5)]
        az = [np.sum(wy * He.hermeval(uz + math.sqrt(T) * y, unit(n))) for n in range(5)]
        ref = np.zeros(37)
        for m in range(5):
            for n in range(5 - m):
                ref += (rho * ax[m] * az[n] / (math.factorial(m) * math.factorial(n))
                        * He.hermeval(r * ex, unit(m)) * He.hermeval(r * ez, unit(n)))
        ref *= w
        assert np.max(np.abs(orc.feq(rho, ux, uz, T) - ref)) < 2e-15


def test_feq_positive_in_config_ranges(orc):
    rng = np.random.default_rng(4)
    for _ in range(200):
        f = orc.feq(rng.uniform(0.9, 1.1), rng.uniform(-0.05, 0.05), rng.uniform(-0.05, 0.05),
                    rng.uniform(0.94, 1.06))
        assert f.min() > 1e-4
