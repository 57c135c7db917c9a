/*
 * lbm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, loop-based CPU FP64 implementation of the per-time-step update of the
 * thermal D2Q37 Lattice-Boltzmann model of arxiv/paper_1405_1253, written from
 * the paper (and, where the paper is silent, from the readings listed in DESIGN.md /
 * SURVEY.md section 8(c)).  It shares no code, header, table or constant generator with the
 * CUDA path under paper_1405_1253_b200/.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 *
 * Parity status of each function (what pins it, see tests/test_oracle_pins.py):
 *   orc_tables             pinned: M = 37, max |e| = 3,
 *                                  r ~ 1.1969 (tests/golden/paper_constants.txt),
 *                                  Gaussian moment identities up to order 8, all w > 0, sum w = 1.
 *   orc_feq                pinned: eq. 7 closure, closed-form higher moments of the
 *                                  Maxwellian, independent Gauss-Hermite projection of the
 *                                  continuous Maxwellian (the "definition written out").
 *   orc_propagate          pinned: brute-force push-vs-pull, inverse round trip bitwise, mass
 *                                  multiset conservation with walls, x-translation invariance.
 *                                  The wall rule itself (half-way bounce-back) is a READING of
 *                                  "rigid boundary conditions": parity with the
 *                                  authors' wall scheme is UNPINNED (paper does not give it).
 *   orc_collide            pinned: conservation (g = 0), closed form (rho,u,T)->(rho,u+g,T) for
 *                                  g != 0, rest fixed point, shear-wave viscosity nu=(tau-1/2)T/r^2,
 *                                  thermal diffusivity with Pr = 1.
 *   orc_moments            pinned: by construction from eq. 7 + PAPER.md:94 and the hydrostatic
 *                                  rest test (bulk |u^(H)| <= 1e-10).
 *   orc_init_rt            pinned: T_d=T_m=T_u reduces to eq. 1 exactly; pressure continuity
 *                                  (eq. 2); discrete hydrostatic balance.  The tanh smoothing,
 *                                  geometry constants and the perturbation RNG are READINGS:
 *                                  parity with the authors' exact initial field is UNPINNED.
 *   orc_mixing_widths      pinned: closed form on step/tanh profiles (eq. 8, 9, 12).
 *   orc_bc_isothermal      pinned (tests/test_oracle_walls.py): after a step the three wall rows carry u^(H) = 0
 *                                  and T^(H) = T_wall to rounding; mass conserved to rounding; rest state at
 *                                  T_wall is a fixed point; slowest shear mode decays as between no-slip
 *                                  planes at the innermost imposed rows; steady conduction between walls at
 *                                  different temperatures is a linear T(z) (uniform conductivity at uniform
 *                                  pressure) carrying the flux k dT/dz with k = c_p (tau - 1/2) p / r^2.
 *                                  The rule itself is a READING of "rigid boundary conditions ... adjusts
 *                                  population values at sites with z = 0, 1, 2": parity with
 *                                  the authors' wall scheme is UNPINNED (reading 19).
 *
 * Conventions: sites (i,k), i = 0..Lx-1 (x, periodic), k = 0..Lz-1
 * (z, up); arrays are dense f[l][k][i], x fastest; population order: ascending e_z, then
 * ascending e_x (l = 0 is (-1,-3), l = 18 is (0,0), l = 36 is (1,3)), so that the opposite
 * velocity of l is 36 - l.  dt = 1, lattice spacing = r length units, c_l = r e_l,
 * gravity vector (0, -g) with g > 0.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liblbm_oracle.so lbm_oracle.c -lm
 * (no -ffast-math; -ffp-contract is left at the compiler default, FMA contraction allowed).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NPOP 37
#define DIM 2.0

static int g_ready = 0;
static int EX[NPOP], EZ[NPOP];
static double W[NPOP], R_LAT; /* weights per population, lattice constant r */

/* ---------------------------------------------------------------------------------------
 * Velocity set and quadrature (reading 8(c)-1,2).
 * e_l = all integer vectors with |e|^2 <= 10; the eight shell weights and r are the unique
 * positive solution near r ~ 1.2 of   sum_l w_l c_lx^a c_lz^b = G_a G_b   for the nine
 * (a,b) below, G_n the moments of the unit-variance Gaussian (1, 1, 3, 15, 105).
 * Solved here in long double: for a trial r eight of the equations are linear in w and
 * non-singular (all but (8,0), kept last in MOM_AB); the ninth, (8,0), fixes r (bisection
 * on its residual).
 * ------------------------------------------------------------------------------------- */
static const int SHELL_E2[8] = {0, 1, 2, 4, 5, 8, 9, 10};
static const int MOM_AB[9][2] = {{0, 0}, {2, 0}, {4, 0}, {2, 2}, {6, 0}, {4, 2}, {6, 2}, {4, 4}, {8, 0}};

static long double gauss_moment(int n)
{
    long double v = 1.0L;
    for (int j = n - 1; j > 0; j -= 2) v *= (long double)j;
    return v; /* (n-1)!! for even n */
}

static long double ipowl(long double x, int n)
{
    long double v = 1.0L;
    for (int j = 0; j < n; ++j) v *= x;
    return v;
}

/* integer lattice sums S[eq][shell] = sum_{e in shell} ex^a ez^b */
static void shell_sums(long double S[9][8])
{
    for (int q = 0; q < 9; ++q)
        for (int s = 0; s < 8; ++s) {
            long double acc = 0.0L;
            for (int ez = -3; ez <= 3; ++ez)
                for (int ex = -3; ex <= 3; ++ex)
                    if (ex * ex + ez * ez == SHELL_E2[s])
                        acc += ipowl((long double)ex, MOM_AB[q][0]) * ipowl((long double)ez, MOM_AB[q][1]);
            S[q][s] = acc;
        }
}

/* solve the first 8 equations for w at lattice constant r; return residual of the 9th */
static long double weights_at(long double r, long double w[8])
{
    long double S[9][8], A[8][9];
    shell_sums(S);
    for (int q = 0; q < 8; ++q) {
        int n = MOM_AB[q][0] + MOM_AB[q][1];
        for (int s = 0; s < 8; ++s) A[q][s] = S[q][s];
        A[q][8] = gauss_moment(MOM_AB[q][0]) * gauss_moment(MOM_AB[q][1]) / ipowl(r, n);
    }
    for (int c = 0; c < 8; ++c) { /* Gaussian elimination, partial pivoting */
        int p = c;
        for (int q = c + 1; q < 8; ++q)
            if (fabsl(A[q][c]) > fabsl(A[p][c])) p = q;
        for (int j = 0; j < 9; ++j) { long double t = A[c][j]; A[c][j] = A[p][j]; A[p][j] = t; }
        for (int q = c + 1; q < 8; ++q) {
            long double m = A[q][c] / A[c][c];
            for (int j = c; j < 9; ++j) A[q][j] -= m * A[c][j];
        }
    }
    for (int c = 7; c >= 0; --c) {
        long double acc = A[c][8];
        for (int j = c + 1; j < 8; ++j) acc -= A[c][j] * w[j];
        w[c] = acc / A[c][c];
    }
    long double lhs = 0.0L;
    for (int s = 0; s < 8; ++s) lhs += S[8][s] * w[s];
    int n = MOM_AB[8][0] + MOM_AB[8][1];
    return lhs * ipowl(r, n) - gauss_moment(MOM_AB[8][0]) * gauss_moment(MOM_AB[8][1]);
}

static void ensure_tables(void)
{
    if (g_ready) return;
    int l = 0;
    for (int ez = -3; ez <= 3; ++ez)
        for (int ex = -3; ex <= 3; ++ex)
            if (ex * ex + ez * ez <= 10) { EX[l] = ex; EZ[l] = ez; ++l; }
    /* l == 37 by construction of the set */
    long double w[8], lo = 1.15L, hi = 1.25L;
    long double flo = weights_at(lo, w);
    for (int it = 0; it < 200; ++it) {
        long double mid = 0.5L * (lo + hi);
        long double fm = weights_at(mid, w);
        if ((fm < 0) == (flo < 0)) { lo = mid; flo = fm; } else { hi = mid; }
    }
    long double r = 0.5L * (lo + hi);
    weights_at(r, w);
    R_LAT = (double)r;
    for (l = 0; l < NPOP; ++l) {
        int e2 = EX[l] * EX[l] + EZ[l] * EZ[l];
        for (int s = 0; s < 8; ++s)
            if (SHELL_E2[s] == e2) W[l] = (double)w[s];
    }
    g_ready = 1;
}

void orc_tables(int *ex, int *ez, double *w, double *r)
{
    ensure_tables();
    for (int l = 0; l < NPOP; ++l) { ex[l] = EX[l]; ez[l] = EZ[l]; w[l] = W[l]; }
    *r = R_LAT;
}

void orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------
 * Equilibrium: "local Maxwellian", reading 8(c)-3: the 4th-order Hermite
 * projection of the Maxwellian with density rho, velocity u, temperature T = 1 + theta on
 * the D2Q37 quadrature, D = 2.  With c = c_l, cu = c.u, c2 = |c|^2, u2 = |u|^2:
 *   f_eq = w rho { 1 + cu + 1/2 [cu^2 - u2 + theta (c2 - D)]
 *                 + cu/6 [cu^2 - 3 u2 + 3 theta (c2 - D - 2)]
 *                 + 1/24 [cu^4 - 6 cu^2 u2 + 3 u2^2
 *                         + 6 theta (cu^2 (c2 - D - 4) + u2 (D + 2 - c2))
 *                         + 3 theta^2 (c2^2 - 2 (D+2) c2 + D (D+2))] }
 * ------------------------------------------------------------------------------------- */
void orc_feq(double rho, double ux, double uz, double T, double *out)
{
    ensure_tables();
    const double theta = T - 1.0;
    const double u2 = ux * ux + uz * uz;
    for (int l = 0; l < NPOP; ++l) {
        const double cx = R_LAT * EX[l], cz = R_LAT * EZ[l];
        const double cu = cx * ux + cz * uz;
        const double c2 = cx * cx + cz * cz;
        const double h1 = cu;
        const double h2 = 0.5 * (cu * cu - u2 + theta * (c2 - DIM));
        const double h3 = (cu / 6.0) * (cu * cu - 3.0 * u2 + 3.0 * theta * (c2 - DIM - 2.0));
        const double h4 = (1.0 / 24.0) *
                          (cu * cu * cu * cu - 6.0 * cu * cu * u2 + 3.0 * u2 * u2 +
                           6.0 * theta * (cu * cu * (c2 - DIM - 4.0) + u2 * (DIM + 2.0 - c2)) +
                           3.0 * theta * theta * (c2 * c2 - 2.0 * (DIM + 2.0) * c2 + DIM * (DIM + 2.0)));
        out[l] = W[l] * rho * (1.0 + h1 + h2 + h3 + h4);
    }
}

/* ---------------------------------------------------------------------------------------
 * Kinetic moments of one site, eq. 7:
 *   rho = sum f,  rho u = sum c f,  d rho T = sum |c - u|^2 f.
 * ------------------------------------------------------------------------------------- */
static void site_moments(const double *fl, double *rho, double *ux, double *uz, double *T)
{
    double m0 = 0.0, mx = 0.0, mz = 0.0;
    for (int l = 0; l < NPOP; ++l) {
        m0 += fl[l];
        mx += R_LAT * EX[l] * fl[l];
        mz += R_LAT * EZ[l] * fl[l];
    }
    const double vx = mx / m0, vz = mz / m0;
    double e = 0.0;
    for (int l = 0; l < NPOP; ++l) {
        const double dx = R_LAT * EX[l] - vx, dz = R_LAT * EZ[l] - vz;
        e += (dx * dx + dz * dz) * fl[l];
    }
    *rho = m0; *ux = vx; *uz = vz; *T = e / (DIM * m0);
}

void orc_site_moments(const double *fl, double *out4)
{
    ensure_tables();
    site_moments(fl, &out4[0], &out4[1], &out4[2], &out4[3]);
}

/* ---------------------------------------------------------------------------------------
 * Propagate (pull) + bc, lhs of eq. 5, reading 8(c)-9 for the walls:
 *   fs[l][k][i] = f[l][k - e_lz][(i - e_lx) mod Lx]                      source row inside
 *   fs[l][k][i] = f[36-l][-1 - ks][is]            if ks = k - e_lz < 0    (bottom wall)
 *   fs[l][k][i] = f[36-l][2 Lz - 1 - ks][is]      if ks >= Lz             (top wall)
 * i.e. a population that would have crossed a wall (located half a site outside rows 0 and
 * Lz-1) re-enters in the same step with reversed velocity; only rows 0..2 and Lz-3..Lz-1 are
 * affected.  periodic_z != 0 selects the oracle-only fully periodic mode used
 * by the round-trip and wave-decay pins.  dir = +1 is the model's propagate; dir = -1 moves
 * every population against its velocity (the inverse map in fully periodic mode).
 * ------------------------------------------------------------------------------------- */
void orc_propagate(const double *f, double *fs, int Lx, int Lz, int periodic_z, int dir)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < Lz; ++k)
        for (int l = 0; l < NPOP; ++l) {
            int ks = k - dir * EZ[l];
            int ls = l;
            if (periodic_z) {
                ks = ((ks % Lz) + Lz) % Lz;
            } else if (ks < 0) {
                ks = -1 - ks; ls = NPOP - 1 - l;
            } else if (ks >= Lz) {
                ks = 2 * Lz - 1 - ks; ls = NPOP - 1 - l;
            }
            for (int i = 0; i < Lx; ++i) {
                int is = i - dir * EX[l];
                is = ((is % Lx) + Lx) % Lx;
                fs[l * plane + (size_t)k * Lx + i] = f[ls * plane + (size_t)ks * Lx + is];
            }
        }
}

/* ---------------------------------------------------------------------------------------
 * Collide, rhs of eq. 5 with the shifted equilibrium of eq. 6:
 *   rho, u, T from eq. 7;  u' = u + g_vec tau = (u_x, u_z - g tau);
 *   T' = T + tau (dt - tau) g^2 / d   (dt = 1, d = 2);
 *   f_new = fs - (dt / tau) (fs - f_eq(rho, u', T')).
 * ------------------------------------------------------------------------------------- */
void orc_collide(const double *fs, double *fnew, int Lx, int Lz, double tau, double g)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < Lz; ++k)
        for (int i = 0; i < Lx; ++i) {
            const size_t s = (size_t)k * Lx + i;
            double fl[NPOP], feq[NPOP], rho, ux, uz, T;
            for (int l = 0; l < NPOP; ++l) fl[l] = fs[l * plane + s];
            site_moments(fl, &rho, &ux, &uz, &T);
            const double us_x = ux;
            const double us_z = uz - g * tau;
            const double Ts = T + tau * (1.0 - tau) * g * g / DIM;
            orc_feq(rho, us_x, us_z, Ts, feq);
            for (int l = 0; l < NPOP; ++l)
                fnew[l * plane + s] = fl[l] - (1.0 / tau) * (fl[l] - feq[l]);
        }
}

/* ---------------------------------------------------------------------------------------
 * Isothermal no-slip walls, wall_kind = 1 (reading 19).  PAPER.md:114: "Step bc
 * executes after propagate in order to enforce boundary conditions at the top and bottom of
 * the cell; it adjusts population values at sites with coordinates z = 0, 1, 2 and
 * z = Lz-3, Lz-2 and Lz-1"; the paper gives no formula, its references impose the wall
 * temperature and zero velocity on the three rows.  Reading: after propagate (whose wall-
 * crossing gathers are filled by the bounce-back rule of orc_propagate, which conserves
 * mass), every site of the three rows next to a wall has the EQUILIBRIUM PART of its
 * populations moved to the wall state, keeping density and non-equilibrium part:
 *   (rho*, u*, T*) = moments (eq. 7) of the post-propagate populations fs at the site;
 *   fs_l  <-  fs_l - f_eq_l(rho*, u*, T*) + f_eq_l(rho*, u_w, T_w)
 *   u_w = -g_vec dt/2 = (0, +g/2),   T_w = T_wall - dt^2 g^2 / (4 D),
 * i.e. the kinetic moments that PAPER.md:94 maps to the hydrodynamic fields u^(H) = 0,
 * T^(H) = T_wall.  By the closure of eq. 7 the adjusted populations have exactly the moments
 * (rho*, u_w, T_w); collide then runs unchanged on them.  T_bot applies to rows 0..2, T_top
 * to rows Lz-3..Lz-1.
 * ------------------------------------------------------------------------------------- */
void orc_bc_isothermal(double *fs, int Lx, int Lz, double g, double T_bot, double T_top)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    for (int side = 0; side < 2; ++side)
        for (int j = 0; j < 3; ++j) {
            const int k = side == 0 ? j : Lz - 1 - j;
            const double T_wall = side == 0 ? T_bot : T_top;
            const double uw_x = 0.0, uw_z = 0.5 * g;
            const double Tw = T_wall - g * g / (4.0 * DIM);
            for (int i = 0; i < Lx; ++i) {
                const size_t s = (size_t)k * Lx + i;
                double fl[NPOP], feq_own[NPOP], feq_wall[NPOP], rho, ux, uz, T;
                for (int l = 0; l < NPOP; ++l) fl[l] = fs[l * plane + s];
                site_moments(fl, &rho, &ux, &uz, &T);
                orc_feq(rho, ux, uz, T, feq_own);
                orc_feq(rho, uw_x, uw_z, Tw, feq_wall);
                for (int l = 0; l < NPOP; ++l) fs[l * plane + s] = fl[l] - feq_own[l] + feq_wall[l];
            }
        }
}

/* n time steps with a choice of wall rule: wall_kind 0 = bounce-back only (reading 9),
 * 1 = bounce-back fill followed by the isothermal adjustment above (reading 19). */
void orc_step_walls(double *f, double *tmp, int Lx, int Lz, double tau, double g, int nsteps, int wall_kind,
                    double T_bot, double T_top)
{
    for (int n = 0; n < nsteps; ++n) {
        orc_propagate(f, tmp, Lx, Lz, 0, +1);
        if (wall_kind == 1) orc_bc_isothermal(tmp, Lx, Lz, g, T_bot, T_top);
        orc_collide(tmp, f, Lx, Lz, tau, g);
    }
}

/* n time steps: propagate -> bc -> collide; f is updated in place, tmp is
 * a scratch lattice of the same size (the paper's prv/nxt pair). */
void orc_step(double *f, double *tmp, int Lx, int Lz, double tau, double g, int nsteps, int periodic_z)
{
    for (int n = 0; n < nsteps; ++n) {
        orc_propagate(f, tmp, Lx, Lz, periodic_z, +1);
        orc_collide(tmp, f, Lx, Lz, tau, g);
    }
}

/* ---------------------------------------------------------------------------------------
 * Hydrodynamic fields of the STORED (post-collision) state, PAPER.md:94 + reading 8(c)-8:
 * the collision maps the kinetic moments (rho,u,T) -> (rho, u + g_vec dt, T), so on the
 * stored state  u^(H) = u - g_vec dt/2 = (u_x, u_z + g/2),  T^(H) = T + dt^2 g^2/(4 D).
 * Any output pointer may be NULL.
 * ------------------------------------------------------------------------------------- */
void orc_moments(const double *f, int Lx, int Lz, double g, double *rho, double *ux, double *uz, double *T)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < Lz; ++k)
        for (int i = 0; i < Lx; ++i) {
            const size_t s = (size_t)k * Lx + i;
            double fl[NPOP], m0, vx, vz, t;
            for (int l = 0; l < NPOP; ++l) fl[l] = f[l * plane + s];
            site_moments(fl, &m0, &vx, &vz, &t);
            if (rho) rho[s] = m0;
            if (ux) ux[s] = vx;
            if (uz) uz[s] = vz + 0.5 * g;
            if (T) T[s] = t + g * g / (4.0 * DIM);
        }
}

/* Lattice totals sum f, sum c_x f, sum c_z f, sum |c|^2 f (mass, momentum, 2 x energy). */
void orc_totals(const double *f, int Lx, int Lz, double *out4)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    long double t0 = 0, tx = 0, tz = 0, t2 = 0;
    for (int l = 0; l < NPOP; ++l) {
        long double s = 0;
        for (size_t j = 0; j < plane; ++j) s += f[l * plane + j];
        const double cx = R_LAT * EX[l], cz = R_LAT * EZ[l];
        t0 += s; tx += cx * s; tz += cz * s; t2 += (cx * cx + cz * cz) * s;
    }
    out4[0] = (double)t0; out4[1] = (double)tx; out4[2] = (double)tz; out4[3] = (double)t2;
}

/* ---------------------------------------------------------------------------------------
 * Mixing widths, eq. 8, 9, 12, reading 8(c)-13:
 *   Tbar(k) = (1/Lx) sum_i T^(H)(i,k);
 *   Theta[b] = 2b on (0,1/2), 2(1-b) on (1/2,1), zero outside [0,1];
 *   L_u = sum_k Theta[(Tbar - T_u)/(T_m - T_u)],  L_d = sum_k Theta[(Tbar - T_m)/(T_d - T_m)]
 * in sites (dz = 1).  Tbar (length Lz) may be NULL.
 * ------------------------------------------------------------------------------------- */
static double tent(double b)
{
    if (b <= 0.0 || b >= 1.0) return 0.0;
    return b < 0.5 ? 2.0 * b : 2.0 * (1.0 - b);
}

void orc_mixing_widths(const double *f, int Lx, int Lz, double g, double T_d, double T_m, double T_u,
                       double *L_u, double *L_d, double *Tbar)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    double lu = 0.0, ld = 0.0;
    for (int k = 0; k < Lz; ++k) {
        double acc = 0.0;
        for (int i = 0; i < Lx; ++i) {
            const size_t s = (size_t)k * Lx + i;
            double fl[NPOP], m0, vx, vz, t;
            for (int l = 0; l < NPOP; ++l) fl[l] = f[l * plane + s];
            site_moments(fl, &m0, &vx, &vz, &t);
            acc += t + g * g / (4.0 * DIM);
        }
        const double tb = acc / Lx;
        if (Tbar) Tbar[k] = tb;
        lu += tent((tb - T_u) / (T_m - T_u));
        ld += tent((tb - T_m) / (T_d - T_m));
    }
    *L_u = lu; *L_d = ld;
}

/* ---------------------------------------------------------------------------------------
 * Populations at the equilibrium of given kinetic fields (no shift): f = f_eq(rho,u,T).
 * Fields are [Lz][Lx], x fastest.
 * ------------------------------------------------------------------------------------- */
void orc_init_equilibrium(double *f, int Lx, int Lz, const double *rho, const double *ux, const double *uz,
                          const double *T)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    for (size_t s = 0; s < plane; ++s) {
        double feq[NPOP];
        orc_feq(rho[s], ux[s], uz[s], T[s], feq);
        for (int l = 0; l < NPOP; ++l) f[l * plane + s] = feq[l];
    }
}

/* ---------------------------------------------------------------------------------------
 * Interface perturbation and RNG, reading 8(c)-12 (paper: "white noise", PAPER.md:222;
 * amplitudes from BASELINE.json).  SplitMix64 stream; U = (next >> 11) * 2^-53.
 * Consumption order: lower interface first, then upper (single front, delta = 0: one set,
 * used for both).  pert_kind 0: none.  1: modes m = 1..n_modes, each draws its amplitude
 * a_m = amp_lo + (amp_hi - amp_lo) U only if amp_hi != amp_lo (else a_m = amp_lo, no draw),
 * then its phase phi_m = 2 pi U;  h(i) = sum_m a_m cos(2 pi m i / Lx + phi_m).
 * 2: white noise h(i) = amp_hi (2U - 1), i = 0..Lx-1.
 * ------------------------------------------------------------------------------------- */
static uint64_t splitmix64(uint64_t *state)
{
    uint64_t z = (*state += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static double uniform01(uint64_t *state) { return (double)(splitmix64(state) >> 11) * (1.0 / 9007199254740992.0); }

static void draw_interface(uint64_t *state, int Lx, int pert_kind, int n_modes, double amp_lo, double amp_hi,
                           double *h)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int i = 0; i < Lx; ++i) h[i] = 0.0;
    if (pert_kind == 1) {
        for (int m = 1; m <= n_modes; ++m) {
            double a = amp_lo;
            if (amp_hi != amp_lo) a = amp_lo + (amp_hi - amp_lo) * uniform01(state);
            const double phi = two_pi * uniform01(state);
            for (int i = 0; i < Lx; ++i) h[i] += a * cos(two_pi * (double)m * (double)i / (double)Lx + phi);
        }
    } else if (pert_kind == 2) {
        for (int i = 0; i < Lx; ++i) h[i] = amp_hi * (2.0 * uniform01(state) - 1.0);
    }
}

void orc_interfaces(uint64_t seed, int Lx, double delta, int pert_kind, int n_modes, double amp_lo,
                    double amp_hi, double *h_lo, double *h_hi)
{
    uint64_t state = seed;
    draw_interface(&state, Lx, pert_kind, n_modes, amp_lo, amp_hi, h_lo);
    if (delta == 0.0) {
        for (int i = 0; i < Lx; ++i) h_hi[i] = h_lo[i];
    } else {
        draw_interface(&state, Lx, pert_kind, n_modes, amp_lo, amp_hi, h_hi);
    }
}

/* ---------------------------------------------------------------------------------------
 * Hydrostatic three-layer initial state, eq. 1-2 with the tanh smoothing of
 * Fig. 1, reading 8(c)-11.  Site-centre height z_k = k - (Lz-1)/2 (site units,
 * walls at +-Lz/2); one site is r length units, so eq. 1's exponent is g r z / T (8(c)-4).
 * Per column i: a_lo = -delta/2 + h_lo(i), a_hi = +delta/2 + h_hi(i); with beta = 1/T0 and
 * S(s) = (1 + tanh s)/2 (Heaviside with S(0) = 1/2 when w = 0):
 *   beta(z)  = beta_d + (beta_m - beta_d) S((z - a_lo)/w) + (beta_u - beta_m) S((z - a_hi)/w)
 *   ln p(z)  = ln(rho_m / beta(0)) - g r [ beta_d z + (beta_m - beta_d) I(z; a_lo)
 *                                              + (beta_u - beta_m) I(z; a_hi) ]
 *   I(z; a)  = int_0^z S((z'-a)/w) dz' = [ z + w lncosh((z-a)/w) - w lncosh(a/w) ] / 2
 *            (w = 0:  max(z-a,0) - max(-a,0))
 *   T0 = 1/beta,  rho0 = p beta.
 * This is exactly hydrostatic (dp/dz = -g r rho0), has rho0 = rho_m at z = 0, continuous
 * pressure across the interfaces (eq. 2), and equals eq. 1 when w -> 0.
 * Stored populations (8(c)-8): f = f_eq(rho0, (0, -g/2), T0 - g^2/8), so that the
 * hydrodynamic fields are u^(H) = 0, T^(H) = T0.
 * Optional outputs rho0_out, T0_out ([Lz][Lx]) may be NULL.
 * ------------------------------------------------------------------------------------- */
static double lncosh(double s)
{
    const double a = fabs(s);
    return a + log1p(exp(-2.0 * a)) - 0.69314718055994530941723212145818;
}

static double smooth_step(double z, double a, double w)
{
    if (w > 0.0) return 0.5 * (1.0 + tanh((z - a) / w));
    return z > a ? 1.0 : (z < a ? 0.0 : 0.5);
}

static double smooth_step_integral(double z, double a, double w)
{
    if (w > 0.0) return 0.5 * (z + w * lncosh((z - a) / w) - w * lncosh(a / w));
    return fmax(z - a, 0.0) - fmax(-a, 0.0);
}

void orc_rt_profile(int Lx, int Lz, double g, double T_d, double T_m, double T_u, double rho_m, double delta,
                    double w, const double *h_lo, const double *h_hi, double *rho0, double *T0)
{
    ensure_tables();
    const double bd = 1.0 / T_d, bm = 1.0 / T_m, bu = 1.0 / T_u;
    for (int k = 0; k < Lz; ++k) {
        const double z = (double)k - 0.5 * (double)(Lz - 1);
        for (int i = 0; i < Lx; ++i) {
            const double a_lo = -0.5 * delta + h_lo[i], a_hi = 0.5 * delta + h_hi[i];
            const double beta = bd + (bm - bd) * smooth_step(z, a_lo, w) + (bu - bm) * smooth_step(z, a_hi, w);
            const double beta0 = bd + (bm - bd) * smooth_step(0.0, a_lo, w) + (bu - bm) * smooth_step(0.0, a_hi, w);
            const double lnp = log(rho_m / beta0) -
                               g * R_LAT *
                                   (bd * z + (bm - bd) * smooth_step_integral(z, a_lo, w) +
                                    (bu - bm) * smooth_step_integral(z, a_hi, w));
            const size_t s = (size_t)k * Lx + i;
            T0[s] = 1.0 / beta;
            rho0[s] = exp(lnp) * beta;
        }
    }
}

void orc_init_rt(double *f, int Lx, int Lz, double g, uint64_t seed, double T_d, double T_m, double T_u,
                 double rho_m, double delta, double smooth_w, int pert_kind, int n_modes, double amp_lo,
                 double amp_hi, double *rho0_out, double *T0_out)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    double *h_lo = (double *)malloc(sizeof(double) * Lx), *h_hi = (double *)malloc(sizeof(double) * Lx);
    double *rho0 = (double *)malloc(sizeof(double) * plane), *T0 = (double *)malloc(sizeof(double) * plane);
    orc_interfaces(seed, Lx, delta, pert_kind, n_modes, amp_lo, amp_hi, h_lo, h_hi);
    orc_rt_profile(Lx, Lz, g, T_d, T_m, T_u, rho_m, delta, smooth_w, h_lo, h_hi, rho0, T0);
    for (size_t s = 0; s < plane; ++s) {
        double feq[NPOP];
        orc_feq(rho0[s], 0.0, -0.5 * g, T0[s] - g * g / (4.0 * DIM), feq);
        for (int l = 0; l < NPOP; ++l) f[l * plane + s] = feq[l];
    }
    if (rho0_out) memcpy(rho0_out, rho0, sizeof(double) * plane);
    if (T0_out) memcpy(T0_out, T0, sizeof(double) * plane);
    free(h_lo); free(h_hi); free(rho0); free(T0);
}

/* ---------------------------------------------------------------------------------------
 * Row profiles used in section IV of the paper, from the hydrodynamic fields of the stored
 * state:
 *   Tbar(k)  = <T>_x
 *   Trms(k)  = sqrt( < (T - <T>_x)^2 >_x )             (Fig. 8)
 *   Ekbar(k) = <E_k>_x,  Ekrms(k) = sqrt( < (E_k - <E_k>_x)^2 >_x )   (Fig. 9)
 * READING (the paper does not define E_k): E_k = rho |u^(H)|^2 / 2, the kinetic energy
 * density.  Two passes per row (mean, then squared deviations).  Pinned by closed forms on
 * cosine-modulated rows; parity with the authors' E_k definition is UNPINNED.
 * Any output (length Lz) may be NULL.
 * ------------------------------------------------------------------------------------- */
void orc_profiles(const double *f, int Lx, int Lz, double g, double *Tbar, double *Trms, double *Ekbar,
                  double *Ekrms)
{
    ensure_tables();
    const size_t plane = (size_t)Lx * (size_t)Lz;
    double *Trow = (double *)malloc(sizeof(double) * Lx), *Erow = (double *)malloc(sizeof(double) * Lx);
    for (int k = 0; k < Lz; ++k) {
        double sT = 0.0, sE = 0.0;
        for (int i = 0; i < Lx; ++i) {
            const size_t s = (size_t)k * Lx + i;
            double fl[NPOP], m0, vx, vz, t;
            for (int l = 0; l < NPOP; ++l) fl[l] = f[l * plane + s];
            site_moments(fl, &m0, &vx, &vz, &t);
            const double uzh = vz + 0.5 * g;
            Trow[i] = t + g * g / (4.0 * DIM);
            Erow[i] = 0.5 * m0 * (vx * vx + uzh * uzh);
            sT += Trow[i]; sE += Erow[i];
        }
        const double mT = sT / Lx, mE = sE / Lx;
        double vT = 0.0, vE = 0.0;
        for (int i = 0; i < Lx; ++i) {
            vT += (Trow[i] - mT) * (Trow[i] - mT);
            vE += (Erow[i] - mE) * (Erow[i] - mE);
        }
        if (Tbar) Tbar[k] = mT;
        if (Trms) Trms[k] = sqrt(vT / Lx);
        if (Ekbar) Ekbar[k] = mE;
        if (Ekrms) Ekrms[k] = sqrt(vE / Lx);
    }
    free(Trow); free(Erow);
}

/* ---------------------------------------------------------------------------------------
 * Growth rate from a logged mixing length, eq. 11 / 14:
 *   [dL/dt]^2 = 4 alpha g At L   =>   alpha(t_j) = (dL/dt)_j^2 / (4 g At L_j),
 * "local in time".  dL/dt by centred differences on the (possibly non-uniform)
 * sample times, one-sided at the two ends.  For the double front pass L_tot and the total At
 * (alpha_tot of eq. 14).  alpha_j = 0 where L_j <= 0.
 * ------------------------------------------------------------------------------------- */
void orc_growth_rate(int n, const double *t, const double *L, double g, double At, double *alpha)
{
    for (int j = 0; j < n; ++j) {
        const int a = j > 0 ? j - 1 : j, b = j < n - 1 ? j + 1 : j;
        const double dLdt = (b > a) ? (L[b] - L[a]) / (t[b] - t[a]) : 0.0;
        alpha[j] = L[j] > 0.0 ? dLdt * dLdt / (4.0 * g * At * L[j]) : 0.0;
    }
}
