// d2q37.cuh -- the D2Q37 velocity set and the per-site collision arithmetic, device side.
//
// Velocity set (Fig. 2; reading 1): all integer e with |e|^2 <= 10,
// ordered by ascending e_z then e_x, so that rows of the set are
//   e_z = -3: l =  0.. 2 (e_x = -1..1)      e_z = +1: l = 22..28 (e_x = -3..3)
//   e_z = -2: l =  3.. 7 (e_x = -2..2)      e_z = +2: l = 29..33 (e_x = -2..2)
//   e_z = -1: l =  8..14 (e_x = -3..3)      e_z = +3: l = 34..36 (e_x = -1..1)
//   e_z =  0: l = 15..21 (e_x = -3..3)
// and the opposite velocity of l is 36 - l.  c_l = r e_l.
//
// Everything here is evaluated per site in registers (north_star: "the collision's moment and
// equilibrium evaluation kept in registers").  Loops over l are unrolled at compile time so that every
// e_x, e_z, |e|^2 and weight is an immediate.
#pragma once
#include <type_traits>
#include <utility>

#include "d2q37_constants.h"

namespace d2q37 {

constexpr int NPOP = 37;

__host__ __device__ constexpr int pop_ez(int l)
{
    return l < 3 ? -3 : l < 8 ? -2 : l < 15 ? -1 : l < 22 ? 0 : l < 29 ? 1 : l < 34 ? 2 : 3;
}
__host__ __device__ constexpr int row_first(int ez)  // index of the first population with this e_z
{
    return ez == -3 ? 0 : ez == -2 ? 3 : ez == -1 ? 8 : ez == 0 ? 15 : ez == 1 ? 22 : ez == 2 ? 29 : 34;
}
__host__ __device__ constexpr int row_half(int ez)  // e_x runs over -half..half
{
    return (ez == 3 || ez == -3) ? 1 : (ez == 2 || ez == -2) ? 2 : 3;
}
__host__ __device__ constexpr int pop_ex(int l) { return l - row_first(pop_ez(l)) - row_half(pop_ez(l)); }
__host__ __device__ constexpr int pop_e2(int l) { return pop_ex(l) * pop_ex(l) + pop_ez(l) * pop_ez(l); }
__host__ __device__ constexpr int pop_index(int ex, int ez) { return row_first(ez) + row_half(ez) + ex; }
__host__ __device__ constexpr double shell_weight(int e2)
{
    return e2 == 0 ? D2Q37_W0 : e2 == 1 ? D2Q37_W1 : e2 == 2 ? D2Q37_W2 : e2 == 4 ? D2Q37_W4 :
           e2 == 5 ? D2Q37_W5 : e2 == 8 ? D2Q37_W8 : e2 == 9 ? D2Q37_W9 : D2Q37_W10;
}
__host__ __device__ constexpr int shell_slot(int e2)  // 0..7
{
    return e2 == 0 ? 0 : e2 == 1 ? 1 : e2 == 2 ? 2 : e2 == 4 ? 3 : e2 == 5 ? 4 : e2 == 8 ? 5 : e2 == 9 ? 6 : 7;
}
__host__ __device__ constexpr int shell_e2(int slot)
{
    return slot == 0 ? 0 : slot == 1 ? 1 : slot == 2 ? 2 : slot == 3 ? 4 : slot == 4 ? 5 : slot == 5 ? 8 : slot == 6 ? 9 : 10;
}

// Per-shell constants of the equilibrium polynomial (see equilibrium_blend_from), kept in the constant bank so
// that they are instruction operands (c[bank][offset]) rather than 64-bit immediates rebuilt with UMOV pairs.
struct ShellConst {
    double k1, k2, k3, k4, k5, w;
};
__host__ __device__ constexpr ShellConst shell_const(int slot)
{
    const double c2 = D2Q37_R2 * shell_e2(slot);
    return ShellConst{0.5 * (c2 - 2.0), 0.25 * (4.0 - c2), 0.125 * (c2 * c2 - 8.0 * c2 + 8.0),
                      0.5 * (c2 - 4.0), 0.25 * (c2 - 6.0), shell_weight(shell_e2(slot))};
}
static __constant__ ShellConst c_shell[8] = {shell_const(0), shell_const(1), shell_const(2), shell_const(3),
                                             shell_const(4), shell_const(5), shell_const(6), shell_const(7)};
static __constant__ double c_lat[4] = {D2Q37_R, D2Q37_R2, 1.0 / 6.0, 1.0 / 24.0};

// first population (ascending l) with a given e_x / e_z: the accumulators of raw_moments_from start there
__host__ __device__ constexpr int first_with_ex(int ex)
{
    for (int l = 0; l < NPOP; ++l)
        if (pop_ex(l) == ex) return l;
    return -1;
}
__host__ __device__ constexpr int first_with_ez(int ez) { return row_first(ez); }

// compile-time loop: f(std::integral_constant<int, B>{}), ..., f(<E-1>)
template <int B, int E, class F>
__host__ __device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// Raw lattice moments of one site in integer-velocity form:
//   m0 = sum f, jx = sum e_x f, jz = sum e_z f, m2 = sum |e|^2 f.
// Column sums C[e_x] and row sums R[e_z] are formed first (74 adds), the weighted sums from them.
// `load(L)` returns population l = L::value (registers, shared memory, ...); it is called once per l, in
// ascending l, so every caller accumulates in the same order (bit-identical results).
struct RawMoments {
    double m0, jx, jz, m2;
};

template <class Load>
__device__ __forceinline__ RawMoments raw_moments_from(Load &&load)
{
    double C[7], R[7];
    static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int ex = pop_ex(l), ez = pop_ez(l);
        const double v = load(L);
        if constexpr (l == first_with_ex(ex)) C[ex + 3] = v;
        else C[ex + 3] += v;
        if constexpr (l == first_with_ez(ez)) R[ez + 3] = v;
        else R[ez + 3] += v;
    });
    RawMoments m;
    const double c1 = C[4] + C[2], c2 = C[5] + C[1], c3 = C[6] + C[0];
    const double r1 = R[4] + R[2], r2 = R[5] + R[1], r3 = R[6] + R[0];
    m.m0 = (C[3] + c1) + (c2 + c3);
    m.jx = (C[4] - C[2]) + 2.0 * (C[5] - C[1]) + 3.0 * (C[6] - C[0]);
    m.jz = (R[4] - R[2]) + 2.0 * (R[5] - R[1]) + 3.0 * (R[6] - R[0]);
    m.m2 = (c1 + r1) + 4.0 * (c2 + r2) + 9.0 * (c3 + r3);
    return m;
}

__device__ __forceinline__ RawMoments raw_moments(const double (&f)[NPOP])
{
    return raw_moments_from([&](auto L) { return f[decltype(L)::value]; });
}

// Kinetic moments of eq. 7: rho = sum f, rho u = sum c f, d rho T = sum |c-u|^2 f, d = 2,
// with c = r e:  u = r j / rho,  T = (r^2 m2 / rho - |u|^2) / 2.
struct Kinetic {
    double rho, ux, uz, T;
};

__device__ __forceinline__ Kinetic kinetic_from_raw(const RawMoments &m)
{
    const double inv = 1.0 / m.m0;
    Kinetic k;
    k.rho = m.m0;
    k.ux = (c_lat[0] * m.jx) * inv;
    k.uz = (c_lat[0] * m.jz) * inv;
    k.T = 0.5 * ((c_lat[1] * m.m2) * inv - (k.ux * k.ux + k.uz * k.uz));
    return k;
}

__device__ __forceinline__ Kinetic kinetic_moments(const double (&f)[NPOP]) { return kinetic_from_raw(raw_moments(f)); }

// store(L, keep * load(L) + scale * f_eq_l(rho = 1, u, T)) for all l.
//
// f_eq is the 4th-order Hermite projection of the Maxwellian on this quadrature ("local Maxwellian",
// PAPER.md:80; reading 3).  With s = c.u, q = |u|^2, theta = T - 1, D = 2 it is a quartic in s
// whose coefficients depend on the shell |c|^2 only:
//   f_eq / (w rho) = g0 + g1 s + g2 s^2 + s^3/6 + s^4/24
//   g0 = 1 - q/2 + q^2/8 + theta [ (c2-2)/2 + q (4-c2)/4 ] + theta^2 (c2^2 - 8 c2 + 8)/8
//   g1 = 1 - q/2 + theta (c2-4)/2
//   g2 = 1/2 - q/4 + theta (c2-6)/4
// Opposite populations l and 36 - l share the shell and have s of opposite sign, so the quartic is evaluated once
// per PAIR as an even and an odd part in t = s^2,
//   E = g0 + t (g2 + t/24),  O = s (g1 + t/6),   f_eq(l) = E + O,  f_eq(36-l) = E - O
// (10 FP64 operations per pair including s and the two relaxations, against 12 for two Horner evaluations, and
// two independent dependency chains per pair instead of one per population).  The 18 pairs are processed in four
// batches of shells, stage by stage across the pairs of a batch, so that 8-12 independent chains are in flight per
// thread and only one batch's coefficients are live at a time (register pressure).
//   collision (rhs of eq. 5): keep = 1 - 1/tau, scale = rho/tau, load = post-propagate f
//   plain equilibrium:                      keep = 0,         scale = rho
// WIDE = true: shells {0,1,2} {3,5,6} {4} {7}, 4-6 pairs per batch (kernels with ~168 registers); WIDE = false: one
// shell per batch, 2-4 pairs (kernels held to 128 registers).  Batching changes the schedule only: every value is
// the same expression either way, so the two forms are bit-identical.
template <bool WIDE>
__host__ __device__ constexpr int shell_batch(int slot)
{
    return !WIDE ? slot : slot <= 2 ? 0 : slot == 4 ? 2 : slot == 7 ? 3 : 1;
}

template <bool KEEP, bool WIDE = false, class Load, class Store>
__device__ __forceinline__ void equilibrium_blend_from(Load &&load, Store &&store, double keep, double scale,
                                                       double ux, double uz, double T)
{
    const double theta = T - 1.0;
    const double q = ux * ux + uz * uz;
    const double b1 = 1.0 - 0.5 * q;             // shell-independent parts
    const double b0 = b1 + 0.125 * (q * q);
    const double b2 = 0.5 - 0.25 * q;
    // s = e_x A + e_z B with A = r u_x, B = r u_z
    const double A1 = c_lat[0] * ux, B1 = c_lat[0] * uz;
    const double A[4] = {0.0, A1, 2.0 * A1, 3.0 * A1};
    const double B[4] = {0.0, B1, 2.0 * B1, 3.0 * B1};
    constexpr int REST = NPOP / 2;               // l = 18, e = (0, 0)

    static_for<0, (WIDE ? 4 : 8)>([&](auto BI) {
        constexpr int bi = decltype(BI)::value;
        double g0[8], g1[8], g2[8], g3[8], g4[8];                    // per shell of the batch (others never touched)
        static_for<0, 8>([&](auto S) {
            constexpr int sl = decltype(S)::value;
            if constexpr (shell_batch<WIDE>(sl) == bi) {
                const ShellConst &c = c_shell[sl];
                const double ws = scale * c.w;
                g0[sl] = ws * fma(theta, fma(theta, c.k3, fma(q, c.k2, c.k1)), b0);
                g1[sl] = ws * fma(theta, c.k4, b1);
                g2[sl] = ws * fma(theta, c.k5, b2);
                g3[sl] = ws * c_lat[2];
                g4[sl] = ws * c_lat[3];
            }
        });
        if constexpr (bi == 0) {
            if constexpr (KEEP) store(std::integral_constant<int, REST>{}, fma(keep, load(std::integral_constant<int, REST>{}), g0[0]));
            else store(std::integral_constant<int, REST>{}, g0[0]);
        }
        // pairs (l, 36 - l), l = 19..36, of the shells of this batch: stage by stage
        double s[NPOP], t[NPOP], ev[NPOP], od[NPOP];
        static_for<REST + 1, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            if constexpr (shell_batch<WIDE>(shell_slot(pop_e2(l))) == bi) {
                constexpr int ex = pop_ex(l), ez = pop_ez(l);
                constexpr int ax = ex < 0 ? -ex : ex, az = ez < 0 ? -ez : ez;
                if constexpr (ez == 0) s[l] = ex > 0 ? A[ax] : -A[ax];
                else if constexpr (ex == 0) s[l] = ez > 0 ? B[az] : -B[az];
                else s[l] = (ex > 0 ? A[ax] : -A[ax]) + (ez > 0 ? B[az] : -B[az]);
                t[l] = s[l] * s[l];
            }
        });
        static_for<REST + 1, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            constexpr int sl = shell_slot(pop_e2(l));
            if constexpr (shell_batch<WIDE>(sl) == bi) {
                ev[l] = fma(g4[sl], t[l], g2[sl]);
                od[l] = fma(g3[sl], t[l], g1[sl]);
            }
        });
        static_for<REST + 1, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            constexpr int sl = shell_slot(pop_e2(l));
            if constexpr (shell_batch<WIDE>(sl) == bi) {
                ev[l] = fma(ev[l], t[l], g0[sl]);
                od[l] = od[l] * s[l];
            }
        });
        static_for<REST + 1, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            if constexpr (shell_batch<WIDE>(shell_slot(pop_e2(l))) == bi) {
                using LB = std::integral_constant<int, NPOP - 1 - l>;
                if constexpr (KEEP) {
                    store(L, fma(keep, load(L), ev[l]) + od[l]);
                    store(LB{}, fma(keep, load(LB{}), ev[l]) - od[l]);
                } else {
                    store(L, ev[l] + od[l]);
                    store(LB{}, ev[l] - od[l]);
                }
            }
        });
    });
}

template <bool KEEP, bool WIDE = false>
__device__ __forceinline__ void equilibrium_blend(const double (&fin)[NPOP], double (&out)[NPOP], double keep,
                                                  double scale, double ux, double uz, double T)
{
    equilibrium_blend_from<KEEP, WIDE>([&](auto L) { return fin[decltype(L)::value]; },
                                 [&](auto L, double v) { out[decltype(L)::value] = v; }, keep, scale, ux, uz, T);
}

// Isothermal no-slip wall rows (reading 19; "bc ... adjusts population values at sites with
// coordinates z = 0, 1, 2 and z = Lz-3, Lz-2, Lz-1"): the equilibrium part of the post-propagate populations is moved
// to the wall state, density and non-equilibrium part kept,
//   f <- f - f_eq(rho*, u*, T*) + f_eq(rho*, u_w, T_w),   u_w = (0, g/2),  T_w = T_wall - g^2/8,
// the kinetic moments that PAPER.md:94 maps to u^(H) = 0, T^(H) = T_wall.  The collision then runs unchanged.
__device__ __forceinline__ void wall_adjust(double (&f)[NPOP], double uwz, double Tw)
{
    const Kinetic k = kinetic_moments(f);
    equilibrium_blend<true>(f, f, 1.0, -k.rho, k.ux, k.uz, k.T);
    equilibrium_blend<true>(f, f, 1.0, k.rho, 0.0, uwz, Tw);
}

// One collision: moments of the post-propagate populations, equilibrium shifted by
// u' = u + g_vec tau = (u_x, u_z - g tau), T' = T + tau (dt - tau) g^2 / d, BGK relaxation.
//   omega = dt/tau, gtau = g tau, dT = tau (1 - tau) g^2 / 2.
// `load` is called twice per population (moments, then relaxation), `store` once.
template <class Load, class Store>
__device__ __forceinline__ void collide_from(Load &&load, Store &&store, double omega, double gtau, double dT)
{
    const Kinetic k = kinetic_from_raw(raw_moments_from(load));
    equilibrium_blend_from<true>(load, store, 1.0 - omega, omega * k.rho, k.ux, k.uz - gtau, k.T + dT);
}

__device__ __forceinline__ void collide_site(double (&f)[NPOP], double omega, double gtau, double dT)
{
    collide_from([&](auto L) { return f[decltype(L)::value]; },
                 [&](auto L, double v) { f[decltype(L)::value] = v; }, omega, gtau, dT);
}

}  // namespace d2q37
