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
struct RawMoments {
    double m0, jx, jz, m2;
};

__device__ __forceinline__ RawMoments raw_moments(const double (&f)[NPOP])
{
    double C[7] = {0, 0, 0, 0, 0, 0, 0}, R[7] = {0, 0, 0, 0, 0, 0, 0};
    static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        C[pop_ex(l) + 3] += f[l];
        R[pop_ez(l) + 3] += f[l];
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

// Kinetic moments of eq. 7: rho = sum f, rho u = sum c f, d rho T = sum |c-u|^2 f, d = 2,
// with c = r e:  u = r j / rho,  T = (r^2 m2 / rho - |u|^2) / 2.
struct Kinetic {
    double rho, ux, uz, T;
};

__device__ __forceinline__ Kinetic kinetic_moments(const double (&f)[NPOP])
{
    const RawMoments m = raw_moments(f);
    const double inv = 1.0 / m.m0;
    Kinetic k;
    k.rho = m.m0;
    k.ux = (D2Q37_R * m.jx) * inv;
    k.uz = (D2Q37_R * m.jz) * inv;
    k.T = 0.5 * ((D2Q37_R2 * m.m2) * inv - (k.ux * k.ux + k.uz * k.uz));
    return k;
}

// out[l] = keep * fin[l] + scale * f_eq_l(rho = 1, u, T), for all l.
//
// f_eq is the 4th-order Hermite projection of the Maxwellian on this quadrature ("local Maxwellian",
// PAPER.md:80; reading 3).  With s = c.u, q = |u|^2, theta = T - 1, D = 2 it is a quartic in s
// whose coefficients depend on the shell |c|^2 only:
//   f_eq / (w rho) = g0 + g1 s + g2 s^2 + s^3/6 + s^4/24
//   g0 = 1 - q/2 + q^2/8 + theta [ (c2-2)/2 + q (4-c2)/4 ] + theta^2 (c2^2 - 8 c2 + 8)/8
//   g1 = 1 - q/2 + theta (c2-4)/2
//   g2 = 1/2 - q/4 + theta (c2-6)/4
// so each population costs one Horner evaluation (4 FMA) plus the relaxation FMA.
//   collision (rhs of eq. 5): keep = 1 - 1/tau, scale = rho/tau, fin = post-propagate f
//   plain equilibrium:                      keep = 0,         scale = rho
template <bool KEEP>
__device__ __forceinline__ void equilibrium_blend(const double (&fin)[NPOP], double (&out)[NPOP], double keep,
                                                  double scale, double ux, double uz, double T)
{
    const double theta = T - 1.0;
    const double q = ux * ux + uz * uz;
    const double b1 = 1.0 - 0.5 * q;             // shell-independent parts
    const double b0 = b1 + 0.125 * (q * q);
    const double b2 = 0.5 - 0.25 * q;
    // s = e_x A + e_z B with A = r u_x, B = r u_z
    const double A1 = D2Q37_R * ux, B1 = D2Q37_R * uz;
    const double A[4] = {0.0, A1, 2.0 * A1, 3.0 * A1};
    const double B[4] = {0.0, B1, 2.0 * B1, 3.0 * B1};

    double G0[8], G1[8], G2[8], G3[8], G4[8];
    static_for<0, 8>([&](auto S) {
        constexpr int sl = decltype(S)::value;
        constexpr double c2 = D2Q37_R2 * shell_e2(sl);
        constexpr double k1 = 0.5 * (c2 - 2.0), k2 = 0.25 * (4.0 - c2), k3 = 0.125 * (c2 * c2 - 8.0 * c2 + 8.0);
        constexpr double k4 = 0.5 * (c2 - 4.0), k5 = 0.25 * (c2 - 6.0);
        const double ws = scale * shell_weight(shell_e2(sl));
        const double g0 = fma(theta, fma(theta, k3, fma(q, k2, k1)), b0);
        const double g1 = fma(theta, k4, b1);
        const double g2 = fma(theta, k5, b2);
        G0[sl] = ws * g0;
        G1[sl] = ws * g1;
        G2[sl] = ws * g2;
        G3[sl] = ws * (1.0 / 6.0);
        G4[sl] = ws * (1.0 / 24.0);
    });

    static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int ex = pop_ex(l), ez = pop_ez(l), sl = shell_slot(pop_e2(l));
        constexpr int ax = ex < 0 ? -ex : ex, az = ez < 0 ? -ez : ez;
        double s;
        if constexpr (ex == 0 && ez == 0) s = 0.0;
        else if constexpr (ez == 0) s = ex > 0 ? A[ax] : -A[ax];
        else if constexpr (ex == 0) s = ez > 0 ? B[az] : -B[az];
        else s = (ex > 0 ? A[ax] : -A[ax]) + (ez > 0 ? B[az] : -B[az]);
        double p;
        if constexpr (ex == 0 && ez == 0) p = G0[sl];
        else p = fma(fma(fma(fma(G4[sl], s, G3[sl]), s, G2[sl]), s, G1[sl]), s, G0[sl]);
        if constexpr (KEEP) out[l] = fma(keep, fin[l], p);
        else out[l] = p;
    });
}

// One collision: moments of the post-propagate populations, equilibrium shifted by
// u' = u + g_vec tau = (u_x, u_z - g tau), T' = T + tau (dt - tau) g^2 / d, BGK relaxation.
//   omega = dt/tau, gtau = g tau, dT = tau (1 - tau) g^2 / 2.
__device__ __forceinline__ void collide_site(double (&f)[NPOP], double omega, double gtau, double dT)
{
    const Kinetic k = kinetic_moments(f);
    equilibrium_blend<true>(f, f, 1.0 - omega, omega * k.rho, k.ux, k.uz - gtau, k.T + dT);
}

}  // namespace d2q37
