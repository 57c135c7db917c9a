// lbm_aux.cuh -- initial states, layout conversion, wrap-column refresh, z-slab messages and the moments /
// diagnostics kernels (row a6).
#pragma once
#include <cstdint>

#include "d2q37.cuh"
#include "lbm_step.cuh"

namespace lbm {

// The stored lattice as the aux kernels see it.  `buf` points at site (0, 0) of population 0 (the wrap columns of
// DESIGN.md section 5 lie at negative column offsets).  Dense user arrays cover the OWNED rows only: rows
// [k0, k0 + nz) of the stored lattice (a whole lattice owns all its rows; a z-slab also stores ghost rows).
struct Layout {
    int Lx, Lz, pitch;
    long long plane;
    int k0, nz;
    bool layout_m;      // in-place path after an odd number of steps (lbm_step.cuh)
};

constexpr int AUX_TX = 128;  // threads per block along x for the per-site aux kernels
constexpr int RED_T = 256;   // threads per block of the row reductions

// the 37 populations of stored site (i, k), whatever the layout
__device__ __forceinline__ void load_site(const double *src, const Layout &g, int i, int k, double (&f)[NPOP])
{
    each_stored_site(src, g.Lx, g.Lz, g.pitch, g.plane, g.layout_m, i, k,
                     [&](auto L, const double *p) { f[decltype(L)::value] = __ldg(p); });
}

__device__ __forceinline__ void store_site(double *dst, const Layout &g, int i, int k, const double (&f)[NPOP])
{
    double *p = dst + (long long)k * g.pitch + i;
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        p[(long long)l * g.plane] = f[l];
    });
}

// populations = f_eq(rho, u, T) of given kinetic fields (dense [nz][Lx]); grid.y = nz
__global__ void __launch_bounds__(AUX_TX)
init_equilibrium_kernel(double *dst, Layout g, const double *__restrict__ rho, const double *__restrict__ ux,
                        const double *__restrict__ uz, const double *__restrict__ T)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y;
    if (i >= g.Lx) return;
    const long long s = (long long)j * g.Lx + i;
    double f[NPOP];
    d2q37::equilibrium_blend<false>(f, f, 0.0, rho[s], ux[s], uz[s], T[s]);
    store_site(dst, g, i, g.k0 + j, f);
}

// Hydrostatic three-layer state, eq. 1-2 with tanh-smoothed jumps;
// DESIGN.md reading 11.  z_k = k - (Lz-1)/2 in sites of the GLOBAL lattice, one site = r length units, beta = 1/T0.
struct RtArgs {
    double g, beta_d, beta_m, beta_u, rho_m, delta, w;
    int Lz_glob;        // height of the whole lattice
    int zshift;         // global row of stored row 0 (0 for a whole lattice; a slab stores ghost rows below its own)
};

__device__ __forceinline__ double rt_lncosh(double s)
{
    const double a = fabs(s);
    return a + log1p(exp(-2.0 * a)) - 0.69314718055994530941723212145818;
}
__device__ __forceinline__ double rt_step(double z, double a, double w)
{
    if (w > 0.0) return 0.5 * (1.0 + tanh((z - a) / w));
    return z > a ? 1.0 : (z < a ? 0.0 : 0.5);
}
__device__ __forceinline__ double rt_step_integral(double z, double a, double w)
{
    if (w > 0.0) return 0.5 * (z + w * rt_lncosh((z - a) / w) - w * rt_lncosh(a / w));
    return fmax(z - a, 0.0) - fmax(-a, 0.0);
}

// grid.y = all stored rows (a slab's ghost rows are initialised from the same closed form)
__global__ void __launch_bounds__(AUX_TX)
init_rt_kernel(double *dst, Layout g, RtArgs p, const double *__restrict__ h_lo, const double *__restrict__ h_hi)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, k = blockIdx.y;
    if (i >= g.Lx) return;
    const double z = (double)(k + p.zshift) - 0.5 * (double)(p.Lz_glob - 1);
    const double a_lo = -0.5 * p.delta + h_lo[i], a_hi = 0.5 * p.delta + h_hi[i];
    const double dlo = p.beta_m - p.beta_d, dhi = p.beta_u - p.beta_m;
    const double beta = p.beta_d + dlo * rt_step(z, a_lo, p.w) + dhi * rt_step(z, a_hi, p.w);
    const double beta0 = p.beta_d + dlo * rt_step(0.0, a_lo, p.w) + dhi * rt_step(0.0, a_hi, p.w);
    const double lnp = log(p.rho_m / beta0) -
                       p.g * D2Q37_R *
                           (p.beta_d * z + dlo * rt_step_integral(z, a_lo, p.w) + dhi * rt_step_integral(z, a_hi, p.w));
    const double T0 = 1.0 / beta, rho0 = exp(lnp) * beta;
    // stored state: u = (0, -g/2), T = T0 - g^2/8, so that u^(H) = 0 and T^(H) = T0
    double f[NPOP];
    d2q37::equilibrium_blend<false>(f, f, 0.0, rho0, 0.0, -0.5 * p.g, T0 - 0.125 * p.g * p.g);
    store_site(dst, g, i, k, f);
}

// canonical dense [nl][nz][Lx] (populations l0 .. l0+nl-1)  <->  the stored lattice; grid = (ceil(Lx/AUX_TX), nz, nl).
// pack always writes the ordinary layout; unpack reads either layout.
__global__ void __launch_bounds__(AUX_TX) pack_kernel(double *dst, Layout g, const double *__restrict__ dense, int l0)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y, l = l0 + blockIdx.z;
    if (i >= g.Lx) return;
    dst[(long long)l * g.plane + (long long)(g.k0 + j) * g.pitch + i] = dense[((long long)blockIdx.z * g.nz + j) * g.Lx + i];
}
__global__ void __launch_bounds__(AUX_TX) unpack_kernel(const double *__restrict__ src, Layout g, double *dense, int l0)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y, l = l0 + blockIdx.z;
    if (i >= g.Lx) return;
    const double *p = nullptr;
    each_stored_site(src, g.Lx, g.Lz, g.pitch, g.plane, g.layout_m, i, g.k0 + j, [&](auto L, const double *q) {
        if (decltype(L)::value == l) p = q;
    });
    dense[((long long)blockIdx.z * g.nz + j) * g.Lx + i] = *p;
}

// dense [37][nk][ni] window of the stored state: rows k0 .. k0+nk-1 of the OWN rows, columns i0 .. i0+ni-1 (mod Lx);
// grid = (ceil(ni/AUX_TX), nk, NPOP)
__global__ void __launch_bounds__(AUX_TX)
window_kernel(const double *__restrict__ src, Layout g, int k0, int nk, int i0, int ni, double *dense)
{
    const int c = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y, l = blockIdx.z;
    if (c >= ni) return;
    int i = (i0 + c) % g.Lx;
    if (i < 0) i += g.Lx;
    const double *p = nullptr;
    each_stored_site(src, g.Lx, g.Lz, g.pitch, g.plane, g.layout_m, i, g.k0 + k0 + j, [&](auto L, const double *q) {
        if (decltype(L)::value == l) p = q;
    });
    dense[((long long)l * nk + j) * ni + c] = *p;
}

// a1 for the two-step kernel's TMA loads: the XW wrap columns on either side of a row hold the periodic images
// (column j < 0 holds column j mod Lx, column Lx + j holds column j mod Lx).  The two-step kernel's consumers keep
// them current themselves; this kernel refreshes them after anything else has written the lattice.
// grid = Lz, block = NPOP x 2 XW threads (one row of all populations per block).
template <int XW>
__global__ void __launch_bounds__(2 * XW * NPOP) wrap_columns_kernel(double *buf, Layout g)
{
    double *row = buf + (long long)(threadIdx.x / (2 * XW)) * g.plane + (long long)blockIdx.x * g.pitch;
    const int t = threadIdx.x % (2 * XW);
    const int j = t < XW ? t - XW : g.Lx + t - XW;           // halo column
    int s = j % g.Lx;
    if (s < 0) s += g.Lx;
    row[j] = row[s];
}

// z-slab messages (26 population-rows per direction).  The neighbour on `side` reads from its ghost
// row at distance d = 1, 2, 3 only the populations that move towards it by at least d rows: 15 + 8 + 3 of them.
// msg = [26][Lx]; entry j is population sel.l[j] of stored row sel.row[j].  grid = (ceil(Lx/AUX_TX), 26).
struct SlabRows {
    int row[26];
    int l[26];
};
__global__ void __launch_bounds__(AUX_TX) slab_pack_kernel(const double *__restrict__ src, Layout g, SlabRows sel, double *msg)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y;
    if (i >= g.Lx) return;
    msg[(long long)j * g.Lx + i] = src[(long long)sel.l[j] * g.plane + (long long)sel.row[j] * g.pitch + i];
}
__global__ void __launch_bounds__(AUX_TX) slab_unpack_kernel(double *dst, Layout g, SlabRows sel, const double *__restrict__ msg)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y;
    if (i >= g.Lx) return;
    dst[(long long)sel.l[j] * g.plane + (long long)sel.row[j] * g.pitch + i] = msg[(long long)j * g.Lx + i];
}

// z-slab messages of the two-step path: whole rows, all 37 populations, wrap columns included (the receiver's TMA
// boxes read them), `nrows` consecutive stored rows from `row0`.  msg = [nrows][NPOP][Lx + 2 XW].
// grid = (ceil((Lx + 2 XW)/AUX_TX), nrows, NPOP)
template <int XW, bool PACK>
__global__ void __launch_bounds__(AUX_TX) slab_rows_kernel(double *buf, Layout g, int row0, double *msg)
{
    const int c = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y, l = blockIdx.z;
    const int wcols = g.Lx + 2 * XW;
    if (c >= wcols) return;
    double *p = buf + (long long)l * g.plane + (long long)(row0 + j) * g.pitch + (c - XW);
    double *m = msg + ((long long)j * NPOP + l) * wcols + c;
    if (PACK) *m = *p;
    else *p = *m;
}

// Hydrodynamic fields of the stored (post-collision) state: rho, u^(H) = u - g_vec dt/2 = (u_x, u_z + g/2),
// T^(H) = T + g^2/8 (PAPER.md:94 applied after the collision's u -> u + g_vec dt; reading 8).  grid.y = nz
__global__ void __launch_bounds__(AUX_TX)
moments_kernel(const double *__restrict__ src, Layout g, double grav, double *rho, double *ux, double *uz, double *T)
{
    const int i = blockIdx.x * AUX_TX + threadIdx.x, j = blockIdx.y;
    if (i >= g.Lx) return;
    double f[NPOP];
    load_site(src, g, i, g.k0 + j, f);
    const d2q37::Kinetic m = d2q37::kinetic_moments(f);
    const long long s = (long long)j * g.Lx + i;
    if (rho) rho[s] = m.rho;
    if (ux) ux[s] = m.ux;
    if (uz) uz[s] = m.uz + 0.5 * grav;
    if (T) T[s] = m.T + 0.125 * grav * grav;
}

// deterministic block sum (fixed shuffle tree, fixed warp order); result valid in thread 0
__device__ __forceinline__ double block_sum(double v, double *smem /* RED_T/32 doubles */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) smem[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < RED_T / 32; ++w) t += smem[w];
    __syncthreads();
    return t;
}

// One pass over the lattice for every per-row diagnostic (one block per owned row, deterministic):
//   out[0][j] = Tbar(j)  = <T^(H)>_x
//   out[1][j] = Trms(j)  = sqrt(<(T - <T>_x)^2>_x)         (Fig. 8)
//   out[2][j] = Ekbar(j) = <E_k>_x, E_k = rho |u^(H)|^2/2  (Fig. 9; reading 17)
//   out[3][j] = Ekrms(j)
//   out[4..7][j] = row sums of the raw integer-velocity moments sum f, sum e_x f, sum e_z f, sum |e|^2 f
// WANT_RMS = false skips the second pass over the row (the squared deviations about the row means).  The second pass
// needs every site's T and E_k again: with keep != 0 the first pass leaves them in dynamic shared memory (2 Lx doubles;
// the block is alone on its SM anyway, 226 registers x 256 threads) -- the same values the recomputation gives, so the
// results are bit-identical -- else it re-reads the row, which comes from DRAM, not L2, on large lattices (ncu:
// 19.7 GB per launch at 4096x8192 = twice the lattice, profiles/r3_a6_kernels.md).
template <bool WANT_RMS>
__global__ void __launch_bounds__(RED_T) row_diagnostics_kernel(const double *__restrict__ src, Layout g, double grav, double *out,
                                                                int keep)
{
    extern __shared__ double rowbuf[];                       // [2][Lx] if WANT_RMS && keep
    __shared__ double sm[RED_T / 32];
    __shared__ double mean[2];
    const int j = blockIdx.x, k = g.k0 + j;
    double aT = 0.0, aE = 0.0, a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int i = threadIdx.x; i < g.Lx; i += RED_T) {
        double f[NPOP];
        load_site(src, g, i, k, f);
        const d2q37::RawMoments r = d2q37::raw_moments(f);
        const d2q37::Kinetic m = d2q37::kinetic_from_raw(r);
        const double uz = m.uz + 0.5 * grav;
        const double Ti = m.T + 0.125 * grav * grav, Ei = 0.5 * m.rho * (m.ux * m.ux + uz * uz);
        aT += Ti;
        aE += Ei;
        a0 += r.m0; a1 += r.jx; a2 += r.jz; a3 += r.m2;
        if constexpr (WANT_RMS)
            if (keep) { rowbuf[i] = Ti; rowbuf[g.Lx + i] = Ei; }
    }
    const double sT = block_sum(aT, sm), sE = block_sum(aE, sm);
    const double s0 = block_sum(a0, sm), s1 = block_sum(a1, sm), s2 = block_sum(a2, sm), s3 = block_sum(a3, sm);
    if (threadIdx.x == 0) {
        mean[0] = sT / (double)g.Lx; mean[1] = sE / (double)g.Lx;
        out[j] = mean[0];
        out[2 * g.nz + j] = mean[1];
        out[4 * g.nz + j] = s0; out[5 * g.nz + j] = s1; out[6 * g.nz + j] = s2; out[7 * g.nz + j] = s3;
    }
    if constexpr (WANT_RMS) {
        __syncthreads();
        const double mT = mean[0], mE = mean[1];
        double vT = 0.0, vE = 0.0;
        for (int i = threadIdx.x; i < g.Lx; i += RED_T) {
            double dT, dE;
            if (keep) {                                      // written by this same thread in the first pass
                dT = rowbuf[i] - mT;
                dE = rowbuf[g.Lx + i] - mE;
            } else {
                double f[NPOP];
                load_site(src, g, i, k, f);
                const d2q37::Kinetic m = d2q37::kinetic_moments(f);
                const double uz = m.uz + 0.5 * grav;
                dT = m.T + 0.125 * grav * grav - mT;
                dE = 0.5 * m.rho * (m.ux * m.ux + uz * uz) - mE;
            }
            vT += dT * dT;
            vE += dE * dE;
        }
        const double qT = block_sum(vT, sm), qE = block_sum(vE, sm);
        if (threadIdx.x == 0) {
            out[g.nz + j] = sqrt(qT / (double)g.Lx);
            out[3 * g.nz + j] = sqrt(qE / (double)g.Lx);
        }
    }
}

// tent map of eq. 9, zero outside (0,1)
__device__ __forceinline__ double tent(double b)
{
    if (b <= 0.0 || b >= 1.0) return 0.0;
    return b < 0.5 ? 2.0 * b : 2.0 * (1.0 - b);
}

// Second stage, single block over the nz owned rows of the per-row array `rows` (row_diagnostics_kernel):
//   res[0] = L_u, res[1] = L_d of eq. 12 from Tbar, in sites (skipped if T_m == T_u or T_d == T_m)
//   res[2..5] = sum f, sum c_x f, sum c_z f, sum |c|^2 f, c = r e
__global__ void __launch_bounds__(RED_T)
final_diagnostics_kernel(const double *__restrict__ rows, int nz, double T_d, double T_m, double T_u, double *res)
{
    __shared__ double sm[RED_T / 32];
    const bool widths = T_m != T_u && T_d != T_m;
    double lu = 0.0, ld = 0.0, a[4] = {0, 0, 0, 0};
    for (int k = threadIdx.x; k < nz; k += RED_T) {
        if (widths) {
            const double tb = rows[k];
            lu += tent((tb - T_u) / (T_m - T_u));
            ld += tent((tb - T_m) / (T_d - T_m));
        }
        for (int j = 0; j < 4; ++j) a[j] += rows[(long long)(4 + j) * nz + k];
    }
    const double su = block_sum(lu, sm), sd = block_sum(ld, sm);
    const double s0 = block_sum(a[0], sm), s1 = block_sum(a[1], sm), s2 = block_sum(a[2], sm), s3 = block_sum(a[3], sm);
    if (threadIdx.x == 0) {
        res[0] = su; res[1] = sd;
        res[2] = s0; res[3] = D2Q37_R * s1; res[4] = D2Q37_R * s2; res[5] = D2Q37_R2 * s3;
    }
}

// FP64 peak probe (include/lbm.h lbm_fp64_peak): 8 independent DFMA chains per thread, 8 warps per SM sub-partition.
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *sink, int iters, double a, double b)
{
    double x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = a * (threadIdx.x + j);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 16; ++r)
#pragma unroll
            for (int j = 0; j < 8; ++j) x[j] = fma(x[j], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += x[j];
    if (s == 12345.678) sink[0] = s;      // never true: keeps the chains alive
}

}  // namespace lbm
