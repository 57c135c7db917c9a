// lbm_step.cuh -- the fused propagate + bc + collide kernel (one launch per time step).
//
// Store: structure of arrays, f[l][k][i] at  l*plane + k*pitch + i  doubles,
// x fastest, rows padded to a multiple of 16 doubles (128 B), two copies (src = prv, dst = nxt of
// PAPER.md:110).  One thread updates one site:
//   a1/a2  pull-propagate with periodic x: 37 gathers from src at (i - e_x mod Lx, k - e_z)
//   a3     walls: a source row below 0 / above Lz-1 is replaced by the mirror row and the opposite
//          population (pure index remap, block-uniform because a block works on one row)
//   a4     collide in registers (d2q37.cuh), 37 aligned stores to dst
// No halo rows or wrap columns are stored: the wrap is seven per-thread column indices, the walls are
// seven block-uniform (row, flip) pairs, so interior blocks run a branch-free path.
#pragma once
#include <cstdint>

#include "d2q37.cuh"

namespace lbm {

using d2q37::NPOP;

constexpr int XH = 16;   // spare columns stored on either side of every row (128 bytes: x = 0 stays on a 128-byte line)
constexpr int XW = 8;    // ... of which the nearest XW hold the periodic images (the two-step kernel's boxes reach 8 out)

struct StepArgs {
    const double *src;
    double *dst;
    int Lx, Lz;
    int pitch;          // doubles per row
    long long plane;    // doubles per population plane
    double omega;       // dt / tau
    double gtau;        // g tau
    double dT;          // tau (1 - tau) g^2 / 2
    // isothermal no-slip walls (wall_kind 1, reading 19): flags per wall (0 for wall_kind 0 and for the
    // open side of a z-slab), the imposed kinetic state u_w = (0, uwz), T_w per wall
    int iso_lo, iso_hi;
    double uwz, Tw_lo, Tw_hi;
    int wrap_store;     // two-step kernel: the consumers of the seam strips maintain the wrap columns (Lx >= 2 XW)
    int w;              // two-step kernel: columns per strip
    int zbase, zend;    // two-step kernel: stored rows [zbase, zend) are updated (a whole lattice: [0, Lz); a z-slab: its own rows)
    int zsplit, zbase2, zend2;   // two-step kernel: chunk rows blockIdx.y >= zsplit cover a SECOND row range [zbase2, zend2) (the two
                                 // edge zones of a z-slab in one launch); zsplit = INT_MAX: one range
    int ztrim;          // two-step kernel: chunk c covers rows zbase + [c ZC - ztrim, (c+1) ZC - ztrim) (chunk 0 from 0): wall_kind 1
    // byte offset of population l's pull source relative to the site's own address in plane 0, for sites that
    // need neither wrap nor wall remap: 8 (l plane - e_lz pitch - e_lx).  Host-computed (fill_offsets) so that
    // the kernel adds one opaque uniform constant per load instead of re-deriving it.
    long long gbyte[NPOP];
};

inline void fill_offsets(StepArgs &a)
{
    for (int l = 0; l < NPOP; ++l)
        a.gbyte[l] = 8 * ((long long)l * a.plane - (long long)d2q37::pop_ez(l) * a.pitch - d2q37::pop_ex(l));
}

// Streaming load / store: every population value is read once and written once per step.  Plain
// ld.global.nc / st.global: explicit cache operators (L1::no_allocate, .cs, L2 evict_first) were measured and
// make no difference (profiles/r1_variants.md), and the builtin forms let the compiler fold the constant part
// of each address into the instruction's immediate.
__device__ __forceinline__ double ld_stream(const double *p) { return __ldg(p); }
__device__ __forceinline__ void st_stream(double *p, double v) { *p = v; }

// Pull sources of site (i, k): calls fn(L, p) for l = 0..36 in ascending order, p = address in src of the
// population that propagation brings to (i, k) as population l.  WALL = false: rows 3..Lz-4, no remap.
template <bool WALL, class Fn>
__device__ __forceinline__ void each_source_site(const StepArgs &a, int i, int k, Fn &&fn)
{
    // periodic x (a1): wrapped source column for each e_x in -3..3
    int col[7];
#pragma unroll
    for (int d = -3; d <= 3; ++d) {
        int c = i - d;
        c += (c < 0) ? a.Lx : 0;
        c -= (c >= a.Lx) ? a.Lx : 0;
        col[d + 3] = c;
    }
    // source row for each e_z in -3..3, with the wall remap (a3)
    long long rowoff[7];
    bool flip[7];
#pragma unroll
    for (int d = -3; d <= 3; ++d) {
        int ks = k - d;
        bool fl = false;
        if (WALL) {
            if (ks < 0) { ks = -1 - ks; fl = true; }
            else if (ks >= a.Lz) { ks = 2 * a.Lz - 1 - ks; fl = true; }
        }
        rowoff[d + 3] = (long long)ks * a.pitch;
        flip[d + 3] = fl;
    }
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int ex = d2q37::pop_ex(l), ez = d2q37::pop_ez(l);
        int ls = l;
        if (WALL) ls = flip[ez + 3] ? (NPOP - 1 - l) : l;
        fn(L, a.src + (long long)ls * a.plane + rowoff[ez + 3] + col[ex + 3], WALL && flip[ez + 3]);
    });
}

// Fast path for sites with 3 <= i < Lx-3 and 3 <= k < Lz-3 (no wrap, no wall): every source address is the
// site's own address plus an offset that depends on kernel arguments only, so the offsets live in uniform
// registers and each load costs one 64-bit add (the e_x shift is an immediate).
template <class Fn>
__device__ __forceinline__ void each_source_interior(const StepArgs &a, int i, int k, Fn &&fn)
{
    const char *p = reinterpret_cast<const char *>(a.src + (long long)k * a.pitch + i);
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        fn(L, reinterpret_cast<const double *>(p + a.gbyte[l]), false);
    });
}

// dispatch on the site's position: interior / periodic seam / wall rows
template <class Fn>
__device__ __forceinline__ void each_source_any(const StepArgs &a, int i, int k, Fn &&fn)
{
    const bool bulk_z = k >= 3 && k < a.Lz - 3;
    if (bulk_z && i >= 3 && i < a.Lx - 3) each_source_interior(a, i, k, fn);
    else if (bulk_z) each_source_site<false>(a, i, k, fn);
    else each_source_site<true>(a, i, k, fn);
}

// Gather the 37 post-propagate populations of site (i, k) into registers.
__device__ __forceinline__ void gather_any(const StepArgs &a, int i, int k, double (&f)[NPOP])
{
    each_source_any(a, i, k, [&](auto L, const double *p, bool) { f[decltype(L)::value] = ld_stream(p); });
}

// wall_kind 1: rows 0..2 / Lz-3..Lz-1 next to an isothermal wall get the wall state imposed after the gather (a3)
template <bool ISO>
__device__ __forceinline__ void wall_rows_adjust(const StepArgs &a, int k, double (&f)[NPOP])
{
    if constexpr (ISO) {
        if (a.iso_lo && k < 3) d2q37::wall_adjust(f, a.uwz, a.Tw_lo);
        else if (a.iso_hi && k >= a.Lz - 3) d2q37::wall_adjust(f, a.uwz, a.Tw_hi);
    }
}

__device__ __forceinline__ void scatter_site(const StepArgs &a, int i, int k, const double (&f)[NPOP])
{
    double *p = a.dst + (long long)k * a.pitch + i;
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        st_stream(p + (long long)l * a.plane, f[l]);
    });
}

// One thread per site; a block covers TX consecutive columns of TZ consecutive rows of the row range [k0, k1),
// grid = (ceil(Lx/TX), ceil((k1-k0)/TZ)).  The wall test is per row, hence warp-uniform (TX is a multiple of 32).
// ISO = true: the instance for wall_kind 1 (the adjustment sits in a block-uniform branch taken by six rows).
template <int TX, int TZ, bool ISO>
__global__ void __launch_bounds__(TX *TZ, 512 / (TX * TZ)) step_kernel_site(const StepArgs a, const int k0, const int k1)
{
    const int i = blockIdx.x * TX + threadIdx.x;
    const int k = k0 + blockIdx.y * TZ + threadIdx.y;
    if (i >= a.Lx || k >= k1) return;
    double f[NPOP];
    gather_any(a, i, k, f);
    wall_rows_adjust<ISO>(a, k, f);
    d2q37::collide_site(f, a.omega, a.gtau, a.dT);
    scatter_site(a, i, k, f);
}

// ---- small lattices: n time steps in ONE launch.  A lattice of a few thousand sites is updated in less time than a
// kernel launch takes (64 x 128: ~1 us of work, ~4 us per launched step), so for lattices that fit one site per
// resident thread the whole step loop runs inside a persistent cooperative kernel: every thread owns one site, the
// two copies alternate, and the steps are separated by a grid-wide barrier (one atomic per block on a counter in
// global memory, polled with acquire loads; the block barrier before it and the fence make the block's stores
// visible).  Loads bypass L1 (the other copy was rewritten by other SMs a moment ago).  Same gather, same collision:
// bit-identical to n launches of the one-step kernel.
// The counter only grows.  The host sets it to BARRIER_START = 0xFFFFFFFF before every launch (a byte memset of 0xFF),
// so EVERY launch takes the counter through the 32-bit wrap at its first barrier, and the wait compares the signed
// distance to the target, which is right across the wrap as long as a launch adds fewer than 2^31 arrivals:
// lbm_step issues at most PERSIST_MAX_STEPS steps per launch (2^20 steps x at most a few hundred blocks < 2^29).
constexpr unsigned BARRIER_START = 0xFFFFFFFFu;
constexpr int PERSIST_MAX_STEPS = 1 << 20;
template <int TB, bool ISO>
__global__ void __launch_bounds__(TB) step_persistent_kernel(StepArgs a, double *buf0, double *buf1, int cur, const int nsteps,
                                                             unsigned *counter)
{
    const int site = blockIdx.x * TB + threadIdx.x;
    const int k = site / a.Lx, i = site - k * a.Lx;
    const bool live = k < a.Lz;
    for (int s = 0; s < nsteps; ++s, cur ^= 1) {
        a.src = cur ? buf1 : buf0;
        a.dst = cur ? buf0 : buf1;
        if (live) {
            double f[NPOP];
            each_source_site<true>(a, i, k, [&](auto L, const double *p, bool) { f[decltype(L)::value] = __ldcg(p); });
            wall_rows_adjust<ISO>(a, k, f);
            d2q37::collide_site(f, a.omega, a.gtau, a.dT);
            scatter_site(a, i, k, f);
        }
        if (s + 1 < nsteps) {                                // grid barrier
            __syncthreads();
            if (threadIdx.x == 0) {
                __threadfence();
                atomicAdd(counter, 1u);
                const unsigned target = BARRIER_START + (unsigned)(s + 1) * gridDim.x;     // modulo 2^32
                unsigned seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counter) : "memory");
                } while ((int)(seen - target) < 0);
            }
            __syncthreads();
        }
    }
}

// ---- in-place streaming: ONE lattice copy ("we keep in memory two copies of the lattice ... This choice
// requires more memory").  Every site reads 37 slots and writes its 37 results back into the SAME slots, so no slot
// is touched by two sites in a step and no second copy is needed.  Two alternating kernels:
//   layout N (after an even number of steps):  A[l][x] = F_l(x), the stored post-collision state;
//   EVEN step (N -> M): site x gathers f*_l(x) from the slots s(x,l) the ordinary pull reads (neighbour sites, wrap,
//       wall remap), collides, and writes F'_{36-l}(x) into s(x,l) -- for a wall-reflected gather (slot in the mirror
//       row, population 36-l) it writes F'_{(e_lx, -e_lz)}(x) instead, which is what makes the next step local;
//   layout M:  A[l][y] = F'_{36-l}(y + e_l)  (and the x-flipped variant for the reflected slots);
//   ODD step (M -> N): everything site x needs is at site x: f*_l(x) = A[36-l][x], or A[(e_lx, -e_lz)][x] where
//       the pull source row k - e_lz lies beyond a wall; collide; write F''_l(x) to A[l][x].
// Same gather values, same collision arithmetic: bit-identical to the two-copy kernels.
template <int TX, bool ISO>
__global__ void __launch_bounds__(TX, 512 / TX) step_inplace_even_kernel(const StepArgs a, const int k0, const int k1)
{
    const int i = blockIdx.x * TX + threadIdx.x;
    const int k = k0 + blockIdx.y;
    if (i >= a.Lx || k >= k1) return;
    double f[NPOP];
    gather_any(a, i, k, f);
    wall_rows_adjust<ISO>(a, k, f);
    d2q37::collide_site(f, a.omega, a.gtau, a.dT);
    each_source_any(a, i, k, [&](auto L, const double *p, bool reflected) {
        constexpr int l = decltype(L)::value;
        constexpr int lx = d2q37::pop_index(d2q37::pop_ex(l), -d2q37::pop_ez(l));
        st_stream(const_cast<double *>(p), reflected ? f[lx] : f[NPOP - 1 - l]);
    });
}

template <int TX, bool ISO>
__global__ void __launch_bounds__(TX, 512 / TX) step_inplace_odd_kernel(const StepArgs a, const int k0, const int k1)
{
    const int i = blockIdx.x * TX + threadIdx.x;
    const int k = k0 + blockIdx.y;
    if (i >= a.Lx || k >= k1) return;
    double *p = a.dst + (long long)k * a.pitch + i;           // src == dst: the one copy
    double f[NPOP];
    const bool wall_row = k < 3 || k >= a.Lz - 3;             // block-uniform
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int ez = d2q37::pop_ez(l);
        constexpr int lx = d2q37::pop_index(d2q37::pop_ex(l), -ez);
        int ls = NPOP - 1 - l;
        if (wall_row && (k - ez < 0 || k - ez >= a.Lz)) ls = lx;
        f[l] = ld_stream(p + (long long)ls * a.plane);
    });
    wall_rows_adjust<ISO>(a, k, f);
    d2q37::collide_site(f, a.omega, a.gtau, a.dT);
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        st_stream(p + (long long)l * a.plane, f[l]);
    });
}

// Population m of site (i, k) of the STORED state, for either layout of the in-place path (layout_m = false: the
// ordinary layout, also that of the two-copy path).  Used by the diagnostics and by lbm_get_populations.
template <class Fn>
__device__ __forceinline__ void each_stored_site(const double *buf, int Lx, int Lz, int pitch, long long plane,
                                                 bool layout_m, int i, int k, Fn &&fn)
{
    if (!layout_m) {
        const double *p = buf + (long long)k * pitch + i;
        d2q37::static_for<0, NPOP>([&](auto L) { fn(L, p + (long long)decltype(L)::value * plane); });
        return;
    }
    int col[7];
#pragma unroll
    for (int d = -3; d <= 3; ++d) {
        int c = i + d;
        c += (c < 0) ? Lx : 0;
        c -= (c >= Lx) ? Lx : 0;
        col[d + 3] = c;
    }
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int m = decltype(L)::value;
        constexpr int mx = d2q37::pop_ex(m), mz = d2q37::pop_ez(m);
        int q = k + mz;
        if (q >= 0 && q < Lz) {                               // written by the even step of site (i, k) through an ordinary gather
            fn(L, buf + (long long)(NPOP - 1 - m) * plane + (long long)q * pitch + col[mx + 3]);
        } else {                                              // ... through a wall-reflected gather
            q = q < 0 ? -1 - q : 2 * Lz - 1 - q;
            fn(L, buf + (long long)d2q37::pop_index(-mx, mz) * plane + (long long)q * pitch + col[3 - mx]);
        }
    });
}

}  // namespace lbm
