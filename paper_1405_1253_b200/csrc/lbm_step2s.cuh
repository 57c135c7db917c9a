// lbm_step2s.cuh -- two time steps per launch, WARP-SPECIALISED (producer / consumer) version of lbm_step2.cuh.
//
// Same decomposition as step2_kernel (a block owns a strip of TX output columns and marches up ZC rows, the
// intermediate lattice f1 = step(f0) lives in a shared-memory ring, halo columns are recomputed), but
//   * the first step (pass A: global gather -> collide -> ring) and the second step (pass B: ring gather ->
//     collide -> global store) run on DIFFERENT warps, so one side's memory latency overlaps the other side's
//     FP64 arithmetic instead of all warps marching in phase;
//   * pass A's inputs are prefetched one pass ahead with cp.async into a shared-memory stage (one private
//     37-double slot per producer thread) instead of into 74 registers, so 13 warps fit where 8 did;
//   * the ring keeps, per population, only the rows that can still be read: population l of intermediate row q is
//     read by the output row q + e_lz, so its ring has depth R + 3 + e_lz rows (R .. R + 6) instead of R + 6 for
//     all: 222 instead of 333 row-populations at R = 3, which is what makes room for the stage;
//   * the bottom wall is realised by three GHOST ring rows (rows -3..-1 hold the velocity-reversed copy of rows
//     2..0, written by the producer of those rows; the "ghost row" picture of DESIGN.md reading 9), so pass B's
//     gather is uniform there; at the top wall the mirror rows are still resident and pass B remaps indices.
// Arithmetic is raw_moments / kinetic_from_raw / equilibrium_blend of d2q37.cuh, i.e. exactly collide_site():
// results are bit-identical to two launches of the one-step kernel (tested).
//
// Hand-offs (mbarriers, arrive early / wait late).  Producer pass j writes intermediate rows q in [jR, jR+R)
// (q = row - z0 + 3); consumer pass i reads rows iR .. iR+R+5.
//   FULL : consumer pass i waits for producer passes <= i + LEAD,  LEAD = 1 + 5/R (phase i of the barrier:
//          producers start arriving at pass LEAD, each thread's arrival covers all its earlier passes)
//   EMPTY: producer pass j overwrites slots last read by consumer pass j - LAG, LAG = ceil(7/R), and waits for it.
#pragma once
#include "lbm_step.cuh"
#include "lbm_step2.cuh"   // mbar_* helpers

namespace lbm {

template <int TX_, int R_>
struct Step2sShape {
    static constexpr int TX = TX_;                      // output columns per strip (multiple of 32)
    static constexpr int W1 = TX_ + 6;                  // intermediate columns per strip
    static constexpr int CP = TX_ + 8;                  // ring row pitch (doubles)
    static constexpr int R = R_;                        // rows per pass
    static constexpr int NA = (R_ * (TX_ + 6) + 31) / 32;   // producer warps (one thread per intermediate site)
    static constexpr int NB = R_ * TX_ / 32;                // consumer warps (one thread per output site)
    static constexpr int NAT = NA * 32, NBT = NB * 32;
    static constexpr int THREADS = NAT + NBT;
    static constexpr int MAXREG = 65536 / ((NA + NB + 3) / 4 * 4 * 32) / 8 * 8;   // a block's warps are allocated in fours
    static constexpr int LEAD = 1 + 5 / R_;
    static constexpr int LAG = (7 + R_ - 1) / R_;
    __host__ __device__ static constexpr int depth(int ez) { return R_ + 3 + ez; }
    // first ring row (in units of rows of CP doubles) of population l: populations are stacked, each with its depth
    __host__ __device__ static constexpr int row_base(int l)
    {
        int s = 0;
        for (int m = 0; m < l; ++m) s += depth(d2q37::pop_ez(m));
        return s;
    }
    static constexpr int RING_ROWS = row_base(NPOP);
    static constexpr size_t RING_DOUBLES = (size_t)RING_ROWS * CP;
    static constexpr size_t STAGE_DOUBLES = (size_t)NPOP * NAT;
    static constexpr size_t SMEM = sizeof(double) * (RING_DOUBLES + STAGE_DOUBLES);
    static_assert(TX_ % 32 == 0, "a consumer warp covers 32 columns of one row");
    static_assert(R_ >= 3, "ghost rows use slots 0..2 of every ring");
    static_assert(LAG < LEAD + 3, "producer may run at most one FULL phase ahead of the consumer's wait");
};
using Step2sWide = Step2sShape<64, 3>;   // 7 producer + 6 consumer warps; ring 127 872 B + stage 66 304 B

__device__ __forceinline__ void cp_async8(unsigned dst_smem, const double *src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- producer warps: first step of intermediate rows z0-3 .. zend+2, R rows per pass ----
template <class S>
__device__ __forceinline__ void step2s_producer(const StepArgs &a, double *ring, double *stage, unsigned bar_full,
                                                unsigned bar_empty, int tid, int x0, int z0, int ncols, int rlast, int NP)
{
    const int ar = tid / S::W1, aj = tid - ar * S::W1;
    const bool a_lane = tid < S::R * S::W1 && aj < ncols + 6;
    int ac = (x0 - 3 + aj) % a.Lx;                      // global column, periodic (a1)
    if (ac < 0) ac += a.Lx;
    const unsigned st = (unsigned)__cvta_generic_to_shared(stage + tid);   // slot of population l: st + l NAT 8
    const double *sp = stage + tid;
    int slot[7];                                        // ring slot (in doubles) of this thread's row, per e_z
#pragma unroll
    for (int e = 0; e < 7; ++e) slot[e] = ar * S::CP;

    auto valid = [&](int row) { return a_lane && row >= 0 && row < rlast; };
    auto issue = [&](int row) {                         // gather part of the first step: 37 async copies
        if (valid(row))
            each_source_any(a, ac, row, [&](auto L, const double *p) {
                cp_async8(st + decltype(L)::value * (S::NAT * 8), p);
            });
        cp_async_commit();
    };
    issue(z0 - 3 + ar);
    const int npass = NP + S::LEAD;
    for (int j = 0; j < npass; ++j) {
        const int row = z0 - 3 + j * S::R + ar;
        const bool v = valid(row);
        cp_async_wait_all();
        double f[NPOP];
        d2q37::RawMoments m;
        if (v) {
            d2q37::static_for<0, NPOP>([&](auto L) { f[decltype(L)::value] = sp[decltype(L)::value * S::NAT]; });
            m = d2q37::raw_moments(f);
            asm volatile("" : "+d"(m.m0));              // all 37 stage reads have landed before the slot is reused
        }
        if (j + 1 < npass) issue(row + S::R);
        if (v) {
            const d2q37::Kinetic k = d2q37::kinetic_from_raw(m);
            d2q37::equilibrium_blend<true>(f, f, 1.0 - a.omega, a.omega * k.rho, k.ux, k.uz - a.gtau, k.T + a.dT);
        }
        if (j >= S::LAG) mbar_wait(bar_empty, (unsigned)(j - S::LAG) & 1u);
        if (v) {
            double *rp = ring + aj;
            if (j * S::R >= 6) {
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    rp[S::row_base(l) * S::CP + slot[d2q37::pop_ez(l) + 3]] = f[l];
                });
            } else {
                // warm-up: population l of intermediate row q is first read by output row q + e_lz >= 3 (q = row
                // - z0 + 3).  Rows nobody reads are not stored, so that every store into an occupied slot is one
                // that waits on EMPTY (no producer-producer ordering exists before pass LAG).
                const int qrow = j * S::R + ar;
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    if (qrow + d2q37::pop_ez(l) >= 3) rp[S::row_base(l) * S::CP + slot[d2q37::pop_ez(l) + 3]] = f[l];
                });
            }
            if (z0 == 0 && row < 3) {                   // bottom wall (a3): ghost row -1-row = reversed copy of this row
                // Only the populations that re-enter (e_z > row, read by output row e_z-1-row) are written: the
                // other slots of rows 0..2 of a ring already belong to rows written by the next pass.
                double *gp = rp + (2 - row) * S::CP;
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    if constexpr (d2q37::pop_ez(l) > 0)
                        if (row < d2q37::pop_ez(l)) gp[S::row_base(l) * S::CP] = f[NPOP - 1 - l];
                });
            }
        }
        if (j >= S::LEAD) mbar_arrive(bar_full);        // FULL phase i = "passes <= i + LEAD are in the ring"
#pragma unroll
        for (int e = 0; e < 7; ++e) {
            slot[e] += S::R * S::CP;
            if (slot[e] >= S::depth(e - 3) * S::CP) slot[e] -= S::depth(e - 3) * S::CP;
        }
    }
}

// ---- consumer warps: second step of output rows z0 .. zend-1, R rows per pass ----
template <class S>
__device__ __forceinline__ void step2s_consumer(const StepArgs &a, const double *ring, unsigned bar_full,
                                                unsigned bar_empty, int bt, int x0, int z0, int ncols, int zend, int NP)
{
    const int br = bt / S::TX, bj = bt - br * S::TX;
    const bool b_lane = bj < ncols;
    // ring slot (in doubles) of the SOURCE row k - e_z of this thread's output row k, per e_z: q = k - e_z - z0 + 3
    int slot[7];
#pragma unroll
    for (int e = 0; e < 7; ++e) slot[e] = ((3 + br - (e - 3)) % S::depth(e - 3)) * S::CP;
    const double *q = ring + bj + 3;

    for (int i = 0; i < NP; ++i) {
        const int k = z0 + i * S::R + br;
        const bool bv = b_lane && k < zend;
        mbar_wait(bar_full, (unsigned)i & 1u);
        double f[NPOP];
        if (bv) {
            if (k < a.Lz - 3) {                         // uniform gather (bottom wall included: ghost rows)
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    f[l] = q[S::row_base(l) * S::CP + slot[d2q37::pop_ez(l) + 3] - d2q37::pop_ex(l)];
                });
            } else {                                    // top wall (a3): mirror row, opposite population
                int off[7];
                bool flip[7];
#pragma unroll
                for (int e = -3; e <= 3; ++e) {
                    int ks = k - e;
                    const bool fl = ks >= a.Lz;
                    if (fl) ks = 2 * a.Lz - 1 - ks;
                    off[e + 3] = ((ks - z0 + 3) % (fl ? S::depth(-e) : S::depth(e))) * S::CP;
                    flip[e + 3] = fl;
                }
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    constexpr int ez = d2q37::pop_ez(l);
                    const int base = flip[ez + 3] ? S::row_base(NPOP - 1 - l) * S::CP : S::row_base(l) * S::CP;
                    f[l] = q[base + off[ez + 3] - d2q37::pop_ex(l)];
                });
            }
        }
        mbar_arrive(bar_empty);
        if (bv) {
            d2q37::collide_site(f, a.omega, a.gtau, a.dT);
            scatter_site(a, x0 + bj, k, f);
        }
#pragma unroll
        for (int e = 0; e < 7; ++e) {
            slot[e] += S::R * S::CP;
            if (slot[e] >= S::depth(e - 3) * S::CP) slot[e] -= S::depth(e - 3) * S::CP;
        }
    }
}

template <class S>
__global__ void __maxnreg__(S::MAXREG) step2s_kernel(const StepArgs a, const int ZC)
{
    extern __shared__ double smem2s[];                  // ring [RING_ROWS][CP] | stage [NPOP][NAT]
    __shared__ unsigned long long bars[2];
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * S::TX, z0 = blockIdx.y * ZC;
    const int ncols = min(S::TX, a.Lx - x0);            // output columns of this strip
    const int zend = min(a.Lz, z0 + ZC);                // output rows [z0, zend)
    const int rlast = min(a.Lz, zend + 3);              // intermediate rows [max(0, z0-3), rlast)
    const int NP = (zend - z0 + S::R - 1) / S::R;       // consumer passes
    const unsigned bar_full = (unsigned)__cvta_generic_to_shared(&bars[0]);
    const unsigned bar_empty = (unsigned)__cvta_generic_to_shared(&bars[1]);
    if (tid == 0) { mbar_init(bar_full, S::NAT); mbar_init(bar_empty, S::NBT); }
    __syncthreads();
    if (tid < S::NAT)
        step2s_producer<S>(a, smem2s, smem2s + S::RING_DOUBLES, bar_full, bar_empty, tid, x0, z0, ncols, rlast, NP);
    else
        step2s_consumer<S>(a, smem2s, bar_full, bar_empty, tid - S::NAT, x0, z0, ncols, zend, NP);
}

}  // namespace lbm
