// lbm_step2.cuh -- TWO time steps per launch (temporal blocking): propagate+bc+collide, twice, with the
// intermediate lattice kept in shared memory, so that HBM sees ~296 B read + 296 B written per site per TWO
// steps instead of per step.
//
// A block owns a strip of TX output columns and marches up a chunk of ZC rows.  It keeps a ring of RING = R + 6
// rows of the INTERMEDIATE state f1 = step(f0) for the TX + 6 columns x0-3 .. x0+TX+2 (the three halo columns
// per side are recomputed redundantly instead of exchanged: +9 % first-step work at TX = 64, and their source
// sectors are shared with the neighbouring strip through L2).  Per iteration of R rows:
//   A  (first step, PAPER.md:114 propagate+bc+collide): every thread owns one site of R new f1 rows, gathers its
//      37 populations from the global source lattice (periodic wrap + wall remap exactly as in lbm_step.cuh),
//      collides in registers and stores the 37 results into the ring;
//   B  (second step): every thread owns one site of R output rows, gathers its 37 populations from the ring
//      (rows k-3..k+3, wall remap, no wrap needed: ring columns are strip-local), collides, and writes f2 to the
//      global destination lattice with aligned stores.
// The global loads of the NEXT A pass are issued before B starts and are consumed after it, so HBM latency is
// hidden behind B's arithmetic.  The two hand-offs per iteration are split mbarriers (arrive early, wait late):
// FULL = "this pass's rows are in the ring" (arrive after the stores, wait before B's gather), EMPTY = "B has read
// the ring" (arrive right after B's gather, wait only before the next pass's stores, i.e. after two collisions),
// so warps rendezvous once per iteration.  Arithmetic is the same collide_site() as the one-step kernel, so two
// fused steps are bit-identical to two single steps (tested).
#pragma once
#include "lbm_step.cuh"

namespace lbm {

// Compile-time shape of the two-step kernel.  TX output columns per strip, R rows per iteration.
template <int TX_, int R_, int THREADS_, int BLOCKS_>
struct Step2Shape {
    static constexpr int TX = TX_;            // output columns per strip (multiple of 32)
    static constexpr int W1 = TX_ + 6;        // intermediate columns per strip
    static constexpr int CP = TX_ + 8;        // shared-memory row pitch (doubles)
    static constexpr int R = R_;              // rows per iteration
    static constexpr int RING = R_ + 6;       // intermediate rows resident
    static constexpr int THREADS = THREADS_;  // >= R * W1
    static constexpr int BLOCKS = BLOCKS_;    // resident blocks per SM (shared memory and registers permitting)
    static constexpr size_t SMEM = sizeof(double) * RING * NPOP * CP;
    static_assert(THREADS_ >= R_ * (TX_ + 6), "one thread per intermediate site of a pass");
    static_assert(R_ >= 3 && R_ <= 6, "warm-up is written for 3..6 rows per pass");
};
// 64 columns x 3 rows, 256 threads (up to 255 registers: prefetched inputs + working set), 1 block per SM
using Step2Wide = Step2Shape<64, 3, 256, 1>;      // ring 9 x 37 x 72 doubles = 191 808 B
// (Measured and dropped, profiles/r1_two_step.md: 32 columns x 3 rows with 2 blocks/SM, and 5 or 4 rows per pass
// with 12 or 10 warps at 168 registers, where the second step re-reads the ring instead of holding f.)

// split-phase block barrier on an mbarrier in shared memory (all threads of the block arrive on every phase)
__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}

// Second-step gather of output site (strip column bj, row k) from the ring of intermediate rows.
template <class S, bool WALL>
__device__ __forceinline__ void gather_ring(const double *ring, int Lz, int z0, int bj, int k, double (&f)[NPOP])
{
    int rowoff[7];
    bool flip[7];
#pragma unroll
    for (int d = -3; d <= 3; ++d) {
        int ks = k - d;
        bool fl = false;
        if (WALL) {
            if (ks < 0) { ks = -1 - ks; fl = true; }
            else if (ks >= Lz) { ks = 2 * Lz - 1 - ks; fl = true; }
        }
        rowoff[d + 3] = ((ks - z0 + 3) % S::RING) * (NPOP * S::CP);
        flip[d + 3] = fl;
    }
    const double *q = ring + bj + 3;
    d2q37::static_for<0, NPOP>([&](auto L) {
        constexpr int l = decltype(L)::value;
        constexpr int ex = d2q37::pop_ex(l), ez = d2q37::pop_ez(l);
        int ls = l;
        if (WALL) ls = flip[ez + 3] ? (NPOP - 1 - l) : l;
        f[l] = q[rowoff[ez + 3] + ls * S::CP - ex];
    });
}

template <class S>
__global__ void __launch_bounds__(S::THREADS, S::BLOCKS) step2_kernel(const StepArgs a, const int ZC)
{
    extern __shared__ double ring[];      // [RING][NPOP][CP]
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * S::TX, z0 = blockIdx.y * ZC;
    const int ncols = min(S::TX, a.Lx - x0);          // output columns of this strip
    const int zend = min(a.Lz, z0 + ZC);               // output rows [z0, zend)
    const int rlast = min(a.Lz, zend + 3);             // intermediate rows [max(0, z0-3), rlast)

    // A mapping: thread -> (row within pass, strip-local column), global column wrapped once
    const int ar = tid / S::W1, aj = tid - ar * S::W1;
    const bool a_lane = tid < S::R * S::W1 && aj < ncols + 6;
    int ac = (x0 - 3 + aj) % a.Lx;
    if (ac < 0) ac += a.Lx;
    // B mapping
    const int br = tid / S::TX, bj = tid - br * S::TX;
    const bool b_lane = tid < S::R * S::TX && bj < ncols;

    double g[NPOP];                                    // inputs of the pending A pass

    auto a_valid = [&](int row0, int nrows) {
        const int r = row0 + ar;
        return a_lane && ar < nrows && r >= 0 && r < rlast;
    };
    auto a_issue = [&](int row0, int nrows) {          // first step, gather part: loads stay in flight
        if (a_valid(row0, nrows)) gather_any(a, ac, row0 + ar, g);
    };
    auto a_store = [&](int row0) {                     // first-step results into the ring
        double *p = ring + ((row0 + ar - z0 + 3) % S::RING) * (NPOP * S::CP) + aj;
        d2q37::static_for<0, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            p[l * S::CP] = g[l];
        });
    };

    __shared__ unsigned long long bars[2];
    const unsigned bar_full = (unsigned)__cvta_generic_to_shared(&bars[0]);
    const unsigned bar_empty = (unsigned)__cvta_generic_to_shared(&bars[1]);
    if (tid == 0) { mbar_init(bar_full, S::THREADS); mbar_init(bar_empty, S::THREADS); }
    __syncthreads();

    // warm-up: intermediate rows z0-3 .. z0+2 (one full pass and one of 6 - R rows)
    a_issue(z0 - 3, S::R);
    if (a_valid(z0 - 3, S::R)) { d2q37::collide_site(g, a.omega, a.gtau, a.dT); a_store(z0 - 3); }
    if (S::R < 6) {
        a_issue(z0 - 3 + S::R, 6 - S::R);
        if (a_valid(z0 - 3 + S::R, 6 - S::R)) { d2q37::collide_site(g, a.omega, a.gtau, a.dT); a_store(z0 - 3 + S::R); }
    }
    a_issue(z0 + 3, S::R);

    unsigned phase = 0;
    for (int k0 = z0; k0 < zend; k0 += S::R, phase ^= 1) {
        // first step of rows k0+3 .. k0+2+R: collide, then store once B of the previous iteration has read the ring
        const bool av = a_valid(k0 + 3, S::R);
        if (av) d2q37::collide_site(g, a.omega, a.gtau, a.dT);
        if (k0 > z0) mbar_wait(bar_empty, phase ^ 1);
        if (av) a_store(k0 + 3);
        mbar_arrive(bar_full);
        if (k0 + S::R < zend) a_issue(k0 + S::R + 3, S::R);   // prefetch the next pass behind B
        mbar_wait(bar_full, phase);

        // second step of rows k0 .. k0+R-1
        const int k = k0 + br;
        const bool bv = b_lane && k < zend;
        double f[NPOP];
        if (bv) {
            if (k >= 3 && k < a.Lz - 3) gather_ring<S, false>(ring, a.Lz, z0, bj, k, f);
            else gather_ring<S, true>(ring, a.Lz, z0, bj, k, f);
        }
        mbar_arrive(bar_empty);
        if (bv) {
            d2q37::collide_site(f, a.omega, a.gtau, a.dT);
            scatter_site(a, x0 + bj, k, f);
        }
    }
}

}  // namespace lbm
