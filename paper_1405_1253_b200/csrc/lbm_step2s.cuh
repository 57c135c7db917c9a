// lbm_step2s.cuh -- two time steps per launch, WARP-SPECIALISED (producer / consumer) version of lbm_step2.cuh.
//
// Same decomposition as step2_kernel (a block owns a strip of TX output columns and marches up ZC rows, the
// intermediate lattice f1 = step(f0) lives in a shared-memory ring, halo columns are recomputed), but
//   * the first step (pass A: global gather -> collide -> ring) and the second step (pass B: ring gather ->
//     collide -> global store) run on DIFFERENT warps, so one side's memory latency overlaps the other side's
//     FP64 arithmetic instead of all warps marching in phase;
//   * pass A's inputs are prefetched a pass ahead into a shared-memory stage by a LOADER warp with TMA tensor box
//     loads (seven per pass) instead of into 74 registers per thread, so 14 warps of 128 registers fit where 8 of
//     253 did;
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

template <int TX_, int R_, int NST_>
struct Step2sShape {
    static constexpr int TX = TX_;                      // output columns per strip (multiple of 32)
    static constexpr int W1 = TX_ + 6;                  // intermediate columns per strip
    static constexpr int CP = TX_ + 8;                  // ring row pitch (doubles)
    static constexpr int R = R_;                        // rows per pass
    static constexpr int NST = NST_;                    // stage buffers (passes of input in flight)
    static constexpr int NA = (R_ * (TX_ + 6) + 31) / 32;   // producer warps (one thread per intermediate site)
    static constexpr int NB = R_ * TX_ / 32;                // consumer warps (one thread per output site)
    static constexpr int NAT = NA * 32, NBT = NB * 32;
    static constexpr int NLT = 32;                          // one loader warp
    static constexpr int SP = TX_ + 16;                     // stage row pitch = source span x0-8 .. x0+TX+7 (doubles)
    static constexpr int THREADS = NAT + NBT + NLT;
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
    static constexpr size_t STAGE_DOUBLES = (size_t)NPOP * R_ * SP;   // per buffer
    static constexpr size_t SMEM = sizeof(double) * (RING_DOUBLES + NST_ * STAGE_DOUBLES);
    static_assert(TX_ % 32 == 0, "a consumer warp covers 32 columns of one row");
    static_assert(R_ >= 2 && NST_ >= 1 && NST_ <= 4, "shape");
    static_assert((R_ * SP * 8) % 128 == 0 && (RING_DOUBLES * 8) % 128 == 0, "TMA box destinations are 128-byte aligned");
    static_assert(LAG < LEAD + 3, "producer may run at most one FULL phase ahead of the consumer's wait");
};
using Step2sWide = Step2sShape<64, 3, 1>;   // 7 producer + 6 consumer + 1 loader warps; ring 127 872 B + stage 71 040 B

// Tensor maps of the source lattice (host-encoded, lbm_api.cu): rank 3 (x: Lx, z: Lz, l: 37), strides
// (pitch, plane) doubles, box (SP, R, n) for n = 3, 5, 7 -- the populations with the same e_z are consecutive in l.
struct Step2sMaps {
    alignas(64) unsigned char m[3][128];                // CUtensorMap x 3 (box depth 3, 5, 7 populations)
};

// ---- loader warp: the gather part of the first step (a2), NST passes ahead of the producers ----
// Seven TMA box loads per pass, one per e_z: box = span of SP source columns x0-8 .. x0+TX+3 (64-byte aligned in
// global memory) x the R source rows (row - e_z) x the 3/5/7 populations with that e_z, written densely as
// stage[l][row of the pass][span column]; the e_x shift is applied when the producers read the stage.  Coordinates
// outside the lattice (periodic seam, walls) are zero-filled by the TMA unit and never read: the producer threads
// whose sources wrap or reflect gather their site from global memory themselves (a1, a3).
// (Measured and dropped, profiles/r1_two_step.md: one 1-D bulk copy per row and population -- the TMA unit issues
// ~1 copy per 63 cycles whatever its size, 7000 cycles per pass; per-thread 8-byte cp.async -- ~20 cycles of
// L1TEX per warp instruction.)
template <class S>
__device__ __noinline__ void step2s_loader(const Step2sMaps *maps, double *stage, unsigned bar_sfull, unsigned bar_sempty,
                                           int lane, int x0, int z0, int NP)   // bars: [NST] each
{
    const unsigned st = (unsigned)__cvta_generic_to_shared(stage);
    const int npass = NP + S::LEAD;
    // lane g < 7 loads the populations with e_z = g - 3: first population, map index by count
    const int ez = lane - 3;
    const int l0 = d2q37::row_first(lane < 7 ? ez : 0);
    const int mi = d2q37::row_half(lane < 7 ? ez : 0) - 1;                       // 3, 5, 7 populations -> map 0, 1, 2
    const unsigned char *map = maps->m[mi];
    int b = 0;                                          // stage buffer of pass j: j mod NST, use number j / NST
    unsigned use = 0;
    for (int j = 0; j < npass; ++j) {
        if (use > 0) mbar_wait(bar_sempty + 8 * b, (use - 1) & 1u);   // producers have read pass j-NST out of buffer b
        const unsigned bar = bar_sfull + 8 * b;
        if (lane == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((unsigned)(S::STAGE_DOUBLES * 8)) : "memory");
        __syncwarp();
        if (lane < 7) {
            const unsigned dst = st + (unsigned)((b * S::STAGE_DOUBLES + (size_t)l0 * S::R * S::SP) * 8);
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                         ::"r"(dst), "l"(map), "r"(x0 - 8), "r"(z0 - 3 + j * S::R - ez), "r"(l0), "r"(bar) : "memory");
        }
        if (++b == S::NST) { b = 0; ++use; }
    }
}

// ---- producer warps: first step of intermediate rows z0-3 .. zend+2, R rows per pass ----
template <class S>
__device__ __noinline__ void step2s_producer(const StepArgs &a, double *ring, const double *stage, unsigned bar_full,
                                                unsigned bar_empty, unsigned bar_sfull, unsigned bar_sempty, int tid,
                                                int x0, int z0, int ncols, int rlast, int NP)
{
    const int ar = tid / S::W1, aj = tid - ar * S::W1;
    const bool a_lane = tid < S::R * S::W1 && aj < ncols + 6;
    const double *sp = stage + ar * S::SP + aj + 5;   // stage [l][row of the pass][span column]; span column = aj + 5 - e_lx
    const int c = x0 - 3 + aj;                          // this thread's column, before the periodic wrap (a1)
    const bool xwrap = c - 3 < 0 || c + 3 >= a.Lx;      // a source column wraps: the site is gathered from global memory
    int ac = c % a.Lx;
    if (ac < 0) ac += a.Lx;

    const int npass = NP + S::LEAD;
    int b = 0;
    unsigned use = 0;
    for (int j = 0; j < npass; ++j) {
        const int row = z0 - 3 + j * S::R + ar;
        const bool v = a_lane && row >= 0 && row < rlast;
        double f[NPOP];
        // sites whose sources wrap (seam strips) or reflect (wall rows, a3) bypass the stage; their loads are issued
        // before the wait so that they overlap it
        const bool gl = v && (xwrap || row < 3 || row >= a.Lz - 3);
        if (gl) gather_any(a, ac, row, f);
        mbar_wait(bar_sfull + 8 * b, use & 1u);
        const double *sb = sp + b * S::STAGE_DOUBLES;
        if (v && !gl) d2q37::static_for<0, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            f[l] = sb[l * S::R * S::SP - d2q37::pop_ex(l)];
        });
        mbar_arrive(bar_sempty + 8 * b);                // values are in registers: the buffer may be refilled
        if (++b == S::NST) { b = 0; ++use; }
        if (v) d2q37::collide_site(f, a.omega, a.gtau, a.dT);
        if (j >= S::LAG) mbar_wait(bar_empty, (unsigned)(j - S::LAG) & 1u);
        if (v) {
            double *rp = ring + aj;
            const int qrow = j * S::R + ar;             // intermediate row index within the chunk, q = row - z0 + 3
            int slot[7];                                // ring slot (in doubles) of row q, per e_z: (q mod depth) CP
#pragma unroll                                          // (computed here, after the collision, to keep it out of its registers)
            for (int e = 0; e < 7; ++e) slot[e] = (qrow % S::depth(e - 3)) * S::CP;
            if (j * S::R >= 6) {
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    rp[S::row_base(l) * S::CP + slot[d2q37::pop_ez(l) + 3]] = f[l];
                });
            } else {
                // warm-up: population l of intermediate row q is first read by output row q + e_lz >= 3 (q = row
                // - z0 + 3).  Rows nobody reads are not stored, so that every store into an occupied slot is one
                // that waits on EMPTY (no producer-producer ordering exists before pass LAG).
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
    }
}

// ---- consumer warps: second step of output rows z0 .. zend-1, R rows per pass ----
template <class S>
__device__ __noinline__ void step2s_consumer(const StepArgs &a, const double *ring, unsigned bar_full,
                                                unsigned bar_empty, int bt, int x0, int z0, int ncols, int zend, int NP)
{
    const int br = bt / S::TX, bj = bt - br * S::TX;
    const bool b_lane = bj < ncols;
    const double *q = ring + bj + 3;

    for (int i = 0; i < NP; ++i) {
        const int k = z0 + i * S::R + br;
        const bool bv = b_lane && k < zend;
        mbar_wait(bar_full, (unsigned)i & 1u);
        double f[NPOP];
        if (bv) {
            if (k < a.Lz - 3) {                         // uniform gather (bottom wall included: ghost rows)
                // ring slot (in doubles) of the SOURCE row k - e_z, per e_z: q = k - e_z - z0 + 3
                int slot[7];
#pragma unroll
                for (int e = 0; e < 7; ++e) slot[e] = ((i * S::R + br + 3 - (e - 3)) % S::depth(e - 3)) * S::CP;
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
    }
}

template <class S>
__global__ void __launch_bounds__(S::THREADS, 1) step2s_kernel(const __grid_constant__ StepArgs a, const __grid_constant__ Step2sMaps maps, const int ZC)
{
    extern __shared__ __align__(128) double smem2s[];    // ring [RING_ROWS][CP] | stage [NST][NPOP][R][SP]
    __shared__ unsigned long long bars[2 + 2 * S::NST];
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * S::TX, z0 = blockIdx.y * ZC;
    const int ncols = min(S::TX, a.Lx - x0);            // output columns of this strip
    const int zend = min(a.Lz, z0 + ZC);                // output rows [z0, zend)
    const int rlast = min(a.Lz, zend + 3);              // intermediate rows [max(0, z0-3), rlast)
    const int NP = (zend - z0 + S::R - 1) / S::R;       // consumer passes
    const unsigned bar_full = (unsigned)__cvta_generic_to_shared(&bars[0]);     // ring rows written (producers -> consumers)
    const unsigned bar_empty = (unsigned)__cvta_generic_to_shared(&bars[1]);    // ring rows read    (consumers -> producers)
    const unsigned bar_sfull = (unsigned)__cvta_generic_to_shared(&bars[2]);    // [NST] stage buffer filled (loaders -> producers)
    const unsigned bar_sempty = bar_sfull + 8 * S::NST;                         // [NST] stage buffer read   (producers -> loaders)
    if (tid == 0) {
        mbar_init(bar_full, S::NAT); mbar_init(bar_empty, S::NBT);
        for (int b = 0; b < S::NST; ++b) { mbar_init(bar_sfull + 8 * b, 1); mbar_init(bar_sempty + 8 * b, S::NAT); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    double *stage = smem2s + S::RING_DOUBLES;
    if (tid < S::NAT)
        step2s_producer<S>(a, smem2s, stage, bar_full, bar_empty, bar_sfull, bar_sempty, tid, x0, z0, ncols, rlast, NP);
    else if (tid < S::NAT + S::NBT)
        step2s_consumer<S>(a, smem2s, bar_full, bar_empty, tid - S::NAT, x0, z0, ncols, zend, NP);
    else
        step2s_loader<S>(&maps, stage, bar_sfull, bar_sempty, tid - S::NAT - S::NBT, x0, z0, NP);
}

}  // namespace lbm
