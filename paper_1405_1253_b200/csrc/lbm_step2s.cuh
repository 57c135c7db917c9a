// lbm_step2s.cuh -- TWO time steps per launch (temporal blocking): propagate+bc+collide, twice, with
// the intermediate lattice f1 = step(f0) kept in shared memory, so that HBM sees ~296 B read + 296 B written per
// site per TWO steps instead of per step.  Warp-specialised: loader / producer / consumer warps.
//
// A block owns a strip of w <= TX output columns (w a launch argument) and marches up a chunk of ZC rows of the row
// range [zbase, zend) (the whole lattice, or the own rows of a z-slab whose ghost rows are sources only), R rows per pass.
//   loader (1 warp)   the gather part of the first step: seven TMA tensor box loads per pass (one per e_z) bring the
//                     source rows of the pass into a shared-memory STAGE, NST passes ahead;
//   producers         one thread per site of the R x (w+6) intermediate slab (three halo columns per side are
//                     recomputed, not exchanged): read the 37 populations from the stage with the e_x shift, collide
//                     in registers, store f1 into the RING;
//   consumers         one thread per output site: gather the 37 populations from ring rows k-3..k+3, collide, write
//                     f2 to global memory with aligned full-line stores.
// Ring: population l of intermediate row q is read only by output row q + e_lz, so its ring keeps R + 3 + e_lz rows
// (R .. R+6) instead of R+6 for all -- 37 (R+3) row-populations instead of 37 (R+6), which is what makes room for
// the stage.  Bottom wall (a3): three GHOST ring rows -3..-1 hold the velocity-reversed copy of rows 2..0 (the ghost
// row picture of DESIGN.md reading 9), written by the producers of those rows, so the consumers' gather is uniform
// there; at the top wall the mirror rows are still resident and the consumers remap indices.  Periodic x (a1): every
// row is stored with XH spare columns on either side, of which the nearest XW hold the periodic images (written by
// spare consumer lanes of the seam strips, or refreshed by wrap_columns_kernel after any other writer), so the boxes of the
// seam strips need no special case -- a per-thread global gather for the seam sites cost a factor of two on
// single-wave launches (profiles/r2_two_step.md).  Sites whose first-step sources reflect (wall rows) are gathered
// from global memory by their producer thread; the TMA unit zero-fills those parts of the boxes (rows outside the
// lattice) and they are never read.
// Arithmetic is raw_moments / kinetic_from_raw / equilibrium_blend of d2q37.cuh, i.e. exactly collide_site():
// results are bit-identical to two launches of the one-step kernel (tested).
//
// Hand-offs are mbarriers.  Producer pass j writes intermediate rows q in [jR, jR+R) (q = row - z0 + 3); consumer
// pass i reads rows iR .. iR+R+5.
//   FULL  (producers -> consumers): consumer pass i waits for producer passes <= i + LEAD, LEAD = 1 + 5/R;
//   EMPTY (consumers -> producers): producer pass j overwrites slots last read by consumer pass j - LAG,
//         LAG = ceil(7/R) + SL (SL = optional extra ring depth in passes);
//   STAGE_FULL / STAGE_EMPTY (loader <-> producers), one pair per stage buffer; the TMA loads complete STAGE_FULL.
// A buffer (stage or ring rows) is released only after its values have been CONSUMED by arithmetic, not merely
// loaded: mbarrier.arrive does not wait for shared-memory loads in flight, and a TMA write that the release allows
// was observed to overtake them (profiles/r1_two_step.md).
//
// Measured and dropped on the way (profiles/r1_two_step.md): all warps doing both steps in phase with the first
// step's inputs prefetched into 74 registers (8 warps of 253 registers, 15.0 GLUPS); per-thread 8-byte cp.async into
// the stage (~20 cycles of L1TEX per warp instruction, and L1TEX returns in order, so the issuing warp's next
// local/global load waits for DRAM); one 1-D bulk copy per row and population (the TMA unit issues one copy per
// ~63 cycles whatever its size).
#pragma once
#include "lbm_step.cuh"

namespace lbm {

// shared-memory access through a 32-bit shared-space address plus a compile-time byte offset (one register per base
// instead of a 64-bit generic pointer; the offset is an immediate of the instruction)
template <int OFF>
__device__ __forceinline__ double lds_f64(unsigned addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(addr), "n"(OFF) : "memory");
    return v;
}
template <int OFF>
__device__ __forceinline__ void sts_f64(unsigned addr, double v)
{
    asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(addr), "n"(OFF), "d"(v) : "memory");
}

// split-phase barriers on mbarriers in shared memory
__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}

template <int TX_, int R_, int NST_, int SL_>
struct Step2sShape {
    static constexpr int TX = TX_;                      // output columns per strip, at most (the launch picks w <= TX)
    static constexpr int W1 = TX_ + 6;                  // intermediate columns per strip, at most
    static constexpr int CP = (TX_ + 6 + 1) / 2 * 2;    // ring row pitch (doubles)
    static constexpr int CW = (TX_ + 31) / 32 * 32;     // consumer threads per output row (whole warps)
    static constexpr int R = R_;                        // rows per pass
    static constexpr int NST = NST_;                    // stage buffers (passes of input in flight)
    static constexpr int SL = SL_;                      // ring slack: passes the producers may run ahead of the consumers
    static constexpr int NRB = SL_ + 1;                 // FULL / EMPTY barriers (pass i uses barrier i mod NRB)
    static constexpr int AW = (TX_ + 6 + 31) / 32 * 32;     // producer threads per intermediate row (whole warps)
    static constexpr int NA = R_ * AW / 32;                 // producer warps (one thread per intermediate site)
    static constexpr int NB = R_ * CW / 32;                 // consumer warps (one thread per output site)
    static constexpr int NAT = NA * 32, NBT = NB * 32;
    static constexpr int NLT = 32;                          // one loader warp
    // stage row pitch (doubles): the source span x0-6 .. x0+TX+5 padded so that a box of R rows is a multiple of 128 B
    static constexpr int SP = (TX_ + 12 + (R_ % 2 ? 15 : 7)) / (R_ % 2 ? 16 : 8) * (R_ % 2 ? 16 : 8);
    static constexpr int XPAD = ((SP - TX_ - 12) / 2 + 1) / 2 * 2;   // the box starts at column x0 - 6 - XPAD, kept EVEN: a box
                                                                     // row must start on a 16-byte boundary of global memory
    static constexpr int THREADS = NAT + NBT + NLT;
    static constexpr int LEAD = 1 + 5 / R_;
    static constexpr int LAG = (7 + R_ - 1) / R_ + SL_;
    __host__ __device__ static constexpr int depth(int ez) { return R_ + 3 + ez + SL_ * R_; }
    // first ring row (in units of rows of CP doubles) of population l: populations are stacked, each with its depth
    __host__ __device__ static constexpr int row_base(int l)
    {
        int s = 0;
        for (int m = 0; m < l; ++m) s += depth(d2q37::pop_ez(m));
        return s;
    }
    static constexpr int RING_ROWS = row_base(NPOP);
    static constexpr size_t RING_DOUBLES = ((size_t)RING_ROWS * CP + 15) / 16 * 16;   // stage starts on a 128-byte line
    static constexpr size_t STAGE_DOUBLES = (size_t)NPOP * R_ * SP;   // per buffer
    static constexpr size_t SMEM = sizeof(double) * (RING_DOUBLES + NST_ * STAGE_DOUBLES);
    static_assert((CW & (CW - 1)) == 0, "consumer lanes per row: a power of two");
    static_assert(R_ >= 1 && NST_ >= 1 && NST_ <= 4 && TX_ % 2 == 0 && XPAD <= SP - TX_ - 12, "shape");
    static_assert((R_ * SP * 8) % 128 == 0 && (RING_DOUBLES * 8) % 128 == 0, "TMA box destinations are 128-byte aligned");
};
// Shape <TX, R, NST, SL>, measured at 4096x8192 (profiles/r1_two_step.md):
//   <56,2,3,0> 17.3 GLUPS   4 producer + 4 consumer warps = two collisions per SM sub-partition and pass, three stage
//                           buffers; strips of 56 columns = 14 whole 32-byte sectors per row segment
//   <58,2,3,0> 17.2         same warp balance, but strips start off the sector grid
//   <64,2,2,0> 16.5         5 + 4 compute warps: one sub-partition does three collisions per pass and everybody waits
//   <60,2,3,0> 15.7         (5 producer warps again)
//   <64,2,1,1> 14.2, <64,3,1,0> 14.7   one stage buffer: the producers wait for the TMA round trip
//   <112,1,2,0> 16.8, <120,1,1,0> 14.8  one row per pass, wide strips (5 % halo work instead of 11 %), fewer buffers
// Round 2: the strip width is a launch argument w <= TX (a multiple of 4, chosen by the host so that the strips divide
// Lx without a sliver); 64 producer lanes per intermediate row whatever w, so no warp straddles two rows.
#ifndef S2S_TX   // shape experiments: -DS2S_TX=.. -DS2S_R=.. -DS2S_NST=.. -DS2S_SL=..
#define S2S_TX 56
#define S2S_R 2
#define S2S_NST 3
#define S2S_SL 0
#endif
using Step2sWide = Step2sShape<S2S_TX, S2S_R, S2S_NST, S2S_SL>;

// Tensor maps of the source lattice (host-encoded, lbm_api.cu): rank 3 (x: XH + Lx + XH stored columns, z: stored rows, l: 37), strides
// (pitch, plane) doubles, box (SP, R, n) for n = 3, 5, 7 -- the populations with the same e_z are consecutive in l.
struct Step2sMaps {
    alignas(64) unsigned char m[3][128];                // CUtensorMap x 3 (box depth 3, 5, 7 populations)
};

// ---- loader warp: the gather part of the first step (a2), NST passes ahead of the producers ----
// Seven TMA box loads per pass, one per e_z: box = span of SP source columns from x0-6-XPAD (16-byte aligned in
// global memory) x the R source rows (row - e_z) x the 3/5/7 populations with that e_z, written densely as
// stage[l][row of the pass][span column]; the e_x shift is applied when the producers read the stage.  Coordinates
// outside the lattice (rows beyond the walls) are zero-filled by the TMA unit and never read: the producer threads
// of wall rows gather their site from global memory themselves (a3); the periodic seam is covered by the wrap
// columns (a1).
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
            // x coordinate in the tensor map, whose column 0 is stored column -XH (the wrap columns are part of the tensor)
            asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                         ::"r"(dst), "l"(map), "r"(x0 - 6 - S::XPAD + XH), "r"(z0 - 3 + j * S::R - ez), "r"(l0), "r"(bar) : "memory");
        }
        if (++b == S::NST) { b = 0; ++use; }
    }
}

// ---- producer warps: first step of intermediate rows z0-3 .. zend+2, R rows per pass ----
template <class S, bool ISO>
__device__ __noinline__ void step2s_producer(const StepArgs &a, double *ring, const double *stage, unsigned bar_full,
                                                int tid, int x0, int z0, int ncols, int rlast, int NP)
{
    // the four barrier arrays are consecutive (step2s_kernel): one base register
    const unsigned bar_empty = bar_full + 8 * S::NRB, bar_sfull = bar_empty + 8 * S::NRB, bar_sempty = bar_sfull + 8 * S::NST;
    // AW lanes per intermediate row (whole warps, so that no warp straddles two rows of the stage or of the ring)
    const int ar = tid / S::AW, aj = tid - ar * S::AW;
    const bool a_lane = aj < ncols + 6;
    // stage [l][row of the pass][span column]; span column = aj + 3 + XPAD - e_lx
    const unsigned sp = (unsigned)__cvta_generic_to_shared(stage) + (unsigned)((ar * S::SP + aj + 3 + S::XPAD) * 8);
    const unsigned rp0 = (unsigned)__cvta_generic_to_shared(ring) + (unsigned)(aj * 8);   // ring column of this thread
    const int c = x0 - 3 + aj;                          // this thread's column, before the periodic wrap (a1)
    int ac = c % a.Lx;
    if (ac < 0) ac += a.Lx;
    const int Lz = a.Lz;                                // kernel arguments into registers once (see the consumer)
    const double omega = a.omega, gtau = a.gtau, dT = a.dT;

    const int npass = NP + S::LEAD;
    for (int j = 0; j < npass; ++j) {
        const int b = j % S::NST;                       // stage buffer of this pass, and how often it was used before
        const unsigned use = (unsigned)(j / S::NST);
        const int row = z0 - 3 + j * S::R + ar;
        const bool v = a_lane && row >= 0 && row < rlast;
        double f[NPOP];
        // sites whose sources reflect (wall rows, a3) bypass the stage; their loads are issued before the wait so that
        // they overlap it.  (Periodic x, a1, needs no such path: the boxes of the seam strips read the wrap columns.)
        const bool gl = v && (row < 3 || row >= Lz - 3);
        if (gl) each_source_site<true>(a, ac, row, [&](auto L, const double *p, bool) { f[decltype(L)::value] = ld_stream(p); });
        mbar_wait(bar_sfull + 8 * b, use & 1u);
        const unsigned sb = sp + (unsigned)(b * (S::STAGE_DOUBLES * 8));
        if (v && !gl) d2q37::static_for<0, NPOP>([&](auto L) {
            constexpr int l = decltype(L)::value;
            f[l] = lds_f64<(l * S::R * S::SP - d2q37::pop_ex(l)) * 8>(sb);
        });
        // The buffer is released only after the moments have CONSUMED the 37 values (not merely after the loads were
        // issued): mbarrier.arrive does not wait for shared-memory loads in flight, and the TMA write that the
        // release allows was seen to overtake them (L2-resident source rows, loads held back behind the global
        // gathers of the same warp) -- a one-in-10^5-blocks error, profiles/r1_two_step.md.
        d2q37::RawMoments m;
        if (v) {
            if (gl) wall_rows_adjust<ISO>(a, row, f);       // wall_kind 1: rows next to an isothermal wall (a3)
            m = d2q37::raw_moments(f);
            // keeps the arrive below the sums in the instruction stream: a DADD cannot issue before its operands
            // have returned from shared memory, and a warp issues in order (tests/test_library_cpu.py checks the
            // order in the SASS; making the barrier address depend on the sums instead costs 3.5 %)
            asm volatile("" : "+d"(m.m0), "+d"(m.jx), "+d"(m.jz), "+d"(m.m2));
        }
        // generic-proxy reads of the stage -> async-proxy (TMA) rewrite of the same buffer: the arrive alone does not
        // order across proxies, so the reads are fenced into the async proxy before the release (the pattern for
        // generic reads of TMA-filled shared memory; the consume-before-release order above stays as a second guard)
        fence_proxy_async_smem();
        mbar_arrive(bar_sempty + 8 * b);
        if (v) {
            const d2q37::Kinetic kin = d2q37::kinetic_from_raw(m);
            d2q37::equilibrium_blend<true, true>(f, f, 1.0 - omega, omega * kin.rho, kin.ux, kin.uz - gtau, kin.T + dT);
        }
        if (j >= S::LAG) mbar_wait(bar_empty + 8 * ((j - S::LAG) % S::NRB), (unsigned)((j - S::LAG) / S::NRB) & 1u);
        if (v) {
            const int qrow = j * S::R + ar;             // intermediate row index within the chunk, q = row - z0 + 3
            int slot[7];                                // ring slot (in doubles) of row q, per e_z: (q mod depth) CP
#pragma unroll                                          // (computed here, after the collision, to keep it out of its registers)
            for (int e = 0; e < 7; ++e) slot[e] = (qrow % S::depth(e - 3)) * (S::CP * 8);   // bytes
            if (j * S::R >= 6) {
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    sts_f64<S::row_base(l) * S::CP * 8>(rp0 + slot[d2q37::pop_ez(l) + 3], f[l]);
                });
            } else {
                // warm-up: population l of intermediate row q is first read by output row q + e_lz >= 3 (q = row
                // - z0 + 3).  Rows nobody reads are not stored, so that every store into an occupied slot is one
                // that waits on EMPTY (no producer-producer ordering exists before pass LAG).
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    if (qrow + d2q37::pop_ez(l) >= 3) sts_f64<S::row_base(l) * S::CP * 8>(rp0 + slot[d2q37::pop_ez(l) + 3], f[l]);
                });
            }
            if (z0 == 0 && row < 3) {                   // bottom wall (a3): ghost row -1-row = reversed copy of this row
                // Only the populations that re-enter (e_z > row, read by output row e_z-1-row) are written: the
                // other slots of rows 0..2 of a ring already belong to rows written by the next pass.
                const unsigned gp = rp0 + (unsigned)((2 - row) * (S::CP * 8));
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    if constexpr (d2q37::pop_ez(l) > 0)
                        if (row < d2q37::pop_ez(l)) sts_f64<S::row_base(l) * S::CP * 8>(gp, f[NPOP - 1 - l]);
                });
            }
        }
        if (j >= S::LEAD) mbar_arrive(bar_full + 8 * ((j - S::LEAD) % S::NRB));   // FULL of consumer pass i = j - LEAD: "passes <= i + LEAD are in the ring"
    }
}

// ---- consumer warps: second step of output rows z0 .. zend-1, R rows per pass ----
template <class S, bool ISO>
__device__ __noinline__ void step2s_consumer(const StepArgs &a, const double *ring, unsigned bar_full,
                                                unsigned bar_empty, int bt, int x0, int z0, int ncols, int zend)
{
    const int br = bt / S::CW, bj = bt - br * S::CW;
    // Periodic x (a1): the next launch's boxes read the wrap columns of THIS launch's destination copy (columns
    // 0..XW-1 repeat after column Lx-1, columns Lx-XW..Lx-1 before column 0).  The CW - ncols spare lanes of a row
    // write them: in the two seam strips a spare lane computes the same site as the lane that owns the seam column
    // (same ring values, same arithmetic, same result) and stores it at the image position.  Only the starting values
    // of two per-thread pointers differ, so the loop is untouched -- it has no register to spare: consumers that
    // stored the image as a second store spilled and lost 10-25 %, a loader warp copying the columns (per-lane
    // loads / stores, or TMA boxes) slowed the seam strips by 1.3-1.8x (profiles/r2_two_step.md).
    int cj = bj, img = 0;                               // strip column this lane computes; offset of its store
    bool b_lane = bj < ncols;
    if (a.wrap_store) {
        const bool lo = x0 == 0, hi = x0 + ncols == a.Lx;          // first / last strip (or both)
        const int t = bj - ncols, th = t - (lo ? XW : 0);            // spare lane index; ... after the low seam's
        if (lo && t >= 0 && t < XW) { cj = t; img = a.Lx; b_lane = true; }
        else if (hi && th >= 0 && th < XW) { cj = ncols - XW + th; img = -a.Lx; b_lane = true; }
    }
    const unsigned q = (unsigned)__cvta_generic_to_shared(ring) + (unsigned)((cj + 3) * 8);   // ring column of this thread
    // kernel arguments into registers once: `a` is reached through a pointer here (non-inlined role), and every
    // global store would otherwise force its fields to be re-loaded.  Rows are counted relative to the chunk
    // (kq = k - z0) to keep the loop state small: the collision needs nearly all 168 registers.
    const int zr = zend - z0;                           // output rows of the chunk
    const int lt = a.Lz - z0;                           // kq of the first row above the top wall
    const double omega = a.omega, gtau = a.gtau, dT = a.dT;
    const long long plane = a.plane;
    double *p = a.dst + (long long)(z0 + br) * a.pitch + x0 + cj + img;    // this thread's site of the pass, population 0
    const long long pass_stride = (long long)S::R * a.pitch;

    for (int i = 0; i * S::R < zr; ++i, p += pass_stride) {
        const int kq = i * S::R + br;
        const bool bv = b_lane && kq < zr;
        mbar_wait(bar_full + 8 * (i % S::NRB), (unsigned)(i / S::NRB) & 1u);
        double f[NPOP];
        if (bv) {
            if (kq < lt - 3) {                          // uniform gather (bottom wall included: ghost rows)
                // ring slot (in doubles) of the SOURCE row k - e_z, per e_z: q = k - e_z - z0 + 3
                int slot[7];
#pragma unroll
                for (int e = 0; e < 7; ++e) slot[e] = ((kq + 3 - (e - 3)) % S::depth(e - 3)) * (S::CP * 8);   // bytes
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    f[l] = lds_f64<(S::row_base(l) * S::CP - d2q37::pop_ex(l)) * 8>(q + slot[d2q37::pop_ez(l) + 3]);
                });
            } else {                                    // top wall (a3): mirror row, opposite population
                int off[7];
                bool flip[7];
#pragma unroll
                for (int e = -3; e <= 3; ++e) {
                    int ks = kq - e;                    // source row relative to the chunk
                    const bool fl = ks >= lt;
                    if (fl) ks = 2 * lt - 1 - ks;
                    off[e + 3] = ((ks + 3) % (fl ? S::depth(-e) : S::depth(e))) * (S::CP * 8);
                    flip[e + 3] = fl;
                }
                d2q37::static_for<0, NPOP>([&](auto L) {
                    constexpr int l = decltype(L)::value;
                    constexpr int ez = d2q37::pop_ez(l);
                    const int base = flip[ez + 3] ? S::row_base(NPOP - 1 - l) * S::CP * 8 : S::row_base(l) * S::CP * 8;
                    f[l] = lds_f64<-d2q37::pop_ex(l) * 8>(q + base + off[ez + 3]);
                });
            }
        }
        d2q37::RawMoments m;                            // release the ring rows after the values were consumed (see the producer)
        if (bv) {
            if constexpr (ISO)
                if (kq + z0 < 3 || kq >= lt - 3) wall_rows_adjust<ISO>(a, kq + z0, f);
            m = d2q37::raw_moments(f);
            asm volatile("" : "+d"(m.m0), "+d"(m.jx), "+d"(m.jz), "+d"(m.m2));
        }
        mbar_arrive(bar_empty + 8 * (i % S::NRB));
        if (bv) {
            const d2q37::Kinetic kin = d2q37::kinetic_from_raw(m);
            d2q37::equilibrium_blend<true, true>(f, f, 1.0 - omega, omega * kin.rho, kin.ux, kin.uz - gtau, kin.T + dT);
            d2q37::static_for<0, NPOP>([&](auto L) {     // 37 aligned stores, full 128-byte lines per warp
                constexpr int l = decltype(L)::value;
                st_stream(p + l * plane, f[l]);
            });
        }
    }
}

template <class S, bool ISO>
__global__ void __launch_bounds__(S::THREADS, 1) step2s_kernel(const __grid_constant__ StepArgs a, const __grid_constant__ Step2sMaps maps, const int ZC)
{
    extern __shared__ __align__(128) double smem2s[];    // ring [RING_ROWS][CP] | stage [NST][NPOP][R][SP]
    __shared__ unsigned long long bars[2 * S::NRB + 2 * S::NST];
    const int tid = threadIdx.x;
    const int w = a.w;                                   // strips of w <= TX columns (w even: TMA boxes start on 16 bytes)
    // a z-slab updates its own rows; its ghost rows are sources only.  ztrim (wall_kind 1): the chunk on an isothermal
    // wall is that many rows shorter, which is what its wall adjustments cost (lbm_api.cu make_plan)
    int by = blockIdx.y, zb = a.zbase, ze = a.zend;
    if (by >= a.zsplit) { by -= a.zsplit; zb = a.zbase2; ze = a.zend2; }   // second row range of the launch (slab edges)
    const int x0 = blockIdx.x * w, z0 = zb + by * ZC - (by ? a.ztrim : 0);
    const int ncols = min(w, a.Lx - x0);                // output columns of this strip
    const int zend = min(ze, zb + (by + 1) * ZC - a.ztrim);   // output rows [z0, zend)
    const int rlast = min(a.Lz, zend + 3);              // intermediate rows [max(0, z0-3), rlast)
    const int NP = (zend - z0 + S::R - 1) / S::R;       // consumer passes
    const unsigned bar_full = (unsigned)__cvta_generic_to_shared(&bars[0]);     // [NRB] ring rows written (producers -> consumers)
    const unsigned bar_empty = bar_full + 8 * S::NRB;                           // [NRB] ring rows read    (consumers -> producers)
    const unsigned bar_sfull = bar_empty + 8 * S::NRB;                          // [NST] stage buffer filled (loaders -> producers)
    const unsigned bar_sempty = bar_sfull + 8 * S::NST;                         // [NST] stage buffer read   (producers -> loaders)
    if (tid == 0) {
        for (int b = 0; b < S::NRB; ++b) { mbar_init(bar_full + 8 * b, S::NAT); mbar_init(bar_empty + 8 * b, S::NBT); }
        for (int b = 0; b < S::NST; ++b) { mbar_init(bar_sfull + 8 * b, 1); mbar_init(bar_sempty + 8 * b, S::NAT); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    double *stage = smem2s + S::RING_DOUBLES;
    // wall_kind 1 (ISO): only the chunks that hold one of the three rows next to an isothermal wall -- as intermediate
    // rows [z0-3, zend+3) or as output rows -- run the roles with the wall adjustment; every other block of the launch
    // runs the plain roles (separate non-inlined functions, so the larger code and the spills of the wall roles cost
    // the bulk of the lattice nothing: "computational impact is fully negligible").
    bool wall_chunk = false;
    if constexpr (ISO) wall_chunk = (a.iso_lo && z0 < 6) || (a.iso_hi && zend + 6 > a.Lz);
    if (tid < S::NAT) {
        if (wall_chunk) step2s_producer<S, true>(a, smem2s, stage, bar_full, tid, x0, z0, ncols, rlast, NP);
        else step2s_producer<S, false>(a, smem2s, stage, bar_full, tid, x0, z0, ncols, rlast, NP);
    } else if (tid < S::NAT + S::NBT) {
        if (wall_chunk) step2s_consumer<S, true>(a, smem2s, bar_full, bar_empty, tid - S::NAT, x0, z0, ncols, zend);
        else step2s_consumer<S, false>(a, smem2s, bar_full, bar_empty, tid - S::NAT, x0, z0, ncols, zend);
    } else {
        step2s_loader<S>(&maps, stage, bar_sfull, bar_sempty, tid - S::NAT - S::NBT, x0, z0, NP);
    }
}

}  // namespace lbm
