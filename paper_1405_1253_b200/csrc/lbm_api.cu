// lbm_api.cu -- the C ABI declared in include/lbm.h: handle, argument checks, kernel launches.
// Every arithmetic step of the path runs in the kernels of lbm_step.cuh / lbm_step2s.cuh / lbm_aux.cuh; this file
// only validates, draws the interface perturbation (host, O(Lx)), plans launches, launches and copies.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lbm.h"
#include "lbm_aux.cuh"
#include "lbm_step.cuh"
#include "lbm_step2s.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(expr)                                                                                  \
    do {                                                                                                \
        cudaError_t e_ = (expr);                                                                        \
        if (e_ != cudaSuccess) return fail(LBM_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_));      \
    } while (0)

constexpr int ROW_ALIGN = 16;     // doubles: rows start on 128-byte lines
constexpr int PLANE_PAD = 272;    // doubles (17 x 128 B): keeps the 37 plane bases off a power-of-two stride
constexpr int GHOST = 3;          // ghost rows one step reads beyond an open side of a z-slab (max |e_z|)
constexpr int GHOST_STORED = 6;   // ghost rows stored per open side: two fused steps read 6

// row = [XH spare | Lx sites | XH spare], padded to 128 bytes
int pitch_of(int Lx) { return (Lx + 2 * lbm::XH + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN; }
long long plane_of(int Lx, int rows) { return (long long)pitch_of(Lx) * rows + PLANE_PAD; }

// SplitMix64 (reading 12); U = (x >> 11) 2^-53
struct SplitMix {
    uint64_t s;
    double next()
    {
        uint64_t z = (s += 0x9E3779B97F4A7C15ull);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        z ^= z >> 31;
        return (double)(z >> 11) * 0x1.0p-53;
    }
};

void draw_interface(SplitMix &rng, const lbm_rt_init &ic, int Lx, std::vector<double> &h)
{
    const double two_pi = 6.283185307179586476925286766559;
    h.assign(Lx, 0.0);
    if (ic.pert_kind == 1) {
        for (int m = 1; m <= ic.n_modes; ++m) {
            double amp = ic.amp_lo;
            if (ic.amp_hi != ic.amp_lo) amp = ic.amp_lo + (ic.amp_hi - ic.amp_lo) * rng.next();
            const double phase = two_pi * rng.next();
            for (int i = 0; i < Lx; ++i) h[i] += amp * std::cos(two_pi * (double)m * (double)i / (double)Lx + phase);
        }
    } else if (ic.pert_kind == 2) {
        for (int i = 0; i < Lx; ++i) h[i] = ic.amp_hi * (2.0 * rng.next() - 1.0);
    }
}

// Tensor maps for the TMA loads of the warp-specialised two-step kernel (lbm_step2s.cuh): the lattice copy as a
// rank-3 tensor (x: XH + Lx + XH stored columns, z: Lz, l: 37) with strides (pitch, plane), box (SP, R, n) for
// n = 3, 5, 7.  `ubuf` is the start of the allocation (stored column -XH of row 0).
// cuTensorMapEncodeTiled is fetched through the runtime (no link-time dependency on libcuda).
bool encode_step2s_maps(const double *ubuf, int Lx, int Lz, int pitch, long long plane, lbm::Step2sMaps &out)
{
    using S = lbm::Step2sWide;
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                 const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn) {
            cudaGetLastError();
            return false;
        }
        encode = (EncodeFn)fn;
    }
    static_assert(sizeof(CUtensorMap) == 128, "Step2sMaps holds three 128-byte tensor maps");
    for (int i = 0; i < 3; ++i) {
        const cuuint64_t dims[3] = {(cuuint64_t)(Lx + 2 * lbm::XH), (cuuint64_t)Lz, (cuuint64_t)LBM_NPOP};
        const cuuint64_t strides[2] = {(cuuint64_t)pitch * 8, (cuuint64_t)plane * 8};
        const cuuint32_t box[3] = {(cuuint32_t)S::SP, (cuuint32_t)S::R, (cuuint32_t)(3 + 2 * i)};
        const cuuint32_t estr[3] = {1, 1, 1};
        if (encode((CUtensorMap *)out.m[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)ubuf, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

}  // namespace

// launch plan of lbm_step (make_plan)
struct lbm_plan {
    bool valid, fused;
    int w, strips, ZC, chunks;
    int trim;       // wall_kind 1: rows the chunks next to an isothermal wall are shorter by (chunk boundaries shift down by it)
};

struct lbm_handle {
    int dev;               // CUDA device the handle was created on (every call must run with it current)
    int Lx, Lz, pitch;     // Lz = STORED rows (a z-slab: its own rows plus ghost rows)
    long long plane;
    double tau, g;
    int wall_kind;
    double T_wall_lo, T_wall_hi;
    double *ubuf[2];       // the caller's buffers
    double *buf[2];        // site (0,0) of population 0 in each copy (ubuf + XH); buf[1] = null: in-place, one copy
    bool inplace, layout_m;   // in-place path: layout_m after an odd number of steps (lbm_step.cuh)
    bool wrap_ok[2];       // the wrap columns of copy i hold the periodic images of its current contents
    bool cap_seen;         // refresh_wrap_columns: the last stream capture that recorded a refresh
    unsigned long long cap_id;
    // z-slab (lbm_create_slab): height of the whole lattice, first own global row, own rows, ghost rows below / above
    bool slab;
    int Lz_glob, z0, nz, glo, ghi;
    int slab_phase;        // 0: ready for lbm_slab_step(INTERIOR), 1: interior launched, edges pending
    int cur;               // index of the current lattice
    long long steps, launches;
    int variant;
    int zchunk;            // rows per block of the two-step kernel (0 = automatic)
    int sm_count;
    lbm_plan plan;         // cached; invalidated by lbm_set_variant / lbm_set_zchunk
    lbm_plan plan_interior;   // lbm_slab_step2_part: the plan over the interior rows of a slab
    bool tma_ok;           // tensor maps of both lattice copies encoded (two-step kernel)
    lbm::Step2sMaps maps[2];
    double *scratch;       // device: row diagnostics [8][nz] | results[8] | h_lo[Lx] | h_hi[Lx]
    double *stage[4];      // device staging fields for lbm_run_host (lazy)
    int persist_tb, persist_blocks;   // persistent small-lattice kernel: block size and grid (0 = not applicable)
    unsigned *d_counter;   // device: grid-barrier counter of the persistent kernel
    double *plane_stage;   // device staging of one dense population plane for the _host copies of in-place handles (lazy)
    lbm::Layout layout() const { return lbm::Layout{Lx, Lz, pitch, plane, glo, nz, layout_m}; }
    double *d_rows() const { return scratch; }
    double *d_result() const { return scratch + 8LL * nz; }
    double *d_hlo() const { return scratch + 8LL * nz + 8; }
    double *d_hhi() const { return scratch + 8LL * nz + 8 + Lx; }
    bool wall_lo() const { return !slab || z0 == 0; }
    bool wall_hi() const { return !slab || z0 + nz == Lz_glob; }
};

namespace {

int check_handle(const lbm_t *h, const char *fn)
{
    if (!h) return fail(LBM_ERR_INVALID, "%s: null handle", fn);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(LBM_ERR_NODEVICE, "%s: no CUDA device", fn); }
    if (dev != h->dev)
        return fail(LBM_ERR_INVALID, "%s: the handle lives on device %d but device %d is current", fn, h->dev, dev);
    return LBM_OK;
}
#define NEED(h) do { int rc_ = check_handle((h), __func__); if (rc_) return rc_; } while (0)
#define NEED_HOST(h) do { if (!(h)) return fail(LBM_ERR_INVALID, "%s: null handle", __func__); } while (0)
#define LAUNCHED(h) do { CUDA_TRY(cudaGetLastError()); (h)->launches++; } while (0)

dim3 own_grid(const lbm_t *h, int tx) { return dim3((h->Lx + tx - 1) / tx, h->nz, 1); }

lbm::StepArgs step_args(const lbm_t *h)
{
    lbm::StepArgs a;
    a.Lx = h->Lx; a.Lz = h->Lz; a.pitch = h->pitch; a.plane = h->plane;
    a.omega = 1.0 / h->tau;
    a.gtau = h->g * h->tau;
    a.dT = 0.5 * h->tau * (1.0 - h->tau) * h->g * h->g;
    // wall_kind 1 (reading 19): kinetic wall state u_w = (0, g/2), T_w = T_wall - g^2/8 (PAPER.md:94 backwards)
    a.iso_lo = h->wall_kind == 1 && h->wall_lo();
    a.iso_hi = h->wall_kind == 1 && h->wall_hi();
    a.uwz = 0.5 * h->g;
    a.Tw_lo = h->T_wall_lo - 0.125 * h->g * h->g;
    a.Tw_hi = h->T_wall_hi - 0.125 * h->g * h->g;
    a.wrap_store = 0;
    a.w = 0;
    a.ztrim = 0;
    a.zsplit = INT_MAX; a.zbase2 = a.zend2 = 0;
    a.zbase = h->glo; a.zend = h->glo + h->nz;
    lbm::fill_offsets(a);
    return a;
}

// Launch plan of lbm_step for this lattice.  The two-step kernel runs strips of w <= TX columns in chunks of ZC rows,
// one block per SM at a time, every block (ZC + 6)/R passes of about the same duration: the plan minimises
//   (waves + 0.15) x (ZC + 6 + fill) x (1 + ZC/16000),  waves = ceil(strips x chunks / SMs),  fill = 10 rows' worth
// over the strip count and ZC (whole waves: no tail; few chunks: little warm-up -- a chunk recomputes the 6
// intermediate rows below it and waits for its first boxes; + 0.15: the blocks of a wave do not finish together --
// wall chunks gather three rows from global memory -- so a launch waits for its slowest block), and takes the
// one-step kernel where that is predicted to be faster (small lattices).  Constants fitted to the chunk-size runs of
// profiles/r2_two_step.md section 3.
lbm_plan compute_plan(const lbm_t *h, int rows)
{
    using S2 = lbm::Step2sWide;
    lbm_plan p = lbm_plan{};
    const int Lx = h->Lx, Lz = rows, sms = h->sm_count > 0 ? h->sm_count : 148;
    const bool iso_lo = h->wall_kind == 1 && h->wall_lo(), iso_hi = h->wall_kind == 1 && h->wall_hi();
    constexpr int ISO_TRIM = 14;
    const int ns_min = (Lx + S2::TX - 1) / S2::TX;
    double best = 1e300;
    for (int ns = ns_min; ns <= ns_min + ns_min / 4 + 1; ++ns) {
        // strips start on 32-byte sectors (w a multiple of 4): consumer rows are whole sectors
        int w = 4 * ((Lx + 4 * ns - 1) / (4 * ns));
        if (w > S2::TX) continue;
        if (w < 8) w = 8;
        const int strips = (Lx + w - 1) / w;
        for (int chunks = 1; chunks <= (Lz + 15) / 16; ++chunks) {
            // wall_kind 1: a block on an isothermal wall spends four of its passes on the wall adjustment of rows
            // 0..2 / Lz-3..Lz-1 in both steps (two more equilibrium evaluations per site, ~2.9 us per such pass against
            // ~1.7 us: +11 us measured at 512x1024, profiles/r3_wall_kind1.md), and a launch waits for its slowest
            // block: those chunks are ISO_TRIM rows shorter, the others share the rows.
            int tlo = iso_lo ? ISO_TRIM : 0, thi = iso_hi ? ISO_TRIM : 0;
            int ZC = (Lz + tlo + thi + chunks - 1) / chunks;
            ZC = (ZC + 1) / 2 * 2;                            // whole passes of R = 2 rows
            if (chunks == 1 || ZC < 4 * ISO_TRIM) {           // nothing to balance against / chunks too short to trim
                tlo = thi = 0;
                ZC = ((Lz + chunks - 1) / chunks + 1) / 2 * 2;
            }
            if (ZC < 6) ZC = 6;
            const int nch = (Lz + tlo + ZC - 1) / ZC;
            const long long waves = ((long long)strips * nch + sms - 1) / sms;
            // x (1 + ZC / 16000): blocks that march for thousands of rows drift apart, and the columns two neighbouring
            // strips both load stop meeting in L2 (4096x8192 in one wave of 4096-row chunks: -6 %)
            const double cost = ((double)waves + 0.15) * (ZC + 6 + 10) * (1.0 + ZC / 16000.0);
            if (cost < best - 1e-9) { best = cost; p.w = w; p.strips = strips; p.ZC = ZC; p.chunks = nch; p.trim = tlo; }
        }
    }
    if (h->zchunk > 0) {                                      // rows per block forced (tests, experiments)
        p.trim = 0;
        p.ZC = h->zchunk;
        p.chunks = (Lz + p.ZC - 1) / p.ZC;
        best = ((double)(((long long)p.strips * p.chunks + sms - 1) / sms) + 0.15) * (p.ZC + 16) * (1.0 + p.ZC / 16000.0);
    }
    // predicted time of two steps, microseconds: the two-step kernel spends ~0.65-0.7 us per unit of the cost above
    // on lattices of up to a few million sites (1.3-1.4 us per pass of two rows; the largest lattices, DRAM- and
    // power-bound, need 0.9) plus ~4 us per launch; the one-step kernel ~92 ps per site and step plus ~3 us per launch
    // (profiles/r2_sweep.md)
    const double t_fused = 0.66 * best + 4.0;
    const double t_single = 2.0 * (92e-6 * (double)Lx * Lz + 3.0);
    const bool can_fuse = h->tma_ok && !h->inplace;
    p.fused = can_fuse && (h->variant == 3 || (h->variant == 0 && t_fused < t_single));
    p.valid = true;
    return p;
}

// the plan of lbm_step / lbm_slab_step2 over the rows to update (a slab: its own rows), cached
const lbm_plan &make_plan(lbm_t *h)
{
    if (!h->plan.valid) h->plan = compute_plan(h, h->nz);
    return h->plan;
}

// periodic images for the two-step kernel's boxes (a1), if copy `i` was last written by anything but that kernel
int refresh_wrap_columns(lbm_t *h, int i, cudaStream_t st)
{
    // Under stream capture the refresh is always recorded: a replay may follow lbm_set_populations / lbm_init_*, whose
    // writes leave the wrap columns stale, and the graph must not depend on what wrap_ok said at capture time.
    // Once per capture is enough: later launches of the same capture read rows the two-step kernel itself wrote.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    unsigned long long cap_id = 0;
    if (cudaStreamGetCaptureInfo(st, &cap, &cap_id) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
    const bool first_of_capture = cap != cudaStreamCaptureStatusNone && (!h->cap_seen || h->cap_id != cap_id);
    if (first_of_capture) { h->cap_seen = true; h->cap_id = cap_id; }
    if (h->wrap_ok[i] && !first_of_capture) return LBM_OK;
    lbm::wrap_columns_kernel<lbm::XW><<<h->Lz, 2 * lbm::XW * LBM_NPOP, 0, st>>>(h->buf[i], h->layout());
    LAUNCHED(h);
    h->wrap_ok[i] = true;
    return LBM_OK;
}

template <bool ISO>
int launch_one_step(lbm_t *h, const lbm::StepArgs &a, int k0, int k1, cudaStream_t st)
{
    if (k1 <= k0) return LBM_OK;
    const int rows = k1 - k0;
    if (h->inplace) {
        // even steps scatter back to the gathered slots, odd steps are local (lbm_step.cuh)
        if ((long long)h->Lx * h->Lz < (1LL << 20)) {
            const dim3 grid((h->Lx + 127) / 128, rows);
            if (!h->layout_m) lbm::step_inplace_even_kernel<128, ISO><<<grid, 128, 0, st>>>(a, k0, k1);
            else lbm::step_inplace_odd_kernel<128, ISO><<<grid, 128, 0, st>>>(a, k0, k1);
        } else {                                   // as for the two-copy kernel: 256 threads on the large lattices (+0.7 %)
            const dim3 grid((h->Lx + 255) / 256, rows);
            if (!h->layout_m) lbm::step_inplace_even_kernel<256, ISO><<<grid, 256, 0, st>>>(a, k0, k1);
            else lbm::step_inplace_odd_kernel<256, ISO><<<grid, 256, 0, st>>>(a, k0, k1);
        }
    } else if (h->variant == 2 || (h->variant == 0 && (long long)h->Lx * h->Lz < (1LL << 20))) {
        // 128-thread blocks are a few per cent faster on the small (L2-resident, few-wave) lattices, 256 on the large
        lbm::step_kernel_site<128, 1, ISO><<<dim3((h->Lx + 127) / 128, rows), dim3(128, 1), 0, st>>>(a, k0, k1);
    } else {  // 256 threads = 2 blocks/SM at 128 registers: fastest one-step shape at 4096x8192
        lbm::step_kernel_site<256, 1, ISO><<<dim3((h->Lx + 255) / 256, rows), dim3(256, 1), 0, st>>>(a, k0, k1);
    }
    LAUNCHED(h);
    return LBM_OK;
}

int one_step_rows(lbm_t *h, lbm::StepArgs &a, int k0, int k1, cudaStream_t st)
{
    a.src = h->buf[h->cur];
    a.dst = h->inplace ? h->buf[h->cur] : h->buf[h->cur ^ 1];
    if (h->wall_kind != 1) return launch_one_step<false>(h, a, k0, k1, st);
    // wall_kind 1: the instance with the wall adjustment (twice the code, a dozen spilled registers) is needed by the
    // three rows next to an isothermal wall only.  Where two extra launches cost nothing (large lattices) those rows
    // get launches of their own and the rest runs the plain instance; rows of a launch are independent of each other.
    if ((long long)h->Lx * h->Lz < (1LL << 20)) return launch_one_step<true>(h, a, k0, k1, st);
    const int lo = a.iso_lo ? std::min(k1, std::max(k0, 3)) : k0;
    const int hi = a.iso_hi ? std::max(lo, std::min(k1, h->Lz - 3)) : k1;
    int rc = launch_one_step<true>(h, a, k0, lo, st);
    if (!rc) rc = launch_one_step<false>(h, a, lo, hi, st);
    if (!rc) rc = launch_one_step<true>(h, a, hi, k1, st);
    return rc;
}

// a5: after a step the other copy is current (two copies) or the layout has alternated (one copy)
void advance(lbm_t *h, int nsteps)
{
    if (h->inplace) {
        if (nsteps % 2) h->layout_m = !h->layout_m;
    } else {
        h->cur ^= 1;
    }
    h->steps += nsteps;
}

// one launch of the two-step kernel over the rows [zbase, zend) of `a`, from the current copy into the other one
int launch_two_step_rows(lbm_t *h, lbm::StepArgs &a, const lbm_plan &plan, cudaStream_t st)
{
    using S2 = lbm::Step2sWide;
    dim3 grid(plan.strips, plan.chunks);
    a.w = plan.w;
    a.ztrim = plan.trim;
    // the consumers' spare lanes of the two seam strips keep the wrap columns of the destination current, if the
    // seam columns [0, XW) and [Lx - XW, Lx) each lie within one strip and that strip has XW lanes to spare (2 XW
    // if it is the only strip); else the columns are refreshed before every launch
    const int last = h->Lx - (plan.strips - 1) * plan.w;      // columns of the last strip
    a.wrap_store = h->Lx >= 2 * lbm::XW && last >= lbm::XW &&
                   (plan.strips > 1 ? plan.w + lbm::XW <= S2::CW : last + 2 * lbm::XW <= S2::CW);
    int rc = refresh_wrap_columns(h, h->cur, st);
    if (rc) return rc;
    a.src = h->buf[h->cur];
    a.dst = h->buf[h->cur ^ 1];
    if (h->wall_kind == 1)
        lbm::step2s_kernel<S2, true><<<grid, S2::THREADS, S2::SMEM, st>>>(a, h->maps[h->cur], plan.ZC);
    else
        lbm::step2s_kernel<S2, false><<<grid, S2::THREADS, S2::SMEM, st>>>(a, h->maps[h->cur], plan.ZC);
    LAUNCHED(h);
    return LBM_OK;
}

// ... over all rows to update, then the other copy is current (lbm_step; lbm_slab_step2)
int launch_two_step(lbm_t *h, lbm::StepArgs &a, const lbm_plan &plan, cudaStream_t st)
{
    int rc = launch_two_step_rows(h, a, plan, st);
    if (rc) return rc;
    h->wrap_ok[h->cur ^ 1] = a.wrap_store != 0;   // the spare lanes of the seam strips wrote the images (own rows)
    advance(h, 2);                               // a5: swap prv / nxt, once per two steps
    return LBM_OK;
}

int create_common(lbm_t **out, int Lx, int rows_stored, const lbm_params *p, const char *fn)
{
    if (!out) return fail(LBM_ERR_INVALID, "%s: out is null", fn);
    *out = nullptr;
    if (!p) return fail(LBM_ERR_INVALID, "%s: params is null", fn);
    // Lx >= 7 keeps the seven wrapped source columns of a site distinct (one wrap suffices); Lz >= 6
    // keeps the three wall rows of the two walls disjoint
    if (Lx < 7 || rows_stored < 6) return fail(LBM_ERR_INVALID, "%s: need Lx >= 7 and Lz >= 6 (got %d x %d)", fn, Lx, rows_stored);
    if (rows_stored > 65535) return fail(LBM_ERR_INVALID, "%s: Lz <= 65535 (got %d)", fn, rows_stored);
    if (!(p->tau > 0.5)) return fail(LBM_ERR_INVALID, "%s: tau must be > 0.5 (got %g)", fn, p->tau);
    if (!(p->g >= 0.0)) return fail(LBM_ERR_INVALID, "%s: g must be >= 0 (got %g)", fn, p->g);
    if (p->wall_kind != 0 && p->wall_kind != 1) return fail(LBM_ERR_INVALID, "%s: wall_kind %d not supported", fn, p->wall_kind);
    if (p->wall_kind == 1 && !(p->T_wall_bottom > 0.0 && p->T_wall_top > 0.0))
        return fail(LBM_ERR_INVALID, "%s: wall_kind 1 needs wall temperatures > 0 (got %g, %g)", fn, p->T_wall_bottom, p->T_wall_top);
    if (!p->pop_buf0 || p->pop_buf0 == p->pop_buf1)
        return fail(LBM_ERR_INVALID, "%s: pop_buf0 must be set and differ from pop_buf1", fn);
    if (((uintptr_t)p->pop_buf0 | (uintptr_t)p->pop_buf1) & 255)
        return fail(LBM_ERR_INVALID, "%s: population buffers must be 256-byte aligned", fn);
    const size_t need = (size_t)plane_of(Lx, rows_stored) * LBM_NPOP * sizeof(double);
    if (p->buf_bytes < need) return fail(LBM_ERR_INVALID, "%s: buffers have %zu bytes, need %zu", fn, p->buf_bytes, need);
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(LBM_ERR_NODEVICE, "%s: no CUDA device", fn);
    }
    if (prop.major != 10) return fail(LBM_ERR_NODEVICE, "%s: built for sm_100a, device is sm_%d%d", fn, prop.major, prop.minor);
    lbm_handle *h = new (std::nothrow) lbm_handle();
    if (!h) return fail(LBM_ERR_INVALID, "%s: out of host memory", fn);
    h->dev = dev;
    h->Lx = Lx; h->Lz = rows_stored; h->pitch = pitch_of(Lx); h->plane = plane_of(Lx, rows_stored);
    h->tau = p->tau; h->g = p->g; h->sm_count = prop.multiProcessorCount;
    h->wall_kind = p->wall_kind; h->T_wall_lo = p->T_wall_bottom; h->T_wall_hi = p->T_wall_top;
    h->ubuf[0] = (double *)p->pop_buf0; h->ubuf[1] = (double *)p->pop_buf1;
    h->buf[0] = h->ubuf[0] + lbm::XH;
    h->buf[1] = h->ubuf[1] ? h->ubuf[1] + lbm::XH : nullptr;
    h->inplace = h->ubuf[1] == nullptr; h->layout_m = false;
    h->wrap_ok[0] = h->wrap_ok[1] = false; h->cap_seen = false; h->cap_id = 0;
    h->slab = false; h->Lz_glob = rows_stored; h->z0 = 0; h->nz = rows_stored; h->glo = h->ghi = 0; h->slab_phase = 0;
    h->cur = 0; h->steps = 0; h->launches = 0; h->variant = 0; h->zchunk = 0; h->scratch = nullptr; h->plane_stage = nullptr;
    h->plan = lbm_plan{}; h->plan_interior = lbm_plan{};
    h->tma_ok = false;
    h->persist_tb = h->persist_blocks = 0; h->d_counter = nullptr;
    for (auto &s : h->stage) s = nullptr;
    *out = h;
    return LBM_OK;
}

int finish_create(lbm_t **out, const char *fn)
{
    lbm_handle *h = *out;
    if (!h->inplace) {
        h->tma_ok = encode_step2s_maps(h->ubuf[0], h->Lx, h->Lz, h->pitch, h->plane, h->maps[0]) &&
                    encode_step2s_maps(h->ubuf[1], h->Lx, h->Lz, h->pitch, h->plane, h->maps[1]);
        // the opt-in to > 48 KB of dynamic shared memory is per device (context), so it is made for every handle
        using S2 = lbm::Step2sWide;
        if (h->tma_ok && (cudaFuncSetAttribute(lbm::step2s_kernel<S2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S2::SMEM) != cudaSuccess ||
                          cudaFuncSetAttribute(lbm::step2s_kernel<S2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S2::SMEM) != cudaSuccess)) {
            cudaGetLastError();
            h->tma_ok = false;
        }
    }
    // Small lattices (one site per co-resident thread): lbm_step(n) is one cooperative launch of the persistent kernel
    if (!h->inplace && !h->slab) {
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->dev);
        const long long sites = (long long)h->Lx * h->Lz;
        const int tb = sites <= 64LL * h->sm_count ? 64 : 128;       // spread a tiny lattice over all SMs
        const long long blocks = (sites + tb - 1) / tb;
        int per_sm = 0;
        cudaError_t eo = tb == 64 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lbm::step_persistent_kernel<64, false>, 64, 0)
                                  : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, lbm::step_persistent_kernel<128, false>, 128, 0);
        if (coop && eo == cudaSuccess && blocks <= (long long)per_sm * h->sm_count && blocks <= 2LL * h->sm_count &&
            cudaMalloc(&h->d_counter, sizeof(unsigned)) == cudaSuccess) {
            h->persist_tb = tb;
            h->persist_blocks = (int)blocks;
        }
        cudaGetLastError();
    }
    cudaError_t e = cudaMalloc(&h->scratch, sizeof(double) * (8LL * h->nz + 8 + 2LL * h->Lx));
    if (e != cudaSuccess) {
        cudaGetLastError();
        h->scratch = nullptr;
        lbm_destroy(h);                  // frees the barrier counter too
        *out = nullptr;
        return fail(LBM_ERR_CUDA, "%s: cudaMalloc scratch: %s", fn, cudaGetErrorString(e));
    }
    return LBM_OK;
}

// the 26 (row, population) pairs of a slab message; `send`: the own rows the neighbour on `side` needs, else the
// ghost rows on `side` that the neighbour's message fills
lbm::SlabRows slab_rows(const lbm_t *h, int side, bool send)
{
    lbm::SlabRows s;
    int j = 0;
    for (int d = 1; d <= GHOST; ++d) {
        // side 1 (above): the upper neighbour's ghost row at distance d below its first row is my own row nz - d;
        // it is read by its rows 0 .. 3-d with e_z >= d.  side 0 (below): mirror image, e_z <= -d.
        int row;
        if (send) row = side == 1 ? h->glo + h->nz - d : h->glo + d - 1;
        else row = side == 1 ? h->glo + h->nz + d - 1 : h->glo - d;
        for (int l = 0; l < LBM_NPOP; ++l) {
            const int ez = d2q37::pop_ez(l);
            const bool wanted = send ? (side == 1 ? ez >= d : ez <= -d) : (side == 1 ? ez <= -d : ez >= d);
            if (wanted) { s.row[j] = row; s.l[j] = l; ++j; }
        }
    }
    return s;  // j == 26
}

}  // namespace

extern "C" {

const char *lbm_last_error(void) { return g_err; }

size_t lbm_buffer_bytes(int Lx, int Lz)
{
    if (Lx < 7 || Lz < 6) return 0;
    return (size_t)plane_of(Lx, Lz) * LBM_NPOP * sizeof(double);
}

size_t lbm_slab_buffer_bytes(int Lx, int Lz_global, int z0, int nz)
{
    if (Lx < 7 || Lz_global < 6 || z0 < 0 || nz < 2 * GHOST || z0 + nz > Lz_global) return 0;   // as lbm_create_slab
    const int rows = nz + (z0 > 0 ? GHOST_STORED : 0) + (z0 + nz < Lz_global ? GHOST_STORED : 0);
    return rows < 6 ? 0 : (size_t)plane_of(Lx, rows) * LBM_NPOP * sizeof(double);
}

int lbm_tables(int *ex, int *ez, double *w, double *r)
{
    for (int l = 0; l < LBM_NPOP; ++l) {
        if (ex) ex[l] = d2q37::pop_ex(l);
        if (ez) ez[l] = d2q37::pop_ez(l);
        if (w) w[l] = d2q37::shell_weight(d2q37::pop_e2(l));
    }
    if (r) *r = D2Q37_R;
    return LBM_OK;
}

int lbm_create(lbm_t **out, int Lx, int Lz, const lbm_params *p)
{
    int rc = create_common(out, Lx, Lz, p, "lbm_create");
    if (rc) return rc;
    return finish_create(out, "lbm_create");
}

int lbm_create_slab(lbm_t **out, int Lx, int Lz_global, int z0, int nz, const lbm_params *p)
{
    if (out) *out = nullptr;
    if (Lz_global < 6 || z0 < 0 || nz < 2 * GHOST || z0 + nz > Lz_global)
        return fail(LBM_ERR_INVALID, "lbm_create_slab: rows [%d, %d) of %d: a slab needs >= %d rows inside the lattice",
                    z0, z0 + nz, Lz_global, 2 * GHOST);
    if (p && !p->pop_buf1) return fail(LBM_ERR_INVALID, "lbm_create_slab: a slab needs two lattice copies");
    const int glo = z0 > 0 ? GHOST_STORED : 0, ghi = z0 + nz < Lz_global ? GHOST_STORED : 0;
    int rc = create_common(out, Lx, glo + nz + ghi, p, "lbm_create_slab");
    if (rc) return rc;
    lbm_handle *h = *out;
    h->slab = true; h->Lz_glob = Lz_global; h->z0 = z0; h->nz = nz; h->glo = glo; h->ghi = ghi;
    return finish_create(out, "lbm_create_slab");
}

int lbm_destroy(lbm_t *h)
{
    if (!h) return LBM_OK;
    cudaFree(h->scratch);
    cudaFree(h->d_counter);
    cudaFree(h->plane_stage);
    for (auto s : h->stage) cudaFree(s);
    delete h;
    return LBM_OK;
}

int lbm_init_rt(lbm_t *h, uint64_t seed, const lbm_rt_init *ic, void *stream)
{
    NEED(h);
    if (!ic) return fail(LBM_ERR_INVALID, "lbm_init_rt: ic is null");
    if (!(ic->T_d > 0 && ic->T_m > 0 && ic->T_u > 0 && ic->rho_m > 0) || ic->delta < 0 || ic->smooth_w < 0 ||
        ic->pert_kind < 0 || ic->pert_kind > 2 || ic->n_modes < 0)
        return fail(LBM_ERR_INVALID, "lbm_init_rt: invalid initial-state parameters");
    cudaStream_t st = (cudaStream_t)stream;
    SplitMix rng{seed};
    std::vector<double> h_lo, h_hi;
    draw_interface(rng, *ic, h->Lx, h_lo);
    if (ic->delta == 0.0) h_hi = h_lo;  // single front: one interface
    else draw_interface(rng, *ic, h->Lx, h_hi);
    CUDA_TRY(cudaMemcpyAsync(h->d_hlo(), h_lo.data(), sizeof(double) * h->Lx, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(h->d_hhi(), h_hi.data(), sizeof(double) * h->Lx, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaStreamSynchronize(st));  // the host vectors go out of scope
    lbm::RtArgs a{h->g, 1.0 / ic->T_d, 1.0 / ic->T_m, 1.0 / ic->T_u, ic->rho_m, ic->delta, ic->smooth_w,
                  h->Lz_glob, h->z0 - h->glo};
    // all stored rows: a slab's ghost rows start from the same closed form as its neighbours' own rows
    lbm::init_rt_kernel<<<dim3((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->Lz), lbm::AUX_TX, 0, st>>>(
        h->buf[h->cur], h->layout(), a, h->d_hlo(), h->d_hhi());
    LAUNCHED(h);
    h->steps = 0; h->layout_m = false; h->wrap_ok[h->cur] = false; h->slab_phase = 0;
    return LBM_OK;
}

int lbm_init_equilibrium(lbm_t *h, const double *rho, const double *ux, const double *uz, const double *T, void *stream)
{
    NEED(h);
    if (!rho || !ux || !uz || !T) return fail(LBM_ERR_INVALID, "lbm_init_equilibrium: null field");
    lbm::init_equilibrium_kernel<<<own_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), rho, ux, uz, T);
    LAUNCHED(h);
    h->steps = 0; h->layout_m = false; h->wrap_ok[h->cur] = false; h->slab_phase = 0;
    return LBM_OK;
}

int lbm_set_populations(lbm_t *h, const double *f_dev, void *stream)
{
    NEED(h);
    if (!f_dev) return fail(LBM_ERR_INVALID, "lbm_set_populations: null pointer");
    dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->nz, LBM_NPOP);
    h->layout_m = false;                 // the uploaded state is stored in the ordinary layout
    lbm::pack_kernel<<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(h->buf[h->cur], h->layout(), f_dev, 0);
    LAUNCHED(h);
    h->wrap_ok[h->cur] = false; h->slab_phase = 0;
    return LBM_OK;
}

int lbm_get_populations(lbm_t *h, double *f_dev, void *stream)
{
    NEED(h);
    if (!f_dev) return fail(LBM_ERR_INVALID, "lbm_get_populations: null pointer");
    dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->nz, LBM_NPOP);
    lbm::unpack_kernel<<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(h->buf[h->cur], h->layout(), f_dev, 0);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_get_window(lbm_t *h, int k0, int nk, int i0, int ni, double *f_dev, void *stream)
{
    NEED(h);
    if (!f_dev) return fail(LBM_ERR_INVALID, "lbm_get_window: null pointer");
    if (k0 < 0 || nk < 1 || k0 + nk > h->nz || ni < 1 || ni > h->Lx)
        return fail(LBM_ERR_INVALID, "lbm_get_window: rows [%d, %d) of %d, %d columns of %d", k0, k0 + nk, h->nz, ni, h->Lx);
    dim3 grid((ni + lbm::AUX_TX - 1) / lbm::AUX_TX, nk, LBM_NPOP);
    lbm::window_kernel<<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(h->buf[h->cur], h->layout(), k0, nk, i0, ni, f_dev);
    LAUNCHED(h);
    return LBM_OK;
}

// Host variants.  Two copies: the whole dense array is staged in the OTHER lattice copy (free between steps), so no
// extra device memory.  One copy (in-place): one dense population plane at a time through a plane-sized buffer.
int lbm_set_populations_host(lbm_t *h, const double *f_host, void *stream)
{
    NEED(h);
    if (!f_host) return fail(LBM_ERR_INVALID, "lbm_set_populations_host: null pointer");
    // two-copy handles stage through the OTHER lattice copy, which holds the interior rows of a half-done slab step
    if (h->slab && h->slab_phase != 0)
        return fail(LBM_ERR_INVALID, "lbm_set_populations_host: a slab step is half done (interior launched, edges pending); finish it first");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t plane_elems = (size_t)h->Lx * h->nz;
    if (!h->inplace) {
        double *tmp = h->ubuf[h->cur ^ 1];
        CUDA_TRY(cudaMemcpyAsync(tmp, f_host, sizeof(double) * LBM_NPOP * plane_elems, cudaMemcpyHostToDevice, st));
        int rc = lbm_set_populations(h, tmp, stream);
        if (rc) return rc;
        h->wrap_ok[h->cur ^ 1] = false;
    } else {
        if (!h->plane_stage) CUDA_TRY(cudaMalloc(&h->plane_stage, sizeof(double) * plane_elems));
        h->layout_m = false;
        dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->nz, 1);
        for (int l = 0; l < LBM_NPOP; ++l) {
            CUDA_TRY(cudaMemcpyAsync(h->plane_stage, f_host + l * plane_elems, sizeof(double) * plane_elems, cudaMemcpyHostToDevice, st));
            lbm::pack_kernel<<<grid, lbm::AUX_TX, 0, st>>>(h->buf[h->cur], h->layout(), h->plane_stage, l);
            LAUNCHED(h);
        }
        h->wrap_ok[h->cur] = false;
    }
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_get_populations_host(lbm_t *h, double *f_host, void *stream)
{
    NEED(h);
    if (!f_host) return fail(LBM_ERR_INVALID, "lbm_get_populations_host: null pointer");
    // two-copy handles stage through the OTHER lattice copy, which holds the interior rows of a half-done slab step
    if (h->slab && h->slab_phase != 0)
        return fail(LBM_ERR_INVALID, "lbm_get_populations_host: a slab step is half done (interior launched, edges pending); finish it first");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t plane_elems = (size_t)h->Lx * h->nz;
    if (!h->inplace) {
        double *tmp = h->ubuf[h->cur ^ 1];
        int rc = lbm_get_populations(h, tmp, stream);
        if (rc) return rc;
        h->wrap_ok[h->cur ^ 1] = false;
        CUDA_TRY(cudaMemcpyAsync(f_host, tmp, sizeof(double) * LBM_NPOP * plane_elems, cudaMemcpyDeviceToHost, st));
    } else {
        if (!h->plane_stage) CUDA_TRY(cudaMalloc(&h->plane_stage, sizeof(double) * plane_elems));
        dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->nz, 1);
        for (int l = 0; l < LBM_NPOP; ++l) {
            lbm::unpack_kernel<<<grid, lbm::AUX_TX, 0, st>>>(h->buf[h->cur], h->layout(), h->plane_stage, l);
            LAUNCHED(h);
            CUDA_TRY(cudaMemcpyAsync(f_host + l * plane_elems, h->plane_stage, sizeof(double) * plane_elems, cudaMemcpyDeviceToHost, st));
        }
    }
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_step(lbm_t *h, int n, void *stream)
{
    NEED(h);
    if (n < 0) return fail(LBM_ERR_INVALID, "lbm_step: n must be >= 0 (got %d)", n);
    if (h->slab) return fail(LBM_ERR_INVALID, "lbm_step: a z-slab is stepped with lbm_slab_step (its ghost rows must be exchanged every step)");
    cudaStream_t st = (cudaStream_t)stream;
    lbm::StepArgs a = step_args(h);
    // Variants: 0 = automatic (make_plan), 1 = one step per launch, 256x1 blocks, 2 = one step, 128x1 blocks,
    // 3 = two steps per launch forced.  An odd last step always runs the one-step kernel.
    using S2 = lbm::Step2sWide;
    const lbm_plan &plan = make_plan(h);
    if (h->variant == 3 && !plan.fused)
        return fail(h->inplace ? LBM_ERR_INVALID : LBM_ERR_CUDA, "lbm_step: the two-step kernel needs two lattice copies and tensor maps%s",
                    h->inplace || h->tma_ok ? "" : " (cuTensorMapEncodeTiled failed)");
    const bool persistent = h->persist_blocks > 0 && h->variant == 0 && !plan.fused && n >= 2;
    // Under stream capture the handle's bookkeeping (which copy is current) advances at capture time, not at replay:
    // a captured sequence must leave the current copy / layout where it was, i.e. swap the copies an even number of times.
    const int swaps = persistent ? n : plan.fused ? n / 2 + n % 2 : n;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) { cudaGetLastError(); cap = cudaStreamCaptureStatusNone; }
    if (cap != cudaStreamCaptureStatusNone && swaps % 2)
        return fail(LBM_ERR_INVALID, "lbm_step: %d steps swap the lattice copies %d times here; a captured sequence must "
                    "swap them an even number of times (the ping-pong must return to the same copy)", n, swaps);
    if (persistent) {       // small lattice: all n steps in one cooperative launch (lbm_step.cuh)
        const void *fn = h->persist_tb == 64
                             ? (h->wall_kind == 1 ? (const void *)lbm::step_persistent_kernel<64, true> : (const void *)lbm::step_persistent_kernel<64, false>)
                             : (h->wall_kind == 1 ? (const void *)lbm::step_persistent_kernel<128, true> : (const void *)lbm::step_persistent_kernel<128, false>);
        // ... in launches of at most PERSIST_MAX_STEPS steps: the barrier counter must not run a whole 2^31 ahead
        bool launched = true;
        cudaError_t le = cudaSuccess;
        while (n > 0 && launched) {
            double *b0 = h->buf[0], *b1 = h->buf[1];
            int cur = h->cur, nn = n < lbm::PERSIST_MAX_STEPS ? n : lbm::PERSIST_MAX_STEPS;
            static_assert(lbm::BARRIER_START == 0xFFFFFFFFu, "the byte memset below writes BARRIER_START");
            CUDA_TRY(cudaMemsetAsync(h->d_counter, 0xFF, sizeof(unsigned), st));
            void *args[] = {&a, &b0, &b1, &cur, &nn, &h->d_counter};
            le = cudaLaunchCooperativeKernel(fn, dim3(h->persist_blocks), dim3(h->persist_tb), args, 0, st);
            launched = le == cudaSuccess;
            if (launched) {
                h->launches++;
                h->wrap_ok[0] = h->wrap_ok[1] = false;
                if (nn % 2) h->cur ^= 1;
                h->steps += nn;
                n -= nn;
            }
        }
        if (launched) return LBM_OK;
        cudaGetLastError();
        // Only "the grid is not co-resident after all" (a shared or partitioned GPU) turns the persistent path off for
        // good: launched steps from now on.  Anything else (a bad stream, a broken capture) is the caller's to see.
        if (le != cudaErrorCooperativeLaunchTooLarge && le != cudaErrorLaunchOutOfResources)
            return fail(LBM_ERR_CUDA, "lbm_step: cooperative launch of the persistent kernel: %s", cudaGetErrorString(le));
        h->persist_blocks = 0;
        if (cap != cudaStreamCaptureStatusNone && n % 2)
            return fail(LBM_ERR_INVALID, "lbm_step: %d launched steps cannot be captured (odd number of swaps)", n);
    }
    int s = 0;
    if (plan.fused && n >= 2) {
        for (; s + 2 <= n; s += 2) {
            int rc = launch_two_step(h, a, plan, st);
            if (rc) return rc;
        }
    }
    for (; s < n; ++s) {
        int rc = one_step_rows(h, a, 0, h->Lz, st);
        if (rc) return rc;
        h->wrap_ok[h->inplace ? h->cur : h->cur ^ 1] = false;
        advance(h, 1);                                   // a5
    }
    return LBM_OK;
}

int lbm_get_plan(lbm_t *h, int *fused, int *strip_width, int *zchunk)
{
    NEED_HOST(h);
    const lbm_plan &p = make_plan(h);
    if (fused) *fused = p.fused ? 1 : 0;
    if (strip_width) *strip_width = p.w;
    if (zchunk) *zchunk = p.ZC;
    return LBM_OK;
}

// ---- z-slabs (Fig. 3-4) -------------------------------------------------------
int lbm_slab_info(const lbm_t *h, int *z0, int *nz, int *open_below, int *open_above, size_t *message_doubles,
                  size_t *message2_doubles)
{
    NEED_HOST(h);
    if (!h->slab) return fail(LBM_ERR_INVALID, "lbm_slab_info: not a slab handle");
    if (z0) *z0 = h->z0;
    if (nz) *nz = h->nz;
    if (open_below) *open_below = h->glo > 0;
    if (open_above) *open_above = h->ghi > 0;
    if (message_doubles) *message_doubles = (size_t)26 * h->Lx;
    if (message2_doubles) *message2_doubles = (size_t)GHOST_STORED * LBM_NPOP * (h->Lx + 2 * lbm::XW);
    return LBM_OK;
}

int lbm_slab_pack(lbm_t *h, int side, double *msg_dev, void *stream)
{
    NEED(h);
    if (!h->slab || (side != 0 && side != 1) || !msg_dev) return fail(LBM_ERR_INVALID, "lbm_slab_pack: slab handle, side 0/1 and a buffer are required");
    if (side == 0 ? h->glo == 0 : h->ghi == 0) return fail(LBM_ERR_INVALID, "lbm_slab_pack: side %d of this slab is a wall", side);
    lbm::slab_pack_kernel<<<dim3((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, 26), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), slab_rows(h, side, true), msg_dev);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_slab_unpack(lbm_t *h, int side, const double *msg_dev, void *stream)
{
    NEED(h);
    if (!h->slab || (side != 0 && side != 1) || !msg_dev) return fail(LBM_ERR_INVALID, "lbm_slab_unpack: slab handle, side 0/1 and a buffer are required");
    if (side == 0 ? h->glo == 0 : h->ghi == 0) return fail(LBM_ERR_INVALID, "lbm_slab_unpack: side %d of this slab is a wall", side);
    lbm::slab_unpack_kernel<<<dim3((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, 26), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), slab_rows(h, side, false), msg_dev);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_slab_step(lbm_t *h, int part, void *stream)
{
    NEED(h);
    if (!h->slab) return fail(LBM_ERR_INVALID, "lbm_slab_step: not a slab handle");
    cudaStream_t st = (cudaStream_t)stream;
    lbm::StepArgs a = step_args(h);
    // own rows that read no ghost row: at least GHOST rows away from an open side
    const int i0 = h->glo + (h->glo ? GHOST : 0), i1 = h->glo + h->nz - (h->ghi ? GHOST : 0);
    if (part == LBM_SLAB_INTERIOR) {
        if (h->slab_phase != 0) return fail(LBM_ERR_INVALID, "lbm_slab_step: interior rows of this step were already launched");
        int rc = one_step_rows(h, a, i0, i1, st);
        if (rc) return rc;
        h->slab_phase = 1;
        return LBM_OK;
    }
    if (part == LBM_SLAB_EDGES) {
        if (h->slab_phase != 1) return fail(LBM_ERR_INVALID, "lbm_slab_step: launch the interior rows first");
        int rc = one_step_rows(h, a, h->glo, i0, st);
        if (!rc) rc = one_step_rows(h, a, i1, h->glo + h->nz, st);
        if (rc) return rc;
        h->slab_phase = 0;
        h->wrap_ok[h->cur ^ 1] = false;
        advance(h, 1);                                   // a5
        return LBM_OK;
    }
    return fail(LBM_ERR_INVALID, "lbm_slab_step: part must be LBM_SLAB_INTERIOR or LBM_SLAB_EDGES (got %d)", part);
}

// Two fused steps of a slab.  They read 6 ghost rows per open side, complete (all populations) and with their wrap
// columns: lbm_slab_pack2 / lbm_slab_unpack2 move whole rows.
int lbm_slab_pack2(lbm_t *h, int side, double *msg_dev, void *stream)
{
    NEED(h);
    if (!h->slab || (side != 0 && side != 1) || !msg_dev) return fail(LBM_ERR_INVALID, "lbm_slab_pack2: slab handle, side 0/1 and a buffer are required");
    if (side == 0 ? h->glo == 0 : h->ghi == 0) return fail(LBM_ERR_INVALID, "lbm_slab_pack2: side %d of this slab is a wall", side);
    if (h->slab_phase != 0) return fail(LBM_ERR_INVALID, "lbm_slab_pack2: a one-step slab step is half done");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = refresh_wrap_columns(h, h->cur, st);          // the message carries the images of my rows
    if (rc) return rc;
    const int row0 = side == 1 ? h->glo + h->nz - GHOST_STORED : h->glo;
    dim3 grid((h->Lx + 2 * lbm::XW + lbm::AUX_TX - 1) / lbm::AUX_TX, GHOST_STORED, LBM_NPOP);
    lbm::slab_rows_kernel<lbm::XW, true><<<grid, lbm::AUX_TX, 0, st>>>(h->buf[h->cur], h->layout(), row0, msg_dev);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_slab_unpack2(lbm_t *h, int side, const double *msg_dev, void *stream)
{
    NEED(h);
    if (!h->slab || (side != 0 && side != 1) || !msg_dev) return fail(LBM_ERR_INVALID, "lbm_slab_unpack2: slab handle, side 0/1 and a buffer are required");
    if (side == 0 ? h->glo == 0 : h->ghi == 0) return fail(LBM_ERR_INVALID, "lbm_slab_unpack2: side %d of this slab is a wall", side);
    const int row0 = side == 1 ? h->glo + h->nz : 0;
    dim3 grid((h->Lx + 2 * lbm::XW + lbm::AUX_TX - 1) / lbm::AUX_TX, GHOST_STORED, LBM_NPOP);
    lbm::slab_rows_kernel<lbm::XW, false><<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), row0, const_cast<double *>(msg_dev));
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_slab_step2(lbm_t *h, void *stream)
{
    NEED(h);
    if (!h->slab) return fail(LBM_ERR_INVALID, "lbm_slab_step2: not a slab handle");
    if (h->slab_phase != 0) return fail(LBM_ERR_INVALID, "lbm_slab_step2: a one-step slab step is half done");
    if (h->nz < GHOST_STORED) return fail(LBM_ERR_INVALID, "lbm_slab_step2: a slab needs at least %d rows", GHOST_STORED);
    if (!h->tma_ok) return fail(LBM_ERR_CUDA, "lbm_slab_step2: the two-step kernel needs tensor maps (cuTensorMapEncodeTiled failed)");
    const lbm_plan &plan = make_plan(h);                     // strips and chunks over the slab's own rows
    lbm::StepArgs a = step_args(h);
    return launch_two_step(h, a, plan, (cudaStream_t)stream);
}

// The same two steps in two parts, so that the exchange of the ghost rows hides behind the bulk (Fig. 4):
// INTERIOR = own rows at least 6 rows away from an open side (they read no ghost row), EDGES = the 6 rows next to each
// open side, after lbm_slab_unpack2.  Three launches of the same kernel over disjoint row ranges: bit-identical to
// lbm_slab_step2.  Slabs too thin to have interior rows run everything in EDGES.
int lbm_slab_step2_part(lbm_t *h, int part, void *stream)
{
    NEED(h);
    if (!h->slab) return fail(LBM_ERR_INVALID, "lbm_slab_step2_part: not a slab handle");
    if (h->nz < GHOST_STORED) return fail(LBM_ERR_INVALID, "lbm_slab_step2_part: a slab needs at least %d rows", GHOST_STORED);
    if (!h->tma_ok) return fail(LBM_ERR_CUDA, "lbm_slab_step2_part: the two-step kernel needs tensor maps (cuTensorMapEncodeTiled failed)");
    cudaStream_t st = (cudaStream_t)stream;
    const int own0 = h->glo, own1 = h->glo + h->nz;
    int i0 = own0 + (h->glo ? GHOST_STORED : 0), i1 = own1 - (h->ghi ? GHOST_STORED : 0);
    if (i1 - i0 < GHOST_STORED) i0 = i1 = own0;              // no interior worth a launch: EDGES = [own0, own1)
    lbm::StepArgs a = step_args(h);
    const lbm_plan &whole = make_plan(h);
    if (part == LBM_SLAB_INTERIOR) {
        if (h->slab_phase != 0) return fail(LBM_ERR_INVALID, "lbm_slab_step2_part: a slab step is half done");
        if (i1 > i0) {
            if (!h->plan_interior.valid) h->plan_interior = compute_plan(h, i1 - i0);
            a.zbase = i0; a.zend = i1;
            int rc = launch_two_step_rows(h, a, h->plan_interior, st);
            if (rc) return rc;
        }
        h->slab_phase = 2;
        return LBM_OK;
    }
    if (part == LBM_SLAB_EDGES) {
        if (h->slab_phase != 2) return fail(LBM_ERR_INVALID, "lbm_slab_step2_part: launch the interior rows first");
        lbm_plan edge = whole;                               // same strips; one chunk of the rows of the range
        edge.trim = 0; edge.chunks = 1;
        const int ranges[2][2] = {{own0, i1 > i0 ? i0 : own1}, {i1 > i0 ? i1 : own1, own1}};
        if (ranges[0][1] - ranges[0][0] == GHOST_STORED && ranges[1][1] - ranges[1][0] == GHOST_STORED) {
            // both sides open: the two edge zones as the two chunk rows of ONE launch (twice the blocks, once the time)
            a.zbase = ranges[0][0]; a.zend = ranges[0][1];
            a.zsplit = 1; a.zbase2 = ranges[1][0]; a.zend2 = ranges[1][1];
            edge.ZC = GHOST_STORED; edge.chunks = 2;
            int rc = launch_two_step_rows(h, a, edge, st);
            if (rc) return rc;
        } else {
            for (auto &r : ranges) {
                if (r[1] <= r[0]) continue;
                a.zbase = r[0]; a.zend = r[1];
                edge.ZC = (r[1] - r[0] + 1) / 2 * 2;
                int rc = launch_two_step_rows(h, a, edge, st);
                if (rc) return rc;
            }
        }
        h->slab_phase = 0;
        h->wrap_ok[h->cur ^ 1] = a.wrap_store != 0;
        advance(h, 2);                                       // a5
        return LBM_OK;
    }
    return fail(LBM_ERR_INVALID, "lbm_slab_step2_part: part must be LBM_SLAB_INTERIOR or LBM_SLAB_EDGES (got %d)", part);
}

// ---- diagnostics (a6) ------------------------------------------------------------------------------------------------
int lbm_moments(lbm_t *h, double *rho, double *ux, double *uz, double *T, void *stream)
{
    NEED(h);
    if (!rho && !ux && !uz && !T) return fail(LBM_ERR_INVALID, "lbm_moments: all four outputs are null");
    lbm::moments_kernel<<<own_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), h->g, rho, ux, uz, T);
    LAUNCHED(h);
    return LBM_OK;
}

// eq. 7 as it stands (moments_kernel with no gravity shift): the inputs lbm_init_equilibrium / lbm_run_host take
int lbm_kinetic_moments(lbm_t *h, double *rho, double *ux, double *uz, double *T, void *stream)
{
    NEED(h);
    if (!rho && !ux && !uz && !T) return fail(LBM_ERR_INVALID, "lbm_kinetic_moments: all four outputs are null");
    lbm::moments_kernel<<<own_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), 0.0, rho, ux, uz, T);
    LAUNCHED(h);
    return LBM_OK;
}

// one pass over the lattice + one small block; results stay in the handle's scratch
static int run_diagnostics(lbm_t *h, bool want_rms, double T_d, double T_m, double T_u, cudaStream_t st)
{
    if (want_rms) {
        // the row's T and E_k stay in shared memory between the two passes if they fit (Lx <= 12 800), else the row is re-read
        const size_t smem = sizeof(double) * 2 * (size_t)h->Lx;
        const int keep = smem <= 200 * 1024;
        if (keep && smem > 48 * 1024)
            CUDA_TRY(cudaFuncSetAttribute(lbm::row_diagnostics_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        lbm::row_diagnostics_kernel<true><<<h->nz, lbm::RED_T, keep ? smem : 0, st>>>(h->buf[h->cur], h->layout(), h->g, h->d_rows(), keep);
    } else {
        lbm::row_diagnostics_kernel<false><<<h->nz, lbm::RED_T, 0, st>>>(h->buf[h->cur], h->layout(), h->g, h->d_rows(), 0);
    }
    LAUNCHED(h);
    lbm::final_diagnostics_kernel<<<1, lbm::RED_T, 0, st>>>(h->d_rows(), h->nz, T_d, T_m, T_u, h->d_result());
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_diagnostics(lbm_t *h, double T_d, double T_m, double T_u, double *widths2, double *totals4, double *Tbar,
                    double *Trms, double *Ekbar, double *Ekrms, void *stream)
{
    NEED(h);
    if (widths2 && (T_m == T_u || T_d == T_m)) return fail(LBM_ERR_INVALID, "lbm_diagnostics: layer temperatures must differ");
    cudaStream_t st = (cudaStream_t)stream;
    int rc = run_diagnostics(h, Trms || Ekrms, T_d, T_m, T_u, st);
    if (rc) return rc;
    double res[6];
    CUDA_TRY(cudaMemcpyAsync(res, h->d_result(), sizeof res, cudaMemcpyDeviceToHost, st));
    double *out[4] = {Tbar, Trms, Ekbar, Ekrms};
    for (int j = 0; j < 4; ++j)
        if (out[j]) CUDA_TRY(cudaMemcpyAsync(out[j], h->d_rows() + (long long)j * h->nz, sizeof(double) * h->nz, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (widths2) { widths2[0] = res[0]; widths2[1] = res[1]; }
    if (totals4) for (int j = 0; j < 4; ++j) totals4[j] = res[2 + j];
    return LBM_OK;
}

int lbm_mixing_widths(lbm_t *h, double T_d, double T_m, double T_u, double *L_u, double *L_d, double *Tbar, void *stream)
{
    NEED(h);
    if (!L_u || !L_d) return fail(LBM_ERR_INVALID, "lbm_mixing_widths: null output");
    if (T_m == T_u || T_d == T_m) return fail(LBM_ERR_INVALID, "lbm_mixing_widths: layer temperatures must differ");
    double w[2];
    int rc = lbm_diagnostics(h, T_d, T_m, T_u, w, nullptr, Tbar, nullptr, nullptr, nullptr, stream);
    if (rc) return rc;
    *L_u = w[0];
    *L_d = w[1];
    return LBM_OK;
}

int lbm_profiles(lbm_t *h, double *Tbar, double *Trms, double *Ekbar, double *Ekrms, void *stream)
{
    NEED(h);
    return lbm_diagnostics(h, 0.0, 0.0, 0.0, nullptr, nullptr, Tbar, Trms, Ekbar, Ekrms, stream);
}

int lbm_totals(lbm_t *h, double *out4, void *stream)
{
    NEED(h);
    if (!out4) return fail(LBM_ERR_INVALID, "lbm_totals: null output");
    return lbm_diagnostics(h, 0.0, 0.0, 0.0, nullptr, out4, nullptr, nullptr, nullptr, nullptr, stream);
}

int lbm_growth_rate(int n, const double *t, const double *L, double g, double At, double *alpha)
{
    if (n < 0 || (n > 0 && (!t || !L || !alpha))) return fail(LBM_ERR_INVALID, "lbm_growth_rate: null series");
    if (!(g > 0.0) || !(At > 0.0)) return fail(LBM_ERR_INVALID, "lbm_growth_rate: g and At must be > 0");
    for (int j = 0; j < n; ++j) {
        const int lo = j == 0 ? 0 : j - 1, hi = j == n - 1 ? j : j + 1;
        double slope = 0.0;
        if (hi > lo) {
            if (!(t[hi] > t[lo])) return fail(LBM_ERR_INVALID, "lbm_growth_rate: times must increase");
            slope = (L[hi] - L[lo]) / (t[hi] - t[lo]);
        }
        alpha[j] = L[j] > 0.0 ? (slope * slope) / (4.0 * g * At * L[j]) : 0.0;
    }
    return LBM_OK;
}

int lbm_rt_scales(double Lx, double g, double T_d, double T_u, double *At, double *tau_rt)
{
    if (!(Lx > 0.0) || !(g > 0.0) || !(T_d > T_u) || !(T_u > 0.0)) return fail(LBM_ERR_INVALID, "lbm_rt_scales: need Lx, g > 0 and T_d > T_u > 0");
    const double a = (T_d - T_u) / (T_d + T_u);
    if (At) *At = a;
    if (tau_rt) *tau_rt = std::sqrt(Lx / (g * a));
    return LBM_OK;
}

int lbm_fp64_peak(double *tflops, int iters, void *stream)
{
    if (!tflops) return fail(LBM_ERR_INVALID, "lbm_fp64_peak: null output");
    if (iters <= 0) iters = 4096;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(LBM_ERR_NODEVICE, "lbm_fp64_peak: no CUDA device");
    }
    double *sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, sizeof(double)));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 4;    // 4 x 256 threads = 8 warps per sub-partition
    lbm::fp64_peak_kernel<<<blocks, 256, 0, st>>>(sink, 16, 1.0000001, 1e-9);   // warm-up
    CUDA_TRY(cudaEventRecord(e0, st));
    lbm::fp64_peak_kernel<<<blocks, 256, 0, st>>>(sink, iters, 1.0000001, 1e-9);
    CUDA_TRY(cudaEventRecord(e1, st));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    CUDA_TRY(cudaGetLastError());
    *tflops = 2.0 * 16.0 * 8.0 * (double)iters * 256.0 * blocks / (ms * 1e-3) / 1e12;
    return LBM_OK;
}

int lbm_run_host(lbm_t *h, const double *rho_in, const double *ux_in, const double *uz_in, const double *T_in, int n,
                 double *rho_out, double *ux_out, double *uz_out, double *T_out, void *stream)
{
    NEED(h);
    if (!rho_in || !ux_in || !uz_in || !T_in) return fail(LBM_ERR_INVALID, "lbm_run_host: null input field");
    if (h->slab) return fail(LBM_ERR_INVALID, "lbm_run_host: not available for z-slabs");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = sizeof(double) * (size_t)h->Lx * h->Lz;
    for (auto &s : h->stage)
        if (!s) CUDA_TRY(cudaMalloc(&s, bytes));
    const double *in[4] = {rho_in, ux_in, uz_in, T_in};
    for (int j = 0; j < 4; ++j) CUDA_TRY(cudaMemcpyAsync(h->stage[j], in[j], bytes, cudaMemcpyHostToDevice, st));
    int rc = lbm_init_equilibrium(h, h->stage[0], h->stage[1], h->stage[2], h->stage[3], stream);
    if (rc) return rc;
    rc = lbm_step(h, n, stream);
    if (rc) return rc;
    double *out[4] = {rho_out, ux_out, uz_out, T_out};
    if (out[0] || out[1] || out[2] || out[3]) {
        rc = lbm_moments(h, out[0] ? h->stage[0] : nullptr, out[1] ? h->stage[1] : nullptr, out[2] ? h->stage[2] : nullptr,
                         out[3] ? h->stage[3] : nullptr, stream);
        if (rc) return rc;
    }
    for (int j = 0; j < 4; ++j)
        if (out[j]) CUDA_TRY(cudaMemcpyAsync(out[j], h->stage[j], bytes, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_steps_done(const lbm_t *h, long long *steps)
{
    NEED_HOST(h);
    if (steps) *steps = h->steps;
    return LBM_OK;
}

int lbm_layout(const lbm_t *h, int *pitch, long long *plane_stride)
{
    NEED_HOST(h);
    if (pitch) *pitch = h->pitch;
    if (plane_stride) *plane_stride = h->plane;
    return LBM_OK;
}

int lbm_kernel_launches(const lbm_t *h, long long *launches)
{
    NEED_HOST(h);
    if (launches) *launches = h->launches;
    return LBM_OK;
}

int lbm_set_zchunk(lbm_t *h, int rows)
{
    NEED_HOST(h);
    // chunks above the first must start at row >= 3: only the chunk at z0 = 0 builds the bottom wall's ghost rows
    if (rows < 0 || rows == 1 || rows == 2)
        return fail(LBM_ERR_INVALID, "lbm_set_zchunk: rows must be 0 (automatic) or >= 3 (got %d)", rows);
    h->zchunk = rows;
    h->plan.valid = false; h->plan_interior.valid = false;
    return LBM_OK;
}

int lbm_set_variant(lbm_t *h, int variant)
{
    NEED_HOST(h);
    if (variant < 0 || variant > 3) return fail(LBM_ERR_INVALID, "lbm_set_variant: unknown variant %d", variant);
    h->variant = variant;
    h->plan.valid = false; h->plan_interior.valid = false;
    return LBM_OK;
}

}  // extern "C"

// ---- lbm_diagnostics_noalloc: the diagnostics pass for callers that may not allocate -------------------------------
// Who needs this: code that runs where cudaMalloc is off limits.  Typical cases are a host program whose device memory
// is handed out once by a framework's pool (anything cudaMalloc takes behind the pool's back can push the pool over the
// edge later, and cudaMalloc also synchronises the whole device, which stalls every other stream of a running job), and
// a monitoring hook that is called in the middle of somebody else's time loop and must not disturb its memory or its
// timing.  Such a caller cannot use lbm_create at all (it allocates the handle's scratch), so this entry point takes the
// raw population buffer instead of a handle.
//
// The per-row array that row_diagnostics_kernel writes and final_diagnostics_kernel reads lives in the library image:
// 8 x LBM_NOALLOC_MAX_ROWS doubles = 1 MiB, resident on every GPU that loads liblbm_b200.so until the process exits.
// `g_noalloc_rows` is a device symbol.  On the host its name is only a stand-in (taking its address in host code gives a
// host address a kernel must never see), so the device address is asked for once per device with cudaGetSymbolAddress
// (noalloc_rows_of_current_device) and that pointer is what the kernels get.
static __device__ __align__(256) double g_noalloc_rows[8 * LBM_NOALLOC_MAX_ROWS];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::mutex g_noalloc_mu;
double *g_noalloc_ptr[NOALLOC_MAX_DEVICES];    // device address of g_noalloc_rows on device d; null = not set up yet

// Set-up, once per device, with that device current: architecture check and the device address of the static array.
int noalloc_rows_of_current_device(double **rows)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return fail(LBM_ERR_NODEVICE, "lbm_diagnostics_noalloc: no CUDA device"); }
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES)
        return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: device ordinal %d is beyond the %d this entry point keeps track of", dev, NOALLOC_MAX_DEVICES);
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
            cudaGetLastError();
            return fail(LBM_ERR_NODEVICE, "lbm_diagnostics_noalloc: cannot query device %d", dev);
        }
        if (major != 10) return fail(LBM_ERR_NODEVICE, "lbm_diagnostics_noalloc: built for sm_100a, device %d is sm_%dx", dev, major);
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_rows);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(LBM_ERR_CUDA, "lbm_diagnostics_noalloc: cudaGetSymbolAddress(g_noalloc_rows) on device %d: %s", dev,
                        e != cudaSuccess ? cudaGetErrorString(e) : "null address");
        }
        g_noalloc_ptr[dev] = (double *)p;
    }
    *rows = g_noalloc_ptr[dev];
    return LBM_OK;
}

}  // namespace

extern "C" int lbm_diagnostics_noalloc(const void *pop_buf, size_t buf_bytes, int Lx, int Lz, double g, double T_d, double T_m,
                                       double T_u, double *result6_dev, double *Tbar_dev, void *stream)
{
    // argument checks first: they need no device, and an oversized lattice must never reach the fixed-size array
    if (!pop_buf || !result6_dev) return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: pop_buf and result6_dev are required");
    if (Lx < 7 || Lz < 6) return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: need Lx >= 7 and Lz >= 6 (got %d x %d)", Lx, Lz);
    if (Lz > LBM_NOALLOC_MAX_ROWS)
        return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: Lz = %d rows exceed LBM_NOALLOC_MAX_ROWS = %d, the size of the "
                    "static scratch array; use lbm_create + lbm_diagnostics for taller lattices", Lz, LBM_NOALLOC_MAX_ROWS);
    if ((uintptr_t)pop_buf & 255) return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: pop_buf must be 256-byte aligned");
    const size_t need = (size_t)plane_of(Lx, Lz) * LBM_NPOP * sizeof(double);
    if (buf_bytes < need) return fail(LBM_ERR_INVALID, "lbm_diagnostics_noalloc: the buffer has %zu bytes, a %d x %d lattice needs %zu", buf_bytes, Lx, Lz, need);
    double *rows = nullptr;
    int rc = noalloc_rows_of_current_device(&rows);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const lbm::Layout lay{Lx, Lz, pitch_of(Lx), plane_of(Lx, Lz), 0, Lz, false};
    // The array still holds what the previous call left there.  Every entry the second kernel reads is rewritten by the
    // first one, so a correct run never depends on old contents; the part this call uses is zeroed all the same, so that
    // a row kernel that did not run cannot pass the last lattice's numbers off as this one's.
    CUDA_TRY(cudaMemsetAsync(rows, 0, sizeof(double) * 8 * (size_t)Lz, st));
    lbm::row_diagnostics_kernel<false><<<Lz, lbm::RED_T, 0, st>>>((const double *)pop_buf + lbm::XH, lay, g, rows, 0);
    CUDA_TRY(cudaGetLastError());
    lbm::final_diagnostics_kernel<<<1, lbm::RED_T, 0, st>>>(rows, Lz, T_d, T_m, T_u, result6_dev);
    CUDA_TRY(cudaGetLastError());
    if (Tbar_dev) CUDA_TRY(cudaMemcpyAsync(Tbar_dev, rows, sizeof(double) * (size_t)Lz, cudaMemcpyDeviceToDevice, st));
    return LBM_OK;
}
