// lbm_api.cu -- the C ABI declared in include/lbm.h: handle, argument checks, kernel launches.
// Every arithmetic step of the path runs in the kernels of lbm_step.cuh / lbm_aux.cuh; this file only
// validates, draws the interface perturbation (host, O(Lx)), launches and copies.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
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

int pitch_of(int Lx) { return (Lx + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN; }
long long plane_of(int Lx, int Lz) { return (long long)pitch_of(Lx) * Lz + PLANE_PAD; }

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

// Tensor maps for the TMA loads of the warp-specialised two-step kernel (lbm_step2s.cuh): the lattice copy `buf`
// as a rank-3 tensor (x: Lx, z: Lz, l: 37) with strides (pitch, plane), box (SP, R, n) for n = 3, 5, 7.
// cuTensorMapEncodeTiled is fetched through the runtime (no link-time dependency on libcuda).
bool encode_step2s_maps(const double *buf, int Lx, int Lz, int pitch, long long plane, lbm::Step2sMaps &out)
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
        const cuuint64_t dims[3] = {(cuuint64_t)Lx, (cuuint64_t)Lz, (cuuint64_t)LBM_NPOP};
        const cuuint64_t strides[2] = {(cuuint64_t)pitch * 8, (cuuint64_t)plane * 8};
        const cuuint32_t box[3] = {(cuuint32_t)S::SP, (cuuint32_t)S::R, (cuuint32_t)(3 + 2 * i)};
        const cuuint32_t estr[3] = {1, 1, 1};
        if (encode((CUtensorMap *)out.m[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)buf, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    return true;
}

}  // namespace

struct lbm_handle {
    int Lx, Lz, pitch;
    long long plane;
    double tau, g;
    double *buf[2];
    int cur;               // index of the current lattice
    long long steps, launches;
    int variant;
    int zchunk;            // rows per block of the two-step kernel (multiple of 3; 0 = automatic)
    int sm_count;
    bool tma_ok;              // tensor maps of both lattice copies encoded (two-step kernel)
    lbm::Step2sMaps maps[2];
    double *scratch;       // device: Tbar[Lz] | row partials[4 Lz] | results[8] | h_lo[Lx] | h_hi[Lx]
    double *stage[4];      // device staging fields for lbm_run_host (lazy)
    lbm::Layout layout() const { return lbm::Layout{Lx, Lz, pitch, plane}; }
    double *d_tbar() const { return scratch; }
    double *d_partial() const { return scratch + Lz; }
    double *d_result() const { return scratch + 5LL * Lz; }
    double *d_hlo() const { return scratch + 5LL * Lz + 8; }
    double *d_hhi() const { return scratch + 5LL * Lz + 8 + Lx; }
};

extern "C" {

const char *lbm_last_error(void) { return g_err; }

size_t lbm_buffer_bytes(int Lx, int Lz)
{
    if (Lx < 7 || Lz < 6) return 0;
    return (size_t)plane_of(Lx, Lz) * LBM_NPOP * sizeof(double);
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
    if (!out) return fail(LBM_ERR_INVALID, "lbm_create: out is null");
    *out = nullptr;
    if (!p) return fail(LBM_ERR_INVALID, "lbm_create: params is null");
    // Lx >= 7 keeps the seven wrapped source columns of a site distinct (one wrap suffices); Lz >= 6
    // keeps the three wall rows of the two walls disjoint
    if (Lx < 7 || Lz < 6) return fail(LBM_ERR_INVALID, "lbm_create: need Lx >= 7 and Lz >= 6 (got %d x %d)", Lx, Lz);
    if (Lz > 65535) return fail(LBM_ERR_INVALID, "lbm_create: Lz <= 65535 (got %d)", Lz);
    if (!(p->tau > 0.5)) return fail(LBM_ERR_INVALID, "lbm_create: tau must be > 0.5 (got %g)", p->tau);
    if (!(p->g >= 0.0)) return fail(LBM_ERR_INVALID, "lbm_create: g must be >= 0 (got %g)", p->g);
    if (p->wall_kind != 0) return fail(LBM_ERR_INVALID, "lbm_create: wall_kind %d not supported", p->wall_kind);
    if (!p->pop_buf0 || !p->pop_buf1 || p->pop_buf0 == p->pop_buf1)
        return fail(LBM_ERR_INVALID, "lbm_create: two distinct population buffers are required");
    if (((uintptr_t)p->pop_buf0 | (uintptr_t)p->pop_buf1) & 255)
        return fail(LBM_ERR_INVALID, "lbm_create: population buffers must be 256-byte aligned");
    if (p->buf_bytes < lbm_buffer_bytes(Lx, Lz))
        return fail(LBM_ERR_INVALID, "lbm_create: buffers have %zu bytes, need %zu", p->buf_bytes, lbm_buffer_bytes(Lx, Lz));
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(LBM_ERR_NODEVICE, "lbm_create: no CUDA device");
    }
    if (prop.major != 10) return fail(LBM_ERR_NODEVICE, "lbm_create: built for sm_100a, device is sm_%d%d", prop.major, prop.minor);
    lbm_handle *h = new (std::nothrow) lbm_handle();
    if (!h) return fail(LBM_ERR_INVALID, "lbm_create: out of host memory");
    h->Lx = Lx; h->Lz = Lz; h->pitch = pitch_of(Lx); h->plane = plane_of(Lx, Lz);
    h->tau = p->tau; h->g = p->g; h->sm_count = prop.multiProcessorCount;
    h->buf[0] = (double *)p->pop_buf0; h->buf[1] = (double *)p->pop_buf1;
    h->cur = 0; h->steps = 0; h->launches = 0; h->variant = 0; h->zchunk = 0; h->scratch = nullptr;
    h->tma_ok = encode_step2s_maps(h->buf[0], Lx, Lz, h->pitch, h->plane, h->maps[0]) &&
                encode_step2s_maps(h->buf[1], Lx, Lz, h->pitch, h->plane, h->maps[1]);
    for (auto &s : h->stage) s = nullptr;
    cudaError_t e = cudaMalloc(&h->scratch, sizeof(double) * (5LL * Lz + 8 + 2LL * Lx));
    if (e != cudaSuccess) { delete h; return fail(LBM_ERR_CUDA, "lbm_create: cudaMalloc scratch: %s", cudaGetErrorString(e)); }
    *out = h;
    return LBM_OK;
}

int lbm_destroy(lbm_t *h)
{
    if (!h) return LBM_OK;
    cudaFree(h->scratch);
    for (auto s : h->stage) cudaFree(s);
    delete h;
    return LBM_OK;
}

#define NEED(h) do { if (!(h)) return fail(LBM_ERR_INVALID, "%s: null handle", __func__); } while (0)
#define LAUNCHED(h) do { CUDA_TRY(cudaGetLastError()); (h)->launches++; } while (0)

static dim3 site_grid(const lbm_t *h, int tx) { return dim3((h->Lx + tx - 1) / tx, h->Lz, 1); }

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
    lbm::RtArgs a{h->g, 1.0 / ic->T_d, 1.0 / ic->T_m, 1.0 / ic->T_u, ic->rho_m, ic->delta, ic->smooth_w};
    lbm::init_rt_kernel<<<site_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, st>>>(h->buf[h->cur], h->layout(), a, h->d_hlo(), h->d_hhi());
    LAUNCHED(h);
    h->steps = 0;
    return LBM_OK;
}

int lbm_init_equilibrium(lbm_t *h, const double *rho, const double *ux, const double *uz, const double *T, void *stream)
{
    NEED(h);
    if (!rho || !ux || !uz || !T) return fail(LBM_ERR_INVALID, "lbm_init_equilibrium: null field");
    lbm::init_equilibrium_kernel<<<site_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), rho, ux, uz, T);
    LAUNCHED(h);
    h->steps = 0;
    return LBM_OK;
}

int lbm_set_populations(lbm_t *h, const double *f_dev, void *stream)
{
    NEED(h);
    if (!f_dev) return fail(LBM_ERR_INVALID, "lbm_set_populations: null pointer");
    dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->Lz, LBM_NPOP);
    lbm::pack_kernel<<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(h->buf[h->cur], h->layout(), f_dev);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_get_populations(lbm_t *h, double *f_dev, void *stream)
{
    NEED(h);
    if (!f_dev) return fail(LBM_ERR_INVALID, "lbm_get_populations: null pointer");
    dim3 grid((h->Lx + lbm::AUX_TX - 1) / lbm::AUX_TX, h->Lz, LBM_NPOP);
    lbm::unpack_kernel<<<grid, lbm::AUX_TX, 0, (cudaStream_t)stream>>>(h->buf[h->cur], h->layout(), f_dev);
    LAUNCHED(h);
    return LBM_OK;
}

// host variants stage through the OTHER lattice copy (free between steps), so no extra device memory
int lbm_set_populations_host(lbm_t *h, const double *f_host, void *stream)
{
    NEED(h);
    if (!f_host) return fail(LBM_ERR_INVALID, "lbm_set_populations_host: null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    double *tmp = h->buf[h->cur ^ 1];
    CUDA_TRY(cudaMemcpyAsync(tmp, f_host, sizeof(double) * LBM_NPOP * h->Lx * h->Lz, cudaMemcpyHostToDevice, st));
    int rc = lbm_set_populations(h, tmp, stream);
    if (rc) return rc;
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_get_populations_host(lbm_t *h, double *f_host, void *stream)
{
    NEED(h);
    if (!f_host) return fail(LBM_ERR_INVALID, "lbm_get_populations_host: null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    double *tmp = h->buf[h->cur ^ 1];
    int rc = lbm_get_populations(h, tmp, stream);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(f_host, tmp, sizeof(double) * LBM_NPOP * h->Lx * h->Lz, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_step(lbm_t *h, int n, void *stream)
{
    NEED(h);
    if (n < 0) return fail(LBM_ERR_INVALID, "lbm_step: n must be >= 0 (got %d)", n);
    cudaStream_t st = (cudaStream_t)stream;
    lbm::StepArgs a;
    a.Lx = h->Lx; a.Lz = h->Lz; a.pitch = h->pitch; a.plane = h->plane;
    a.omega = 1.0 / h->tau;
    a.gtau = h->g * h->tau;
    a.dT = 0.5 * h->tau * (1.0 - h->tau) * h->g * h->g;
    lbm::fill_offsets(a);
    // Variants: 0 = automatic (two steps per launch where the lattice is large enough to fill the GPU with
    // strips, else one step per launch), 1 = one step, 256x1 blocks, 2 = one step, 128x1 blocks,
    // 3 = two steps per launch forced.  An odd last step always runs the one-step kernel.
    using S2 = lbm::Step2sWide;
    int ZC = h->zchunk;
    const int strips = (h->Lx + S2::TX - 1) / S2::TX;
    if (ZC == 0) {  // enough blocks for >= 6 waves over the SMs (the tail of the last wave is what costs on mid-size
                    // lattices: 1024x2048 gains 8 % over 4 waves), chunks of 24..192 rows (warm-up is 6 rows per chunk)
        const int want_chunks = (6 * h->sm_count + strips - 1) / strips;
        ZC = (h->Lz + want_chunks - 1) / want_chunks;
        ZC = (ZC + 5) / 6 * 6;   // whole passes for R = 2 or 3 rows
        if (ZC < 24) ZC = 24;
        if (ZC > 192) ZC = 192;
    }
    const long long blocks2 = (long long)strips * ((h->Lz + ZC - 1) / ZC);
    const bool fused = h->variant == 3 ||
                       (h->variant == 0 && h->tma_ok && blocks2 >= 2LL * h->sm_count && h->Lx >= 2 * S2::TX);
    if (h->variant == 3 && !h->tma_ok)
        return fail(LBM_ERR_CUDA, "lbm_step: the two-step kernel needs tensor maps (cuTensorMapEncodeTiled failed)");
    int s = 0;
    if (fused && n >= 2) {
        static bool attr_set = false;
        if (!attr_set) {
            CUDA_TRY(cudaFuncSetAttribute(lbm::step2s_kernel<S2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S2::SMEM));
            attr_set = true;
        }
        dim3 grid(strips, (h->Lz + ZC - 1) / ZC);
        for (; s + 2 <= n; s += 2) {
            a.src = h->buf[h->cur];
            a.dst = h->buf[h->cur ^ 1];
            lbm::step2s_kernel<S2><<<grid, S2::THREADS, S2::SMEM, st>>>(a, h->maps[h->cur], ZC);
            LAUNCHED(h);
            h->cur ^= 1;  // a5: swap prv / nxt, once per two steps
            h->steps += 2;
        }
    }
    for (; s < n; ++s) {
        a.src = h->buf[h->cur];
        a.dst = h->buf[h->cur ^ 1];
        // 128-thread blocks are a few per cent faster on the small (L2-resident, few-wave) lattices, 256 on the large
        if (h->variant == 2 || (h->variant == 0 && (long long)h->Lx * h->Lz < (1LL << 20)))
            lbm::step_kernel_site<128, 1><<<dim3((h->Lx + 127) / 128, h->Lz), dim3(128, 1), 0, st>>>(a);
        else  // 256 threads = 2 blocks/SM at 128 registers: fastest one-step shape at 4096x8192
            lbm::step_kernel_site<256, 1><<<dim3((h->Lx + 255) / 256, h->Lz), dim3(256, 1), 0, st>>>(a);
        LAUNCHED(h);
        h->cur ^= 1;  // a5: swap prv / nxt
        h->steps++;
    }
    return LBM_OK;
}

int lbm_moments(lbm_t *h, double *rho, double *ux, double *uz, double *T, void *stream)
{
    NEED(h);
    lbm::moments_kernel<<<site_grid(h, lbm::AUX_TX), lbm::AUX_TX, 0, (cudaStream_t)stream>>>(
        h->buf[h->cur], h->layout(), h->g, rho, ux, uz, T);
    LAUNCHED(h);
    return LBM_OK;
}

int lbm_mixing_widths(lbm_t *h, double T_d, double T_m, double T_u, double *L_u, double *L_d, double *Tbar, void *stream)
{
    NEED(h);
    if (!L_u || !L_d) return fail(LBM_ERR_INVALID, "lbm_mixing_widths: null output");
    if (T_m == T_u || T_d == T_m) return fail(LBM_ERR_INVALID, "lbm_mixing_widths: layer temperatures must differ");
    cudaStream_t st = (cudaStream_t)stream;
    lbm::row_tbar_kernel<<<h->Lz, lbm::RED_T, 0, st>>>(h->buf[h->cur], h->layout(), h->g, h->d_tbar());
    LAUNCHED(h);
    lbm::widths_kernel<<<1, lbm::RED_T, 0, st>>>(h->d_tbar(), h->Lz, T_d, T_m, T_u, h->d_result());
    LAUNCHED(h);
    double res[2];
    CUDA_TRY(cudaMemcpyAsync(res, h->d_result(), sizeof res, cudaMemcpyDeviceToHost, st));
    if (Tbar) CUDA_TRY(cudaMemcpyAsync(Tbar, h->d_tbar(), sizeof(double) * h->Lz, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    *L_u = res[0];
    *L_d = res[1];
    return LBM_OK;
}

int lbm_profiles(lbm_t *h, double *Tbar, double *Trms, double *Ekbar, double *Ekrms, void *stream)
{
    NEED(h);
    cudaStream_t st = (cudaStream_t)stream;
    double *d = h->d_partial();  // [4][Lz], shared with the totals partials
    lbm::row_profiles_kernel<<<h->Lz, lbm::RED_T, 0, st>>>(h->buf[h->cur], h->layout(), h->g, d);
    LAUNCHED(h);
    double *out[4] = {Tbar, Trms, Ekbar, Ekrms};
    for (int j = 0; j < 4; ++j)
        if (out[j]) CUDA_TRY(cudaMemcpyAsync(out[j], d + (long long)j * h->Lz, sizeof(double) * h->Lz, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
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

int lbm_totals(lbm_t *h, double *out4, void *stream)
{
    NEED(h);
    if (!out4) return fail(LBM_ERR_INVALID, "lbm_totals: null output");
    cudaStream_t st = (cudaStream_t)stream;
    lbm::row_totals_kernel<<<h->Lz, lbm::RED_T, 0, st>>>(h->buf[h->cur], h->layout(), h->d_partial());
    LAUNCHED(h);
    lbm::final_totals_kernel<<<1, lbm::RED_T, 0, st>>>(h->d_partial(), h->Lz, h->d_result() + 2);
    LAUNCHED(h);
    CUDA_TRY(cudaMemcpyAsync(out4, h->d_result() + 2, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_run_host(lbm_t *h, const double *rho_in, const double *ux_in, const double *uz_in, const double *T_in, int n,
                 double *rho_out, double *ux_out, double *uz_out, double *T_out, void *stream)
{
    NEED(h);
    if (!rho_in || !ux_in || !uz_in || !T_in) return fail(LBM_ERR_INVALID, "lbm_run_host: null input field");
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
    rc = lbm_moments(h, out[0] ? h->stage[0] : nullptr, out[1] ? h->stage[1] : nullptr, out[2] ? h->stage[2] : nullptr,
                     out[3] ? h->stage[3] : nullptr, stream);
    if (rc) return rc;
    for (int j = 0; j < 4; ++j)
        if (out[j]) CUDA_TRY(cudaMemcpyAsync(out[j], h->stage[j], bytes, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return LBM_OK;
}

int lbm_steps_done(const lbm_t *h, long long *steps)
{
    NEED(h);
    if (steps) *steps = h->steps;
    return LBM_OK;
}

int lbm_layout(const lbm_t *h, int *pitch, long long *plane_stride)
{
    NEED(h);
    if (pitch) *pitch = h->pitch;
    if (plane_stride) *plane_stride = h->plane;
    return LBM_OK;
}

int lbm_kernel_launches(const lbm_t *h, long long *launches)
{
    NEED(h);
    if (launches) *launches = h->launches;
    return LBM_OK;
}

int lbm_set_zchunk(lbm_t *h, int rows)
{
    NEED(h);
    // chunks above the first must start at row >= 3: only the chunk at z0 = 0 builds the bottom wall's ghost rows
    if (rows < 0 || rows == 1 || rows == 2)
        return fail(LBM_ERR_INVALID, "lbm_set_zchunk: rows must be 0 (automatic) or >= 3 (got %d)", rows);
    h->zchunk = rows;
    return LBM_OK;
}

int lbm_set_variant(lbm_t *h, int variant)
{
    NEED(h);
    if (variant < 0 || variant > 3) return fail(LBM_ERR_INVALID, "lbm_set_variant: unknown variant %d", variant);
    h->variant = variant;
    return LBM_OK;
}

}  // extern "C"
