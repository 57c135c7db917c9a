/*
 * lbm.h -- C ABI of the B200-native thermal D2Q37 Lattice-Boltzmann step (liblbm_b200.so).
 *
 * Implements the per-time-step update of arxiv/paper_1405_1253 (citations are PAPER.md lines):
 * propagate (lhs of eq. 5), rigid top/bottom walls with periodic x and the
 * BGK collision toward the force-shifted equilibrium of eq. 6 with the moments of eq. 7
 * (PAPER.md:88), on an Lx x Lz lattice in FP64, plus the diagnostics of PAPER.md:94, 128 and eq. 12.
 * Every arithmetic step runs in CUDA kernels for sm_100a; there is no CPU fallback.
 * Beyond the time step: isothermal walls (wall_kind 1), one-copy in-place streaming (pop_buf1 = NULL) and z-slabs
 * with exchanged ghost rows (lbm_create_slab) -- SURVEY.md 8(f) rows 2-4.
 *
 * Conventions.  Sites (i,k): i = 0..Lx-1 along x (periodic), k = 0..Lz-1 along z (up, walls half a site
 * outside rows 0 and Lz-1).  Canonical dense arrays are x-fastest: fields [Lz][Lx], populations
 * [37][Lz][Lx].  Population order: ascending e_z, then ascending e_x over all integer e with |e|^2 <= 10
 * (l = 0 is (-1,-3), l = 18 is (0,0), l = 36 is (1,3)); the opposite of l is 36 - l.  dt = 1, c_l = r e_l,
 * gravity (0,-g), g >= 0.  "device" pointers are CUDA device memory of the current device, "host" pointers
 * ordinary host memory.  A handle belongs to the device that was current in lbm_create; every call that touches
 * the device returns LBM_ERR_INVALID if another device is current.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *
 * Errors.  Every call returns 0 on success or a negative lbm_status; no exception crosses the boundary;
 * lbm_last_error() returns a thread-local message for the last failing call.
 * Ownership.  The caller owns every buffer it passes, including the two population buffers given to
 * lbm_create (allocated e.g. by torch); the handle owns only metadata and small device scratch.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LBM_NPOP 37

typedef enum {
    LBM_OK = 0,
    LBM_ERR_INVALID = -1, /* bad argument (size, tau, null or misaligned pointer, undersized buffer) */
    LBM_ERR_CUDA = -2,    /* a CUDA runtime call or kernel launch failed; message has the CUDA error */
    LBM_ERR_NODEVICE = -3 /* no CUDA device / wrong architecture */
} lbm_status;

typedef struct lbm_handle lbm_t;

/* Model parameters and storage.  tau = tau_LB/dt of eq. 5 (> 1/2); g = |gravity| of eq. 3/6 (>= 0).
 * wall_kind ("rigid boundary conditions" on rows 0..2 and Lz-3..Lz-1; the paper gives no formula):
 *   0 = half-way bounce-back through velocity-reversed mirror rows (reading 9): adiabatic, no-slip;
 *   1 = isothermal no-slip walls (reading 19): after propagate (wall-crossing gathers filled as for 0) the
 *       equilibrium part of the populations of the three rows next to each wall is moved to the wall state
 *       u^(H) = 0, T^(H) = T_wall_bottom / T_wall_top, density and non-equilibrium part kept; then collide.
 * pop_buf0/pop_buf1: device buffers of at least lbm_buffer_bytes(Lx,Lz) bytes each, 256-byte aligned;
 * they hold the two lattice copies (prv/nxt of PAPER.md:110) in the library's padded SoA layout.
 * pop_buf1 = NULL selects IN-PLACE streaming with ONE lattice copy (two copies "require more
 * memory"): two alternating one-step kernels that write every result back into the slots they read; results are
 * bit-identical to the two-copy path; the two-step kernel (variant 3) is not available. */
typedef struct {
    double tau;
    double g;
    int wall_kind;
    void *pop_buf0; /* device */
    void *pop_buf1; /* device, or NULL: one copy, in-place streaming */
    size_t buf_bytes;
    double T_wall_bottom; /* wall_kind 1 only */
    double T_wall_top;    /* wall_kind 1 only */
} lbm_params;

/* Rayleigh-Taylor initial state, eq. 1-2 with tanh-smoothed jumps.
 * Layer temperatures T_d (bottom) > T_m > T_u (top); rho_m = density at z = 0; rho_d, rho_u follow from
 * eq. 2.  delta = width of the middle layer in sites (0 = single front).  smooth_w = tanh
 * half-width in sites (0 = sharp).  pert_kind: 0 none, 1 sum of n_modes cosines (amplitude uniform in
 * [amp_lo, amp_hi], drawn only if they differ; phase uniform), 2 white noise of +-amp_hi sites per column
 * (PAPER.md:222).  Random numbers: SplitMix64(seed), lower interface first (reading 12). */
typedef struct {
    double T_d, T_m, T_u;
    double rho_m;
    double delta;
    double smooth_w;
    int pert_kind;
    int n_modes;
    double amp_lo, amp_hi;
} lbm_rt_init;

/* Bytes each population buffer must have for an Lx x Lz lattice (padded rows, 37 planes); 0 if invalid. */
size_t lbm_buffer_bytes(int Lx, int Lz);

/* Creates a handle. Errors: Lx < 7, Lz < 6, Lz > 65535 (stored rows, a slab's ghost rows included: the kernels put
 * rows on grid.y), tau <= 0.5, g < 0, wall_kind not 0/1, wall temperatures <= 0 with wall_kind 1, null pop_buf0 /
 * misaligned / undersized buffers, no sm_100 device.  *out is set to NULL on failure. */
int lbm_create(lbm_t **out, int Lx, int Lz, const lbm_params *p);

/* ---- z-slabs: the lattice split along z over several handles (one per GPU), SURVEY 8(f)4.  The paper splits
 * along x over N_p GPUs and hides the halo exchange behind the bulk propagate on separate streams (PAPER.md:110,
 * 116-118, Fig. 3-4); with x-fastest storage the contiguous cut is along z.
 * A slab owns rows [z0, z0+nz) of an Lx x Lz_global lattice and stores 6 ghost rows per open side (one step reads 3,
 * max |e_z| = 3; two fused steps read 6).
 * Dense arrays of every other call (fields [nz][Lx], populations [37][nz][Lx], row profiles [nz]) cover the OWN rows;
 * lbm_totals and the widths of lbm_mixing_widths are the slab's partial sums (add them over the slabs).
 * One time step of a slab, every step:
 *   lbm_slab_pack(side)      my outermost own rows -> message (26 population-rows), per open side
 *   lbm_slab_step(INTERIOR)  rows that read no ghost row; overlaps the exchange (another stream)
 *   ... the caller moves the messages (cudaMemcpyAsync between devices, ncclSend/ncclRecv, ...) ...
 *   lbm_slab_unpack(side)    neighbour's message -> my ghost rows of the CURRENT copy
 *   lbm_slab_step(EDGES)     the remaining own rows; then the other copy becomes current.
 * Two steps at once with the two-step kernel (lbm_step2s.cuh):
 *   lbm_slab_pack2(side)     my 6 outermost own rows, all populations, wrap columns included -> message
 *   lbm_slab_step2_part(INTERIOR)  own rows at least 6 rows from an open side (no ghost row read); overlaps the
 *                            exchange (Fig. 4); launch it after pack2 in stream order
 *   ... transport ...
 *   lbm_slab_unpack2(side)   neighbour's message -> my 6 ghost rows of the CURRENT copy
 *   lbm_slab_step2_part(EDGES)     the 6 own rows next to each open side; then the other copy becomes current.
 * lbm_slab_step2 = both parts in one launch (after unpack2, no overlap).  A slab too thin for interior rows
 * (fewer than 6 of them) runs all its rows in EDGES.
 * Results are bit-identical to the whole-lattice run.  Slabs need two lattice copies;
 * lbm_step / lbm_run_host return LBM_ERR_INVALID for them.  lbm_init_rt fills ghost rows too (closed form);
 * after lbm_init_equilibrium / lbm_set_populations the first exchange does. */
#define LBM_SLAB_INTERIOR 0
#define LBM_SLAB_EDGES 1
size_t lbm_slab_buffer_bytes(int Lx, int Lz_global, int z0, int nz);   /* 0 if invalid (nz >= 6 rows inside the lattice) */
int lbm_create_slab(lbm_t **out, int Lx, int Lz_global, int z0, int nz, const lbm_params *p);
/* HOST outputs, any may be NULL: own row range, whether the sides are open (1) or walls (0), doubles per message of
 * lbm_slab_pack (26 Lx) and of lbm_slab_pack2 (6 x 37 x (Lx + 16)). */
int lbm_slab_info(const lbm_t *h, int *z0, int *nz, int *open_below, int *open_above, size_t *message_doubles,
                  size_t *message2_doubles);
/* side 0 = towards lower z, 1 = towards higher z; msg_dev: DEVICE buffer of message_doubles doubles; asynchronous.
 * LBM_ERR_INVALID if that side is a wall. */
int lbm_slab_pack(lbm_t *h, int side, double *msg_dev, void *stream);
int lbm_slab_unpack(lbm_t *h, int side, const double *msg_dev, void *stream);
int lbm_slab_step(lbm_t *h, int part, void *stream);
int lbm_slab_pack2(lbm_t *h, int side, double *msg_dev, void *stream);
int lbm_slab_unpack2(lbm_t *h, int side, const double *msg_dev, void *stream);
int lbm_slab_step2(lbm_t *h, void *stream);
int lbm_slab_step2_part(lbm_t *h, int part, void *stream);

/* Frees the handle and its scratch; never the population buffers. NULL is a no-op. */
int lbm_destroy(lbm_t *h);

/* Fills the current lattice with the hydrostatic state of eq. 1-2 at u^(H) = 0, T^(H) = T0 (the stored
 * populations are f_eq(rho0, (0,-g/2), T0 - g^2/8), reading 8) and resets the step counter.
 * Synchronous with respect to the host arrays it builds; kernels run on `stream`. */
int lbm_init_rt(lbm_t *h, uint64_t seed, const lbm_rt_init *ic, void *stream);

/* Populations = f_eq(rho, u, T) of the given KINETIC fields (eq. 7; no shift). Device pointers, [Lz][Lx]. */
int lbm_init_equilibrium(lbm_t *h, const double *rho, const double *ux, const double *uz, const double *T,
                         void *stream);

/* Canonical dense [37][Lz][Lx] populations <-> the library's layout. `f` is a DEVICE pointer
 * (lbm_*_populations) or a HOST pointer (lbm_*_populations_host; these synchronise the stream, stage through the
 * other lattice copy and are refused, LBM_ERR_INVALID, on a slab between lbm_slab_step(INTERIOR) and (EDGES)). */
int lbm_set_populations(lbm_t *h, const double *f_dev, void *stream);
int lbm_get_populations(lbm_t *h, double *f_dev, void *stream);
int lbm_set_populations_host(lbm_t *h, const double *f_host, void *stream);
/* A window of the stored populations, dense [37][nk][ni] into the DEVICE array f_dev: rows k0 .. k0+nk-1, columns
 * i0 .. i0+ni-1 taken modulo Lx (a window may straddle the periodic seam).  For lattices whose whole dense array
 * does not fit beside the lattice (16384 x 16384 in place).  Asynchronous.  Errors: rows outside [0, Lz), ni > Lx. */
int lbm_get_window(lbm_t *h, int k0, int nk, int i0, int ni, double *f_dev, void *stream);
int lbm_get_populations_host(lbm_t *h, double *f_host, void *stream);

/* Enqueues n x (propagate + bc + collide) on `stream`; asynchronous.  Afterwards the
 * current lattice is the post-collision state of step n.
 * Stream capture: the call only enqueues kernels, so it may be captured into a CUDA graph, but the handle's
 * bookkeeping (which lattice copy is current, lbm_steps_done) advances when the call is made, not when the graph
 * is replayed.  A captured sequence must therefore return to the same copy: LBM_ERR_INVALID if the n steps are
 * an odd number of launches here (lbm_get_plan tells whether launches advance one or two steps); no other lbm_*
 * call on the handle may be interleaved with replays; lbm_steps_done does not count replays. */
int lbm_step(lbm_t *h, int n, void *stream);

/* Hydrodynamic fields of the stored state (reading 8): rho, u^(H) = u - g_vec/2,
 * T^(H) = T + g^2/8, each a device pointer [Lz][Lx] or NULL to skip (LBM_ERR_INVALID if all four are NULL).
 * Asynchronous. */
int lbm_moments(lbm_t *h, double *rho, double *ux, double *uz, double *T, void *stream);

/* The KINETIC moments rho, u, T of eq. 7 of the stored state, without the half-force shift of
 * PAPER.md:94 that lbm_moments applies: exactly the fields lbm_init_equilibrium and lbm_run_host take, so a state
 * can be handed from one to the other without arithmetic on the caller's side.  DEVICE arrays [Lz][Lx], any may be
 * NULL (not all).  Asynchronous. */
int lbm_kinetic_moments(lbm_t *h, double *rho, double *ux, double *uz, double *T, void *stream);

/* Mixing widths of eq. 12 from the x-averaged T^(H), in sites, with the
 * tent map of eq. 9 (zero outside [0,1]).  L_u, L_d: HOST doubles; Tbar: HOST array [Lz] or NULL.
 * Synchronises `stream`. */
int lbm_mixing_widths(lbm_t *h, double T_d, double T_m, double T_u, double *L_u, double *L_d, double *Tbar,
                      void *stream);

/* Row profiles of section IV from the hydrodynamic fields of the stored state: Tbar(k) = <T^(H)>_x
 * (PAPER.md:128), Trms(k) = sqrt(<(T - <T>_x)^2>_x) (Fig. 8), and the same two for the kinetic
 * energy density E_k = rho |u^(H)|^2 / 2 (Fig. 9; reading 17).  HOST arrays [Lz], any
 * may be NULL.  Synchronises `stream`. */
int lbm_profiles(lbm_t *h, double *Tbar, double *Trms, double *Ekbar, double *Ekrms, void *stream);

/* Growth rate from a logged mixing length (host-only post-processing, no device work): eq. 11 / 14
 * (PAPER.md:169, 199-202), alpha_j = (dL/dt)_j^2 / (4 g At L_j), dL/dt by centred differences on the sample
 * times t[0..n) (one-sided at both ends), alpha_j = 0 where L_j <= 0.  For the double front pass
 * L_tot = L_u + L_d and the total Atwood number.  HOST arrays.  Errors: null series, g <= 0, At <= 0,
 * non-increasing times. */
int lbm_growth_rate(int n, const double *t, const double *L, double g, double At, double *alpha);

/* Lattice totals sum f, sum c_x f, sum c_z f, sum |c|^2 f into HOST out[4] (deterministic two-stage
 * reduction). Synchronises `stream`. */
int lbm_totals(lbm_t *h, double *out4, void *stream);

/* All of the above diagnostics in ONE pass over the lattice (lbm_mixing_widths, lbm_profiles and lbm_totals are
 * calls of it): widths2 = {L_u, L_d} (eq. 12, needs distinct layer temperatures), totals4, and the row profiles
 * Tbar, Trms, Ekbar, Ekrms [Lz].  HOST outputs, any may be NULL; the squared-deviation pass runs only if Trms or
 * Ekrms is asked for.  Synchronises `stream`. */
int lbm_diagnostics(lbm_t *h, double T_d, double T_m, double T_u, double *widths2, double *totals4, double *Tbar,
                    double *Trms, double *Ekbar, double *Ekrms, void *stream);

/* The widths, totals and Tbar of lbm_diagnostics for callers that are not allowed to allocate device memory.
 * Who that is: a program whose GPU memory is handed out once by a pool it does not control (a framework's caching
 * allocator, a job that was given a fixed carve-out), where a cudaMalloc behind the pool's back can make the pool run
 * out later; and a probe that is called from inside another code's time loop, where cudaMalloc would stall every
 * stream of the device.  lbm_create allocates the handle's scratch, so such a caller has no handle: this call takes
 * the population buffer itself and keeps its scratch (the per-row partial results, eq. 12 / PAPER.md:128, 183-186) in
 * a static device array inside the library, 8 x LBM_NOALLOC_MAX_ROWS doubles = 1 MiB, which every GPU that loads the
 * library holds until the process exits.  It calls no cudaMalloc / cudaFree and no allocating library routine.
 *   pop_buf     DEVICE: a lattice copy exactly as handed to lbm_create (pop_buf0 / pop_buf1), buf_bytes long, 256-byte
 *               aligned, holding the current state of an Lx x Lz lattice in the ordinary layout (a two-copy handle's
 *               current copy, or an in-place handle after an even number of steps).  Read only.
 *   g           gravity of eq. 3 (the hydrodynamic T^(H), u^(H) of PAPER.md:94 need it).
 *   result6_dev DEVICE out[6]: L_u, L_d (eq. 12; both 0 if T_d == T_m or T_m == T_u), sum f, sum c_x f, sum c_z f,
 *               sum |c|^2 f.  Tbar_dev: DEVICE out[Lz] or NULL, Tbar(k) of PAPER.md:128.
 * Asynchronous on `stream`; nothing is synchronised, the outputs are valid once the stream reaches that point.
 * Limit: Lz <= LBM_NOALLOC_MAX_ROWS, else LBM_ERR_INVALID with a message naming the limit (Lx is not limited).
 * Other errors: null / misaligned / undersized buffer, Lx < 7, Lz < 6 (LBM_ERR_INVALID, checked before any device
 * work); no sm_100 device current (LBM_ERR_NODEVICE); a failed launch or cudaGetSymbolAddress (LBM_ERR_CUDA).
 * First call on a device: looks up the device address of the static array (cudaGetSymbolAddress, with that device
 * current) and remembers it per device; make that first call before any stream capture begins.
 * Sharing: all calls on one GPU use the same array, and it keeps the previous call's contents.  The part a call uses
 * is cleared and rewritten by that call on its stream, so calls that follow each other on one stream are independent
 * of each other; two calls whose work may overlap on the GPU (different streams, different host threads) race on the
 * array and give undefined results -- order them with an event or use one stream. */
#define LBM_NOALLOC_MAX_ROWS 16384
int lbm_diagnostics_noalloc(const void *pop_buf, size_t buf_bytes, int Lx, int Lz, double g, double T_d, double T_m,
                            double T_u, double *result6_dev, double *Tbar_dev, void *stream);

/* Scales of a Rayleigh-Taylor run (host arithmetic): Atwood number At = (T_d - T_u)/(T_d + T_u) (Table II,
 * PAPER.md:144) and tau_RT = sqrt(Lx / (g At)), Lx in sites.  HOST outputs, any may be NULL. */
int lbm_rt_scales(double Lx, double g, double T_d, double T_u, double *At, double *tau_rt);

/* Host-buffer convenience used by the end-to-end benchmark: uploads kinetic fields (HOST, [Lz][Lx]),
 * initialises at equilibrium, runs n steps, downloads rho, u^(H), T^(H) (HOST, [Lz][Lx], any may be NULL).
 * Uses the handle's staging buffers (allocated on first use, 4 x Lx x Lz doubles). Synchronous. */
int lbm_run_host(lbm_t *h, const double *rho_in, const double *ux_in, const double *uz_in, const double *T_in,
                 int n, double *rho_out, double *ux_out, double *uz_out, double *T_out, void *stream);

/* Introspection. */
int lbm_steps_done(const lbm_t *h, long long *steps);
int lbm_layout(const lbm_t *h, int *pitch, long long *plane_stride); /* in doubles */
int lbm_kernel_launches(const lbm_t *h, long long *launches);       /* kernels launched through this handle */
/* Measurement aid ("no FP64 entry in MEASURED_PEAKS.json -- measure with a DFMA-chain microbenchmark"):
 * runs 8 independent DFMA chains per thread on every SM for `iters` rounds (0 = default), times them with CUDA
 * events on `stream` and returns the vector-FP64 rate in TFLOP/s (FMA = 2 flops) in HOST *tflops.  Not part of the
 * time step.  Synchronises `stream`. */
int lbm_fp64_peak(double *tflops, int iters, void *stream);
/* Step-kernel variant: 0 automatic (default): the two-step kernel (lbm_step2s.cuh) where its launch plan is
 * predicted faster than two single steps (from about 512x512 up), one cooperative launch for all n steps on
 * lattices of at most ~37 000 sites (persistent kernel with a grid barrier between steps), else one step per
 * launch; 1 one step per launch (256-thread blocks), 2 one step (128), 3 two steps per launch forced
 * (LBM_ERR_INVALID from lbm_step for in-place handles: it needs two copies).  All give bit-identical results. */
int lbm_set_variant(lbm_t *h, int variant);
int lbm_set_zchunk(lbm_t *h, int rows);  /* rows per block of the two-step kernel (>= 3), or 0 = automatic */
/* The launch plan lbm_step uses for this lattice with the current variant / zchunk settings (HOST outputs, any may
 * be NULL): *fused = 1 if a launch advances two time steps (two-step kernel), 0 if one; *strip_width = columns per
 * block of the two-step kernel (strip s covers columns [s w, (s+1) w)); *zchunk = rows per block (chunk c covers
 * rows [c ZC, (c+1) ZC)).  Automatic choice: DESIGN.md section 6 (whole waves of blocks, few chunks).  With
 * wall_kind 1 and an automatic plan of several chunks the chunks on an isothermal wall are 14 rows shorter (their wall
 * adjustments cost about that much): chunk c > 0 then starts at row c ZC - 14, the last chunk ends at Lz. */
int lbm_get_plan(lbm_t *h, int *fused, int *strip_width, int *zchunk);
/* D2Q37 tables as the library uses them (host outputs, any may be NULL): e_x[37], e_z[37], w[37], r. */
int lbm_tables(int *ex, int *ez, double *w, double *r);
const char *lbm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
