/* mm.h -- C ABI of libmm: the GPU-resident bound-motor microscale step (sm_100a).
 *
 * What it computes.  The microscale half of the micro-macro gliding-assay model of Cook & Shinar
 * (arxiv 1908.04279): the bound-motor density M_b of Eq. 4,
 *      d_t M_b + d_s M_b = -k_off M_b + k_on M_f 1_{D_rc},
 * restricted to the capture disc |x + s p - r0| <= r_c, advanced by many explicit
 * substeps that stay resident on the GPU between macro steps (section 3.1 PAPER.md:131-145,
 * Algorithm 2), followed by the per-unit reduction the macroscale consumes
 * (Eq. 10; Alg. 2 l.14 PAPER.md:206-208).  The density is parametrised as
 * BASELINE.json `north_star` states: configuration c = (x, y, theta) x arc length s x stalk offset
 * (xi, eta) = head - tail; one substep = (1) conservative first-order upwind advection in s at the
 * force-dependent walking speed and in (xi, eta) at the head's velocity relative to the anchored
 * tail, (2) Bell-law detachment with enhanced end detachment + uniform attachment inside the disc,
 * and on request (3) the spring-force moments per configuration.  The exact discrete formulas
 * (S1-S9) and every reading of the paper are listed in DESIGN.md.
 *
 * Conventions.
 *  - Plain C, no C++ types, nothing throws across the boundary.  Every call returns an mm_status
 *    (0 = success, negative = error); mm_last_error(ctx) gives a message for the last failure.
 *  - "device pointer" = CUDA device memory of the CURRENT device; "host pointer" = ordinary or
 *    pinned host memory.  Arguments named *_on_device say which one a void* is.
 *  - Canonical density layout: [ix][iy][itheta][j][a][b], b (eta index) fastest; element type is the
 *    context's dtype.  Configuration index c = (ix*ny + iy)*ntheta + itheta, Nc = nx*ny*ntheta.
 *    Flat indices are 64-bit: more than 2^32 elements are supported.
 *  - All work is enqueued on the cudaStream_t given to mm_create.  Calls with device destinations
 *    are stream-ordered and do not synchronise; calls with host sources/destinations synchronise
 *    that stream before returning.
 *  - A handle is not thread-safe; distinct handles are independent.
 *  - There is no CPU fallback: without a CUDA device every compute call fails with MM_ERR_CUDA.
 */
#ifndef MM_H_
#define MM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mm_ctx mm_ctx; /* opaque */

typedef enum { MM_F32 = 0, MM_F64 = 1 } mm_dtype;

typedef enum {
    MM_OK = 0,
    MM_ERR_INVALID_ARG = -1, /* NULL pointer, bad dimension, non-finite or out-of-range parameter */
    MM_ERR_CUDA = -2,        /* a CUDA runtime call or kernel launch failed (message in mm_last_error) */
    MM_ERR_NOMEM = -3,       /* host or device allocation failed */
    MM_ERR_STATE = -4,       /* substep/moments before density and velocities were set */
    MM_ERR_UNSTABLE = -5     /* MM_FLAG_CHECK_DT set and dt violates the positivity bound (S8) */
} mm_status;

/* Grid sizes.  (x, y) periodic labels; theta_k = 2 pi k / ntheta; s, xi, eta cell
 * centred: s_j = s_lo + (j+1/2) ds, xi_a = -R + (a+1/2) 2R/nxi, eta_b likewise. */
typedef struct {
    int32_t nx, ny, ntheta, ns, nxi, neta;
} mm_grid;

#define MM_FLAG_S_PERIODIC 1u              /* test-only: s wraps (default: zero inflow at s_lo, walk-off at s_hi) */
#define MM_FLAG_OFFSET_PERIODIC_NOMASK 2u  /* test-only: (xi, eta) wrap and the disc mask is off */
#define MM_FLAG_CHECK_DT 4u                /* mm_substep returns MM_ERR_UNSTABLE when dt breaks the S8 bound */
#define MM_FLAG_RK2_SUPERBEE 8u            /* second scheme: every substep is the paper's Runge-
                                              Kutta 2 through the half step (Alg. 2 l.9-10)
                                              with the Superbee flux limiter in s instead of forward
                                              Euler + first-order upwind; (xi, eta) stay first-order upwind.  Formulas:
                                              DESIGN.md Q27-Q30.  The S8 bound of MM_FLAG_CHECK_DT is the Euler one. */

/* Model parameters (BASELINE.json configs[0] gives the benchmark values in brackets). */
typedef struct {
    double v0;              /* unloaded walking speed                                   [1]   */
    double f_stall;         /* stall force of the linear force-velocity law, > 0        [6]   */
    double k_spring;        /* stalk spring constant k, >= 0                            [50]  */
    double k_on;            /* attachment rate, >= 0                                    [5]   */
    double k_off0;          /* unloaded detachment rate, >= 0                           [1]   */
    double f_detach;        /* Bell force scale f_d, > 0                                [2]   */
    double end_detach_mult; /* detachment multiplier in the n_end_cells outermost s cells [10] */
    double m_free;          /* unbound source density M_f (constant on this path)       [1]   */
    double R;               /* capture radius r_c; offsets live on [-R, R]^2, > 0       [0.1] */
    double s_lo, s_hi;      /* arc-length interval, s_hi > s_lo                         [-0.5, 0.5] */
    int32_t n_end_cells;    /* >= 0, 2*n_end_cells <= ns                                [1]   */
    uint32_t flags;         /* MM_FLAG_*                                                [0]   */
} mm_params;

/* Tuning / test options for mm_set_option.  Defaults are what bench.py times. */
typedef enum {
    MM_OPT_KERNEL = 0,       /* 0 auto (default: the fastest measured variant for the dtype and grid, DESIGN.md
                                "Kernel selection": kernel 5 where supported, else 1); 1 force the generic
                                global-memory kernels (any grid, all flags); 2 force the warp-streamed 1-D-TMA
                                kernels; 3 force the tiled-TMA kernels; 4 force the coefficient-form kernels
                                (upwind planes of the fused levels in registers / shared memory); 5 force the
                                upwind-sparse kernel (carries in tensor memory, run-time fuse depth)
                                (2..5: MM_ERR_INVALID_ARG from mm_substep if the grid/flags are unsupported) */
    MM_OPT_FUSE_T = 1,       /* max substeps fused per HBM pass (temporal fusion), 1..MM_MAX_FUSE_T; mm_substep uses as
                                few passes as this allows, of balanced depth (10 substeps at depth 6 = 5 + 5);
                                default MM_MAX_FUSE_T */
    MM_OPT_FUSE_MOMENTS = 2, /* 1 (default): the last pass of mm_substep also reduces the moments, so a
                                following mm_moments is a copy; 0: mm_moments always runs its own pass */
    MM_OPT_INPLACE = 3,      /* 1: the coefficient-form, upwind-sparse, fused RK2 and local-step kernels update the
                                current density buffer IN PLACE (plane j of the result depends on input planes <= j
                                only, each already staged on the SM when plane j is stored, and one warp owns a
                                configuration), the other buffer is not touched; same results, same speed, half the
                                memory.  Default 0; always 1 for a context created with ONE density buffer
                                (mm_create, dens_buf1 = NULL) */
    MM_OPT_FREE_COUPLING = 4,/* 1: the source term of the substeps is k_on M_f(r0) from the table of the last
                                mm_update_free_motors (which switches it on); 0: the constant k_on m_free again.
                                MM_ERR_STATE when set to 1 before any mm_update_free_motors */
    MM_OPT_SPREAD_ATOMIC = 6,/* 0 (default): mm_spread_force gathers -- for a fixed (theta, j) the 4 x 4 stencil is the same
                                at every (x, y), so every fluid node sums its shifted sources in a fixed order
                                (reproducible bit for bit); 1: the first version, one fp64 atomic add per point force
                                and stencil node (summation order varies from call to call) */
    MM_OPT_FREE_REFRESH = 5  /* k > 0: with the coupled source, mm_substep redoes the coarse reduction, the cap and M_f
                                (what mm_update_free_motors does) before every k-th substep of a call -- Alg. 2's own
                                cadence, where l.14-20 sit inside the inner loop, is k = 1; at most k
                                substeps are then fused per pass.  0 (default): the table stays frozen between two
                                mm_update_free_motors calls */
} mm_option;
#define MM_MAX_FUSE_T 12  /* kernel 5 (tensor-memory budget of a warp); kernel 4 fuses at most 10 (fp32, 16x16 offset
                             planes) / 6, the streamed / tiled variants at most 4 (deeper settings are clamped) */
#define MM_LOCAL_FUSE_T 4 /* levels per pass of mm_advance_local on kernel 4 (kernel 5 fuses MM_OPT_FUSE_T local steps) */

/* Create a context: the GPU-resident state of the microscale step -- "M_b ... reside[s] only on the GPU" between outer
 * steps, "only the smaller, coarsened data is transferred to/from main memory"; two density buffers
 * as the paper keeps two time levels, or one (in-place passes).
 *  grid, params : copied.  Invalid (MM_ERR_INVALID_ARG): any dim < 1, R <= 0, f_stall <= 0,
 *                 f_detach <= 0, s_hi <= s_lo, negative rates/speeds, 2*n_end_cells > ns, non-finite.
 *  dens_buf0/1  : device pointers to two density buffers of >= cells*sizeof(real) bytes each,
 *                 16-byte aligned, BORROWED (must outlive the context; e.g. torch tensors).  Pass
 *                 NULL, NULL and the library allocates and owns them (MM_ERR_NOMEM on failure).
 *                 dens_buf0 alone (dens_buf1 = NULL) creates a SINGLE-BUFFER context: half the memory, every
 *                 pass in place (MM_OPT_INPLACE), and only the in-place kernels are available -- mm_substep /
 *                 mm_advance_local return MM_ERR_INVALID_ARG for grids or flags that need the generic kernels.
 *                 dens_buf0 = NULL with dens_buf1 != NULL is invalid.
 *  cuda_stream  : a cudaStream_t (NULL = the legacy default stream).
 *  out          : receives the handle.  On error *out is NULL. */
mm_status mm_create(const mm_grid *grid, const mm_params *params, mm_dtype dtype,
                    void *dens_buf0, void *dens_buf1, void *cuda_stream, mm_ctx **out);

/* Upload / download the whole density in canonical layout and the context's dtype.
 * src/dst hold cells elements.  mm_get_density returns the state after the last completed substep. */
mm_status mm_set_density(mm_ctx *ctx, const void *src, int src_on_device);
mm_status mm_get_density(mm_ctx *ctx, void *dst, int dst_on_device);

/* Same for a contiguous range of configurations [c_begin, c_begin + n_configs): lets a caller stream
 * a density that is larger than host memory (checkpoint/restart primitive).  After every
 * configuration has been covered by set calls the density counts as set. */
mm_status mm_set_density_range(mm_ctx *ctx, int64_t c_begin, int64_t n_configs, const void *src, int src_on_device);
mm_status mm_get_density_range(mm_ctx *ctx, int64_t c_begin, int64_t n_configs, void *dst, int dst_on_device);

/* Per-configuration filament velocities (U, V, Omega), Nc elements each, index c, context dtype
 * (the macro-timescale input; "Psi ... is transferred as before"). */
mm_status mm_set_filament_velocity(mm_ctx *ctx, const void *U, const void *V, const void *Omega, int on_device);

/* n_sub explicit substeps of size dt of Eq. 4 (d_t M_b + d_s M_b = -k_off M_b + k_on M_f 1_{D_rc}) for
 * every unit independently, the inner loop of Alg. 2 l.4-13 with the state staying on the GPU; in
 * the discretisation BASELINE.json north_star (1)-(2) fixes (S2-S7: first-order upwind in s and (xi, eta),
 * Bell-law and end detachment, attachment inside the disc, mask).  Asynchronous on the stream.  n_sub >= 0; dt > 0 and
 * finite when n_sub > 0.  MM_ERR_STATE unless density and velocities have been set; MM_ERR_UNSTABLE with
 * MM_FLAG_CHECK_DT when dt breaks the positivity bound S8. */
mm_status mm_substep(mm_ctx *ctx, int32_t n_sub, double dt);

/* local adaptive time step per independent unit ("We instead compute a local
 * dt* for each r0 ... and update M_b at each r0 asynchronously"; Alg. 2 l.2-5).
 * Advances EVERY configuration c from t to t + dt with its own n_c = max(1, ceil(dt lambda_c / cfl)) forward-Euler
 * steps (or RK2 + Superbee steps, see below) of equal size dt / n_c, where lambda_c is the S8 positivity rate maximised over the disc cells of c
 * (readings Q31-Q33 in DESIGN.md).  lambda_c and n_c are computed on the device in fp64 in every dtype; the number
 * of passes (max_c n_c) is read back once per call (one 4-byte copy; the call synchronises the stream for it).
 * With the coupled source (MM_OPT_FREE_COUPLING) the local steps take k_on M_f(r0) from the frozen table -- Alg. 2 as one
 * loop (l.5 with l.20's M_f) -- on kernels 0 / 5.  dt > 0, cfl > 0, finite; MM_ERR_STATE unless density and velocities
 * have been set.  With MM_FLAG_RK2_SUPERBEE every local step is the paper's two-stage scheme (Alg. 2 l.5 driving
 * l.9-10) on the generic stage kernels: any grid, coupled source or not, two density buffers (single-buffer context:
 * MM_ERR_INVALID_ARG), two launches per local step. */
mm_status mm_advance_local(mm_ctx *ctx, double dt, double cfl);
/* n_c [Nc] (int32) and lambda_c [Nc] (fp64) of the last mm_advance_local; either pointer may be NULL.
 * MM_ERR_STATE before the first mm_advance_local or after new velocities were set. */
mm_status mm_local_steps(mm_ctx *ctx, int32_t *n_steps, double *lambda, int dst_on_device);

/* motor-force spreading onto the fluid grid (Eq. 10: F_2(x) = F iiint p
 * delta(y + (l/L) s p - x) Psi M_b ds dr0 dy dtheta).  Readings Q34-Q37 in DESIGN.md: plane j of
 * configuration c = (ix, iy, itheta) carries the S9 spring force before the sum over j, f_j(c) = -k dxi deta sum_ab
 * (xi_a, eta_b) m[c,j,a,b]; its head is at X = (ix/nx, iy/ny) + s_j p_c on the periodic unit square; the delta is
 * Peskin's 4-point kernel phi per direction:
 *     F2[gx][gy][.] = dtheta ds sum_{c,j} Psi_c f_j(c) phi(nx (X - X_g)_x) phi(ny (X - X_g)_y).
 * mm_set_psi : Psi [Nc], fp64 (macroscale data stays double), copied.
 * mm_spread_force : F2 [nx][ny][2] fp64, OVERWRITTEN with the spread force of the current density.  Computed as a
 *                   gather in a fixed summation order: the same inputs give the same bits (MM_OPT_SPREAD_ATOMIC = 1:
 *                   fp64 atomic adds, order varies from call to call).  The head's node coordinate is evaluated as
 *                   ix + s_j cos(theta) nx (translation-invariant), the oracle's ((ix/nx) + s_j cos(theta)) nx to
 *                   rounding.  MM_ERR_STATE unless density and Psi have been set; MM_ERR_INVALID_ARG when ntheta * ns >
 *                   2097120. */
mm_status mm_set_psi(mm_ctx *ctx, const double *psi, int src_on_device);
mm_status mm_spread_force(mm_ctx *ctx, double *F2, int dst_on_device);

/* free-motor coupling (Eq. 5-6; Alg. 2 l.14-20).  Readings
 * Q38-Q42 in DESIGN.md: the anchor of cell (c,j,a,b) is r0 = (ix/nx, iy/ny) + s_j p_c - (xi_a, eta_b), binned to the
 * nearest node of the periodic (x, y) grid;
 *     M_b,coarse[n] = dtheta ds dxi deta sum_{cells -> n} Psi_c m;      M_total = params.m_free at every node;
 * where M_b,coarse[n] > M_total every cell of node n is scaled by M_total / M_b,coarse[n] (the density IS modified) and
 * M_b,coarse[n] = M_total; M_f[n] = M_total - M_b,coarse[n] >= 0.  The call stores M_f and switches the source of the
 * following substeps to k_on M_f(r0) 1_disc (MM_OPT_FREE_COUPLING), frozen until the next call.
 * With the coupled source mm_substep runs kernels 4 / 5 (forward Euler on 16x16 / 8x8 offset planes) or the generic
 * kernels (any grid, RK2 + Superbee; two density buffers).
 * Mb_coarse, M_free: [nx][ny] fp64 outputs, either may be NULL.  Needs mm_set_psi. */
mm_status mm_update_free_motors(mm_ctx *ctx, double *Mb_coarse, double *M_free, int dst_on_device);

/* The same update (Eq. 5-6; Alg. 2 l.14-20; readings Q38-Q42) WITHOUT a context and
 * without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it): no cudaMalloc / cudaFree / allocating library routine is called, now or at first use.  The
 * node tables the three kernels pass between them live in ONE file-scope device array of MM_NOALLOC_MAX_NODES * 32 +
 * 256 bytes (512.25 KB), which every GPU that loads the library holds until exit.
 *   grid, params : as for mm_create (only the geometry and m_free = M_total are used); HOST pointers.
 *   density      : DEVICE pointer, canonical layout [ix][iy][itheta][j][a][b], `dtype` elements; IN/OUT -- cells of a node
 *                  above the cap are rescaled in place, as mm_update_free_motors does with the context's density.
 *   psi          : DEVICE pointer, [nc] fp64 (the filament density Psi per configuration).
 *   Mb_coarse, M_free : DEVICE pointers, [nx][ny] fp64 OUTPUTS, both required.
 *   cuda_stream  : all work is enqueued on it; the call does not synchronise.  The device the stream belongs to must be
 *                  current.
 * Same kernels and kernel choice as mm_update_free_motors; where both take the fixed-point route the results are
 * bitwise equal.  MM_ERR_INVALID_ARG (message via mm_last_error(NULL)) when nx * ny > MM_NOALLOC_MAX_NODES, a pointer is
 * NULL or the geometry is invalid.  Every call on a device shares the array, which keeps the last call's contents (each
 * call clears what must start at zero): calls that overlap on the GPU -- two streams with no ordering between them --
 * RACE; order them (same stream, or events).  It does not touch any mm_ctx. */
#define MM_NOALLOC_MAX_NODES 16384   /* nx * ny, e.g. 128 x 128 (BASELINE configs[4]) */
mm_status mm_free_motors_noalloc(const mm_grid *grid, const mm_params *params, mm_dtype dtype, void *density,
                                 const double *psi, double *Mb_coarse, double *M_free, void *cuda_stream);

/* Moments (S9) of the current density: force [Nc][2] = (Fx, Fy), torque [Nc]; always fp64
 * (macroscale data stays double precision).  Either pointer may be NULL to skip it. */
mm_status mm_moments(mm_ctx *ctx, double *force, double *torque, int dst_on_device);

mm_status mm_set_option(mm_ctx *ctx, mm_option opt, int64_t value);
mm_status mm_get_option(const mm_ctx *ctx, mm_option opt, int64_t *value); /* current setting; MM_ERR_INVALID_ARG on NULL / unknown */

/* The second roof of the fused kernels ("measure and record the box's fp64 and fp32 FMA peaks with a
 * small register-only microbenchmark"): runs a register-only FMA probe of the given dtype on every SM of the current
 * device (about 10 ms, on the given cudaStream_t, synchronises it) and returns the rate in TFLOP/s (2 flops per FMA).
 * Needs no context.  MM_ERR_CUDA without a device. */
mm_status mm_measure_fma_peak(mm_dtype dtype, void *cuda_stream, double *tflops);
/* The same measurement by the number of FRESH register operands per FMA: fresh_operands = 1 is mm_measure_fma_peak (two
 * operands loop-invariant: the FMA unit's rate); 3 = coefficient, value and accumulator all change from one FMA to the
 * next, as in a stencil with per-lane coefficients: the rate the register file sustains (two 32-bit operands per cycle
 * and scheduler: about 2/3 of the peak for fp32).  MM_ERR_INVALID_ARG for other counts. */
mm_status mm_measure_fma_rate(mm_dtype dtype, int32_t fresh_operands, void *cuda_stream, double *tflops);

/* Number of kernels this context has launched so far (bench.py's gpu_launches). */
int64_t mm_launch_count(const mm_ctx *ctx);
/* Name of the substep kernel variant the last mm_substep used ("stream<f64,16x16,T=2>", "generic<f64>", ...). */
const char *mm_kernel_name(const mm_ctx *ctx);

/* Destroy the context (the end of the resident state of PAPER.md:133): synchronises the context's stream, frees
 * library-owned buffers; borrowed density buffers are left to their owner.  NULL is a no-op. */
mm_status mm_destroy(mm_ctx *ctx);

const char *mm_status_string(mm_status s);
const char *mm_last_error(const mm_ctx *ctx); /* "" if none; ctx may be NULL (returns the create-time error) */

#ifdef __cplusplus
}
#endif
#endif /* MM_H_ */
