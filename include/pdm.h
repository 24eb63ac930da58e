/*
 * pdm.h -- C ABI of libpdm: the hot path of explicit f-x poststack depth migration
 * (arXiv 1912.05529; citations are /root/reference/PAPER.md lines; R# = readings in DESIGN.md).
 *
 * What the library computes (and nothing else):
 *
 *   Eq. (1), PAPER.md:45      P(z+dz, w, x) = sum_{k=-L..L} W_k(u(x,z,w)) * P(z, w, x-k)
 *   PAPER.md:65, :83          the 2L+1-tap extrapolator W(u) is LOOKED UP in a pre-designed table,
 *                             per output point, by u = w*dz/v(x,z)                 (R3, R8)
 *   PAPER.md:59-70, :85       marched over every depth level; after each level the depth row is
 *                             image[z][x] = sum_w Re P(z+dz, w, x)                 (R1, R6, R10)
 *
 *   index rule (R3)           q32[z][x] = (float)((double)dz / ((double)v32[z][x] * tab_du))
 *                             idx = clamp(rint_half_even(fl32(w32 * q32)), 0, ntab-1)
 *   edges (R5)                samples with x-k outside [0,nx) contribute zero
 *   rows (R6, R7)             step iz uses velocity row iz; image row iz = field AFTER step iz
 *
 * Every entry point returns PDM_OK (0) or a negative pdm_status; nothing throws or aborts
 * across the ABI.  All sizes are element counts; all arrays are dense row-major.
 * "HOST" / "DEVICE" says where a pointer must point.  There is no CPU fallback: without a
 * compute-capability-10.x device pdm_create fails with PDM_ERR_UNSUPPORTED.
 */
#ifndef PDM_H
#define PDM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pdm_plan pdm_plan;            /* opaque; owned by the library                        */
typedef struct { float re, im; } pdm_c64;    /* == torch.complex64 / numpy.complex64 / cuFloatComplex */

typedef enum {
    PDM_OK = 0,
    PDM_ERR_INVALID_ARG = -1,      /* NULL pointer, dim <= 0, ntaps even or < 1, tab_du <= 0,
                                      non-finite or <= 0 velocity / omega, unknown flag bits       */
    PDM_ERR_TABLE_RANGE = -2,      /* some rint(w*q) > ntab-1 (kernels still clamp defensively)    */
    PDM_ERR_TABLE_ASYMMETRIC = -3, /* only with PDM_REQUIRE_SYMMETRIC: table[j][L+k] != table[j][L-k]
                                      bitwise.  Without that flag such a table selects the general
                                      kernels (full 2L+1 row, 8L+4 lane-ops per sample instead of
                                      6L+4) and pdm_info.table_symmetric reports 0                 */
    PDM_ERR_UNSUPPORTED = -4,      /* not a CC 10.x device; forced path impossible for this nx;
                                      ntaps above PDM_MAX_TAPS; a forced SMEM / TILED / CLUSTER path
                                      with more than 51 taps (the longest unrolled kernel; shorter
                                      filters of any odd length run on the next longer kernel with
                                      zero taps appended, longer ones only on PDM_PATH_NAIVE)      */
    PDM_ERR_NOMEM = -5,            /* host or device allocation failed.  pdm_create compares every large
                                      request with the free device memory BEFORE allocating; the main
                                      form needs grid_ctas*nz*nx*4 B of per-CTA partial images (the
                                      total is pdm_info.workspace_bytes of a plan that was created)  */
    PDM_ERR_CUDA = -6,             /* a CUDA call failed; pdm_info.last_cuda_error has the code    */
    PDM_ERR_TOO_LARGE = -7         /* pdm_migrate_static only: nx*nw exceeds PDM_STATIC_MAX_SAMPLES, the
                                      size of the library's built-in scratch                       */
} pdm_status;

#define PDM_MAX_TAPS 129           /* L <= 64 */

/* flags word of pdm_create: bits 0-3 choose the kernel form, the rest are tuning/debug knobs.     */
#define PDM_PATH_AUTO    0u  /* SMEM marching if a line (ping-pong) fits one CTA, else x-tiled; the  */
                             /* cluster form when there are too few lines to fill the SMs, or when a */
                             /* line fits a pair of CTAs and its tap rows can still be staged        */
#define PDM_PATH_SMEM    1u  /* main form: one CTA keeps a frequency's x-line in shared memory and   */
                             /* marches all nz depth steps in place (north_star)       */
#define PDM_PATH_TILED   2u  /* x-tiled per-depth-step kernel with +-L halos, planes ping-pong in HBM*/
#define PDM_PATH_NAIVE   3u  /* scaffold: one thread per (w,x) sample, one launch per depth level --  */
                             /* the paper's own mapping, kept only as a cross-check    */
#define PDM_PATH_CLUSTER 4u  /* main form with the line split over a thread-block cluster of 2, 4 or */
                             /* 8 CTAs, halos exchanged through distributed shared memory            */
#define PDM_PATH_PACKED  5u  /* x-tiled AND temporally blocked (T depth steps per tile visit, planes   */
                             /* cross HBM once per T steps, tiles moved by TMA) with 8 adjacent       */
                             /* frequencies per quarter warp, which makes the per-sample tap gather   */
                             /* bank-conflict free; any nx.  Tap rows are staged  */
                             /* per tile visit in shared memory; where one pack's row range on a     */
                             /* visit is wider than any slice buffer (velocity varying > ~2x inside  */
                             /* a tile at the top frequencies with 51 taps and 1024 rows) forced,    */
                             /* PDM_PRESTACK and PDM_TAPER plans read the rows from the global table */
                             /* instead (256-thread build, pdm_info.taps_mode = 1; slower, same      */
                             /* bits); AUTO poststack plans take another form.  A forced CTA size of */
                             /* 384 or 512 threads then gives PDM_ERR_UNSUPPORTED                    */
#define PDM_PATH_MASK    0xFu
#define PDM_TAPS_AUTO    (0u << 4)  /* where the kernels read filter rows from                      */
#define PDM_TAPS_GLOBAL  (1u << 4)  /* always from the L2/L1-cached global half-table               */
#define PDM_TAPS_SLICE   (2u << 4)  /* rows a frequency can touch staged in shared memory; whether   */
#define PDM_TAPS_COMPACT (3u << 4)  /* the list is the contiguous range [idx(q_min), idx(q_max)] or  */
                                    /* the exact rows (models with <= 2048 distinct velocities) is   */
                                    /* the library's choice either way: both values request staging, */
                                    /* pdm_info.taps_mode reports 2 (range) or 3 (exact list)        */
#define PDM_TAPS_MASK    (0x3u << 4)
#define PDM_FORCE_GENERAL (1u << 6) /* debug: never take the thread-uniform fast path (every output   */
                                    /* fetches its own tap row even where a warp shares one)        */
#define PDM_NO_BALANCE   (1u << 7)  /* debug: whole lines per CTA (no depth-split load balancing)   */
#define PDM_REQUIRE_SYMMETRIC (1u << 20) /* refuse a table that is not bitwise symmetric in k        */
                                    /* (PDM_ERR_TABLE_ASYMMETRIC) instead of taking the general kernels */
#define PDM_THREADS_SHIFT 8         /* bits 8-15: threads per CTA / 32 (0 = auto); with              */
                                    /* PDM_PATH_PACKED one of 8, 12, 16 (else PDM_ERR_UNSUPPORTED)  */
#define PDM_CTAS_SHIFT    16        /* bits 16-19: CTAs per SM for the persistent grid (0 = auto);  */
                                    /* with PDM_PATH_CLUSTER: the cluster size 2, 4 or 8 (0 = auto) */
                                    /* with PDM_PATH_PACKED: depth steps per tile visit T (0 = auto) */
                                    /* with PDM_PATH_TILED: depth steps per launch, 1 or 2 (0 = auto)*/
#define PDM_PRESTACK      (1u << 21) /* plan for pdm_migrate_shot (shot-profile prestack migration,    */
                                    /* PAPER.md:151): always the PDM_PATH_PACKED form (AUTO or PACKED   */
                                    /* path bits), any table; pdm_migrate refuses such a plan           */
#define PDM_TAPER_SHIFT   22         /* bits 22-29: absorbing edge taper over n = 1..255 samples per side  */
                                    /* (variant R5b of the zero edges R5; the paper is silent on the     */
                                    /* boundary): after every step the new field is multiplied by        */
                                    /* t(x) = sin^2((pi/2)(d+1)/(n+1)), d = min(x, nx-1-x) < n.  Always   */
                                    /* the PDM_PATH_PACKED form (AUTO or PACKED path bits); not with      */
                                    /* PDM_PRESTACK.  0 = plain R5                                        */
#define PDM_TABLE_INTERP  (1u << 30) /* interpolated look-up (variant R3c of the nearest-row rule R3; the    */
                                    /* paper only says the filter is looked up): the     */
                                    /* operator of an output point is the linear blend of the two table    */
                                    /* rows bracketing u = w*dz/v,  j0 = floor(fl32(w*q32)), a = the        */
                                    /* fraction,  W_k = (1-a) table[j0][k] + a table[j0+1][k]; at or beyond */
                                    /* the last row, that row alone.  Runs on the per-depth-step form only  */
                                    /* (pdm_info.path = PDM_PATH_NAIVE; AUTO or NAIVE path bits), plain     */
                                    /* poststack (not with PDM_PRESTACK / PDM_TAPER): the accurate-table    */
                                    /* reference mode, not a fast path                                      */
#define PDM_FLAGS_VALID  0x7FFFFFFFu /* any other bit set: PDM_ERR_INVALID_ARG                       */

typedef struct {
    int    path;                 /* PDM_PATH_* actually chosen                                      */
    int    taps_mode;            /* PDM_TAPS_* >> 4 actually chosen                                 */
    int    nx, nz, nw, ntab, ntaps;
    int    grid_ctas;            /* CTAs of the dominant kernel                                     */
    int    threads_per_cta;
    int    ctas_per_sm;
    int    smem_bytes;           /* dynamic shared memory per CTA of the dominant kernel            */
    int    launches_per_migrate; /* kernels one pdm_migrate call enqueues                           */
    int    sm_count;
    int    last_cuda_error;      /* cudaError_t of the last failing CUDA call (0 if none)           */
    int    table_symmetric;      /* 1: W_k == W_-k bitwise, folded kernels; 0: general kernels      */
    double samples;              /* nx*nz*nw: extrapolated (z,w,x) points per migrate               */
    double counted_flops;        /* 8*(2L+1)*samples (metric definition, BASELINE.json north_star)  */
    double executed_lane_ops;    /* (6L+4)*samples FP32 lane operations with symmetric folding      */
    double workspace_bytes;      /* device memory the plan owns                                     */
} pdm_info;

/*
 * pdm_create -- validate, pre-digest and upload everything that does not depend on the data.
 *   out       HOST  receives the plan; *out = NULL on failure.
 *   nx,nz,nw  lateral samples, depth steps, frequencies.
 *   dx,dz     metres.  dx is metadata only (it enters through the filter design, R9).
 *   omega     HOST  float[nw], rad/s, any order, finite, > 0.
 *   velocity  HOST  float[nz][nx], m/s, finite, > 0: the MIGRATION velocity; the library computes
 *             exactly u = w*dz/velocity (the caller passes v/2 for two-way-time data, R2).
 *   table     HOST  pdm_c64[ntab][ntaps]; table[j][L+k] = W_k(u_j), u_j = j*tab_du, k = -L..L, and
 *             W_k multiplies P(x-k) (Eq. (1), R11).  A table that is bitwise symmetric in k runs
 *             on the folded kernels; any other table on the general ones.
 *   flags     PDM_PATH_* | PDM_TAPS_* | tuning bits.
 * The caller may free all its arrays on return.  The plan is bound to the CUDA device that is
 * current at the call.  Not thread-safe per plan; different plans are independent.
 */
int pdm_create(pdm_plan **out, int nx, int nz, int nw, float dx, float dz,
               const float *omega, const float *velocity,
               const pdm_c64 *table, int ntab, int ntaps, double tab_du,
               unsigned flags);

/*
 * pdm_migrate -- the timed call: march P0 through all nz depth levels and image it.
 *   P0_dev     DEVICE pdm_c64[nw][nx]  f-x section at z = 0, read-only, not modified.
 *   image_dev  DEVICE float[nz][nx]    overwritten with sum_w Re P after every step.
 *   cuda_stream  cudaStream_t (0 = legacy default stream).
 * Asynchronous on the stream; performs no allocation, no host synchronisation and no host<->device
 * copy (CUDA-graph capturable); bit-identical images on repeated calls (fixed summation order, no
 * float atomics).  One migrate in flight per plan (the workspace is per plan).  "Enqueue only" on the
 * PDM_PATH_PACKED form includes one host-side encode of the TMA descriptor of the caller's P0 (a pure
 * CPU computation of ~1 us, no driver state touched), because P0's address is only known at the call.
 * Errors: PDM_ERR_INVALID_ARG (NULL), PDM_ERR_CUDA (launch failure, wrong current device).
 */
int pdm_migrate(pdm_plan *plan, const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream);

/*
 * pdm_migrate_host -- same operation with HOST buffers (the end-to-end call): copies P0 to the
 * device, runs pdm_migrate, copies the image back and synchronises the stream before returning.
 *   P0_host    HOST pdm_c64[nw][nx] (pinned memory makes the copies asynchronous and faster).
 *   image_host HOST float[nz][nx].
 * Uses staging buffers owned by the plan (allocated on first use: PDM_ERR_NOMEM possible) -- except on
 * the main (SMEM-marching) form with BOTH buffers pinned: the kernels then read P0 and write the image
 * through the host mapping, so the transfers overlap the computation (same bits either way).
 */
int pdm_migrate_host(pdm_plan *plan, const pdm_c64 *P0_host, float *image_host, void *cuda_stream);

/*
 * pdm_migrate_shot -- prestack (shot-profile) migration of ONE shot (PAPER.md:151 names the extension;
 * the scheme is reading R17 of DESIGN.md, built from the same step, Eq. (1)):
 *     R(z+dz,w,x) = sum_k      W_k(u)  R(z,w,x-k)      recorded field, continued downward
 *     S(z+dz,w,x) = sum_k conj(W_k(u)) S(z,w,x-k)      source field, propagated forward
 *     image[z][x] (+)= sum_w Re( conj(S(z+dz,w,x)) R(z+dz,w,x) )     zero-lag cross-correlation
 * with the plan's velocity, table, index rule (R3), rows (R6, R7) and zero edges (R5).
 *   plan       created with PDM_PRESTACK.
 *   src_dev    DEVICE pdm_c64[nw][nx]  source wavefield at z = 0, read-only.
 *   rec_dev    DEVICE pdm_c64[nw][nx]  shot gather in f-x at z = 0, read-only.
 *   image_dev  DEVICE float[nz][nx]    overwritten (accumulate == 0) or added to (accumulate != 0:
 *                                      several shots into one image, in call order).
 * Enqueue only, deterministic, one call in flight per plan -- as pdm_migrate.
 * Errors: PDM_ERR_INVALID_ARG (NULL, a plan without PDM_PRESTACK), PDM_ERR_CUDA.
 */
int pdm_migrate_shot(pdm_plan *plan, const pdm_c64 *src_dev, const pdm_c64 *rec_dev, float *image_dev,
                     int accumulate, void *cuda_stream);

/*
 * pdm_migrate_static -- the whole migration (Eq. (1) at every depth level + the imaging sum, same
 * index rule R3, zero edges R5 and row conventions R6/R7 as pdm_migrate) for callers that MUST NOT
 * ALLOCATE device memory: no plan, no pdm_create.
 *
 * Who needs it: code that runs where cudaMalloc / cudaFree are off limits -- an extension inside a host
 * application that owns all device memory and gives plug-ins fixed buffers; a latency-bound loop that
 * cannot afford the device-wide synchronisation an allocation implies; a job sized to the last byte of
 * HBM that must not discover an out-of-memory error in the middle of a survey.  Every other migration
 * call of this library needs a plan, and pdm_create allocates.
 *
 * How: this entry point calls no cudaMalloc, cudaFree or any routine that allocates.  Its only scratch
 * (two wavefield planes, ping-pong between depth steps) is a fixed array compiled into the library:
 * 2 * PDM_STATIC_MAX_SAMPLES * 8 B = 16 MiB of device memory that every GPU on which the library's
 * code gets loaded holds until the process exits, whether or not this call is ever used again.
 * Problems with nx*nw > PDM_STATIC_MAX_SAMPLES are refused with PDM_ERR_TOO_LARGE (nothing is
 * launched); nz is not limited.  It is the per-depth-step form (one thread per (w,x) sample, 2*nz small
 * launches, the mapping of PDM_PATH_NAIVE): correct and allocation-free, not the fast path.
 *
 *   omega_dev     DEVICE float[nw]          rad/s (as pdm_create's omega, but already on the device)
 *   velocity_dev  DEVICE float[nz][nx]      migration velocity, m/s
 *   table_dev     DEVICE pdm_c64[ntab][ntaps], the layout pdm_create reads; symmetric or not
 *   P0_dev        DEVICE pdm_c64[nw][nx]    read-only
 *   image_dev     DEVICE float[nz][nx]      overwritten
 * All five belong to the caller and must stay valid until the stream has run the call.  Their CONTENTS
 * are not validated (that would need a host synchronisation): a table index beyond ntab-1 is clamped,
 * non-finite or non-positive values give undefined images, not errors.
 *
 * First call on a device: the library looks up the device address of its scratch array (once per
 * device, with that device current) before launching.  Make that first call outside any stream
 * capture; later calls on the same device only launch kernels on cuda_stream.
 *
 * One array per process and GPU, shared by ALL calls: a call finds the previous call's wavefield in it.
 * Nothing in it needs clearing -- every element is written in a call before that call reads it -- but two
 * calls that may execute concurrently on one GPU (different streams without an event between them)
 * corrupt each other.  Serialise them.  Deterministic: same inputs, same bits, and the same bits as a
 * PDM_PATH_NAIVE plan.
 * Errors: PDM_ERR_INVALID_ARG (NULL, size <= 0, even ntaps, dz or tab_du <= 0), PDM_ERR_UNSUPPORTED
 * (ntaps > PDM_MAX_TAPS, no CC 10.x device current), PDM_ERR_TOO_LARGE, PDM_ERR_CUDA.
 */
#define PDM_STATIC_MAX_SAMPLES (1 << 20)   /* nx*nw limit of pdm_migrate_static                        */
int pdm_migrate_static(int nx, int nz, int nw, float dz,
                       const float *omega_dev, const float *velocity_dev,
                       const pdm_c64 *table_dev, int ntab, int ntaps, double tab_du,
                       const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream);

/* pdm_destroy -- free all device and host state of the plan.  NULL is allowed. */
int pdm_destroy(pdm_plan *plan);

/* pdm_get_info -- fill *out (HOST) with the plan's launch configuration and work counts. */
int pdm_get_info(const pdm_plan *plan, pdm_info *out);

/* pdm_strerror -- static string for a pdm_status (never NULL). */
const char *pdm_strerror(int code);

/*
 * ================================================================================================
 * MEASUREMENT / DEBUG entry points -- not part of the hot path's contract; used by
 * bench.py for the roofline figures and by the tests for pin P12.  Everything above this banner is
 * the product boundary; pdm_tf_* and pdm_design_table further down are the two setup stages.
 * ================================================================================================
 *
 * pdm_profile_enable / pdm_profile_read -- per-kernel device timing for the roofline report.
 * While enabled, pdm_migrate records CUDA events on the caller's stream before the dominant
 * kernel(s) (A1-A4: the marching kernel, or all nz x-tiled step launches), between them and the
 * imaging reduction (A5), and after it.  Recording an event is capture-safe and costs ~1 us.
 * pdm_profile_read synchronises on the last event of the most recent pdm_migrate and returns
 *   main_ms    HOST float: duration of the dominant kernel(s) of that call, milliseconds
 *   reduce_ms  HOST float: duration of the reduction kernel
 * Errors: PDM_ERR_INVALID_ARG (NULL, profiling not enabled or no migrate since), PDM_ERR_CUDA.
 */
int pdm_profile_enable(pdm_plan *plan, int enable);
int pdm_profile_read(pdm_plan *plan, float *main_ms, float *reduce_ms);

/*
 * pdm_debug_table_index -- DEVICE evaluation of the index rule R3 (pin P12 on the GPU side):
 *   idx_dev[i] = clamp(rint(fl32(omega_dev[i] * q)), 0, ntab-1), q = (float)(dz/(velocity_dev[i]*tab_du))
 * with q formed on the HOST side of the library exactly as pdm_create does (so velocity is HOST).
 *   omega HOST float[n], velocity HOST float[n], idx_out HOST int[n].  Synchronous.
 */
int pdm_debug_table_index(const float *omega, const float *velocity, int n,
                          double dz, double tab_du, int ntab, int *idx_out);

/*
 * pdm_fp32_peak -- FP32-FMA throughput microbenchmark (independent FFMA chains on every SM),
 * the denominator of the "% of FP32 FMA peak" metric.  Runs `iters` chain iterations on
 * `cuda_stream` and returns the best of `repeats` timings.
 *   packed       0 = scalar FFMA, 1 = packed fma.rn.f32x2 (FFMA2)
 *   tflops_out   HOST double: achieved 1e12 flop/s (2 flops per FMA lane-op)
 */
int pdm_fp32_peak(int packed, int iters, int repeats, void *cuda_stream, double *tflops_out);

/*
 * ---- time -> frequency transform of the input section ----------------------
 * PAPER.md:51, Alg. 1 (:58): every trace of the zero-offset section is Fourier transformed along
 * the TIME axis only; the depth loop consumes the resulting f-x section.  For the
 * nw selected DFT bins (omega_j = 2*pi*bins[j] / (nt*dt)) this computes, in FP32,
 *
 *     P0[j][x] = sum_{n=0}^{nt-1} section[n][x] * exp(-2*pi*i * bins[j] * n / nt)     (no scaling)
 *
 * i.e. exactly the layout pdm_migrate reads.  Twiddles come from an nt-entry table built in double
 * at create time and indexed by the exact integer (bins[j]*n) mod nt.
 *
 * pdm_tf_create  -- bins: HOST int[nw], each in [0, nt/2]; copies what it needs.
 *                   Errors: PDM_ERR_INVALID_ARG (NULL, sizes <= 0, bin out of range),
 *                   PDM_ERR_UNSUPPORTED (no CC 10.x device, nt > PDM_TF_MAX_NT), PDM_ERR_NOMEM/CUDA.
 * pdm_tf_forward -- section_dev: DEVICE float[nt][nx] (time-major, x fastest), read-only;
 *                   P0_dev: DEVICE pdm_c64[nw][nx], overwritten.  Enqueue only on cuda_stream
 *                   (no allocation, no host sync, no copies); deterministic.
 * pdm_tf_destroy -- frees the plan; NULL is allowed.
 */
typedef struct pdm_tf pdm_tf;
#define PDM_TF_MAX_NT 8192         /* the twiddle table (8 B per entry) lives in shared memory */
int pdm_tf_create(pdm_tf **out, int nt, int nx, int nw, const int *bins);
int pdm_tf_forward(pdm_tf *tf, const float *section_dev, pdm_c64 *P0_dev, void *cuda_stream);
int pdm_tf_destroy(pdm_tf *tf);

/*
 * ---- extrapolator-table design on the device -------------------------------
 * PAPER.md:39 (the filters trade length against maximum propagation angle), :83 ("Designing filters
 * itself is optimization problem, it takes sometime ... we design the filters in advance and store
 * it on the disk"), refs :163-165, :179-180.  The paper gives no recipe; pdm_design_table runs the
 * projections-onto-convex-sets style iteration DESIGN.md states as D1-D4 for all ntab rows at once
 * (one CTA per row, FP64): row j approximates the one-way phase shift of normalised wavenumber
 * u_j = j*tab_du,
 *     D(kappa) = exp(+i sqrt(u^2 - (r kappa)^2))  for |r kappa| <= u,  exp(-sqrt((r kappa)^2 - u^2)) beyond,
 * kappa = k_x dx in [-pi, pi], r = dz/dx, with a 2L+1-tap symmetric filter that is exact (to the
 * iteration's fixed point) on the passband |kappa| <= min((u/r) sin(angle), kappa_cap) and has
 * |response| <= stop_cap elsewhere; the taps are finally divided by max(1, max|H|)(1+4e-7) so that
 * the complex64 table is stable (|H| <= 1), and mirrored bit for bit (W_-k = W_k).
 *   table_host  HOST pdm_c64[ntab][ntaps], overwritten; the layout pdm_create reads.
 *   opts        HOST, NULL = the defaults in the comments below.
 * Synchronous on cuda_stream (setup call: allocates and frees its own scratch).  Errors:
 * PDM_ERR_INVALID_ARG, PDM_ERR_UNSUPPORTED (no CC 10.x device; L > 64; grid too large for shared
 * memory), PDM_ERR_NOMEM, PDM_ERR_CUDA.
 */
typedef struct {
    int    n_iter;               /* D2 iterations                      (default 200)                */
    int    n_grid;               /* periodic kappa grid N, even        (default 2048)               */
    int    n_check;              /* D3 kappa points on [0, pi]         (default 16384)              */
    double passband_angle_deg;   /* maximum propagation angle          (default 55)                 */
    double kappa_cap;            /* anti-alias cap of the passband     (default 0.8 pi)             */
    double stop_cap;             /* |H| ceiling outside the passband   (default 0.9995)             */
} pdm_design_opts;
int pdm_design_table(pdm_c64 *table_host, int ntab, int ntaps, double tab_du, double dz_over_dx,
                     const pdm_design_opts *opts, void *cuda_stream);

/*
 * ---- 3-D variant ---------------------------------------------------------
 * PAPER.md:41 ("the explicit f-x migration can be easily extended to the 3-D depth migration, which
 * requires 2-D filters as extrapolators"), :47.  Eq. (1) on two lateral axes (reading R18):
 *
 *     P(z+dz, w, y, x) = sum_{ky=-L..L} sum_{kx=-L..L} W_{ky,kx}(u(x,y,z)) * P(z, w, y-ky, x-kx)
 *     image[z][y][x]   = sum_w Re P(z+dz, w, y, x)
 *
 * with the same index rule (R3, from velocity[z][y][x]), zero terms outside the grid on both axes (R5)
 * and rows as in R6/R7.  The table is general: no symmetry is assumed or needed; a table that is bitwise
 * symmetric in kx AND in ky (circularly symmetric extrapolators) runs on folded kernels (L+1 passes over
 * row sums, (L+1)(6L+4) lane-ops per sample instead of 4(2L+1)^2), info.table_symmetric reports which.
 *
 * pdm3_create  -- omega HOST float[nw]; velocity HOST float[nz][ny][nx]; table HOST
 *                 pdm_c64[ntab][ntaps][ntaps], table[j][L+ky][L+kx] = W_{ky,kx}(u_j), u_j = j*tab_du;
 *                 flags: 0, PDM_FORCE_GENERAL, PDM_REQUIRE_SYMMETRIC (refuse a table that is not doubly
 *                 symmetric: PDM_ERR_TABLE_ASYMMETRIC).  Errors as pdm_create; PDM_ERR_UNSUPPORTED for
 *                 ntaps > 15 (the longest unrolled 2-D kernel; shorter odd lengths run on the next
 *                 longer one with zero taps appended).
 * pdm3_migrate -- P0_dev DEVICE pdm_c64[nw][ny][nx] (read-only), image_dev DEVICE float[nz][ny][nx]
 *                 (overwritten).  Enqueue only (nz + 1 launches), deterministic.
 * pdm3_get_info / pdm3_destroy -- as the 2-D calls (info.path reports 6; info.samples = nx*ny*nz*nw,
 *                 counted_flops = 8*ntaps^2 per sample).
 */
typedef struct pdm3_plan pdm3_plan;
int pdm3_create(pdm3_plan **out, int nx, int ny, int nz, int nw, float dz,
                const float *omega, const float *velocity,
                const pdm_c64 *table, int ntab, int ntaps, double tab_du, unsigned flags);
int pdm3_migrate(pdm3_plan *plan, const pdm_c64 *P0_dev, float *image_dev, void *cuda_stream);
int pdm3_get_info(const pdm3_plan *plan, pdm_info *out);
int pdm3_destroy(pdm3_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* PDM_H */
