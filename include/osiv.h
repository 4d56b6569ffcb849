/*
 * osiv.h -- C ABI of libosiv: ordered-subset, TV-regularised statistical iterative
 * reconstruction (OS-TV) of 2-D fan-beam MVCT slices on one NVIDIA B200 (sm_100a).
 *
 * Method: arxiv 1903.10088, "Technical Note: Fast Statistical Iterative Reconstruction for
 * MVCT in TomoTherapy".  Citations "PAPER.md:N" are lines of the extracted paper text;
 * "C1..C12" are the readings adopted where the paper is silent (SURVEY.md section 8(c),
 * restated in DESIGN.md section 3).
 *
 * Problem statement: geometry + measured Poisson counts + TV weight
 * beta + ordered subsets + iterations -> attenuation image.  Every step of the iteration runs
 * in hand-written CUDA kernels; this library has no CPU fallback and every entry point that
 * needs the GPU returns OSIV_ERR_CUDA when none is usable.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  All are owned by the
 *     caller, contiguous, and are neither freed nor retained beyond the call (asynchronous work
 *     enqueued on `cuda_stream` still reads/writes them until the stream reaches that point).
 *   - Images are float32 [batch][ny][nx], row-major, img[iy*nx+ix]; pixel (ix,iy) has its centre
 *     at ((ix-(nx-1)/2)*pixel_mm, (iy-(ny-1)/2)*pixel_mm).  Attenuation in 1/mm.
 *   - Sinograms are float32 [batch][V_S][C] (compact: the views v = m, m+M, m+2M, ... of subset
 *     m of M in that order; V_S = n_views/M, or all n_views when subset < 0).  Line integrals
 *     are dimensionless (mm * 1/mm).
 *   - Counts are float32 [batch][n_views][n_channels] (all views; integers < 2^24 are exact).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Every function returns 0 (OSIV_OK) or a negative osiv_status; nothing throws, aborts or
 *     prints.
 */
#ifndef OSIV_H
#define OSIV_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    OSIV_OK              =  0,
    OSIV_ERR_INVALID_ARG = -1,  /* null pointer, non-positive size, n_views % n_subsets != 0, n_views > 65535,
                                   batch > max_batch, tv_eps <= 0, source inside the grid's circumscribed circle */
    OSIV_ERR_CUDA        = -2,  /* a CUDA runtime call failed (no device, out of memory, launch error) */
    OSIV_ERR_NOT_FINITE  = -3,  /* the monitor D became NaN/Inf for at least one slice */
    OSIV_ERR_SCRATCH_LIMIT = -4 /* osiv_tv_gradient_static: the padded images do not fit OSIV_STATIC_SCRATCH_BYTES */
} osiv_status;

/* Scan geometry (reading C1; the paper prints none, BASELINE.json supplies SAD/SDD/channels).
 * Lengths in mm, angles in rad.  Source of view v: SAD*(cos th_v, sin th_v), th_v = theta0 + 2*pi*v/V.
 * Ray (v,c): the zero-width line from the source in direction -(cos(th_v+ga_c), sin(th_v+ga_c)),
 * ga_c = (c - (C-1)/2 + channel_offset) * dgamma. */
typedef struct {
    int32_t nx, ny;          /* image size in pixels */
    double  pixel_mm;        /* square pixel side */
    int32_t n_views;         /* V, equally spaced over 360 degrees */
    int32_t n_channels;      /* C, equiangular */
    double  sad_mm;          /* source to isocentre */
    double  sdd_mm;          /* source to detector; informational only (line integrals do not use it) */
    double  dgamma_rad;      /* channel pitch; <= 0 selects 2*asin(R_FOV/SAD)/C, R_FOV = min(nx,ny)*pixel/2 */
    double  channel_offset;  /* in channels */
    double  theta0_rad;
    int32_t model;           /* system matrix a(i,r): 0 = exact length of the ray inside the pixel (reading C2, default);
                                1 = Joseph's interpolating model: one sample per image line of the ray's major axis,
                                linear interpolation between the line's two nearest pixels, times the path length per
                                line.  Forward and back use the same a(i,r) in either case. */
    int32_t reserved;        /* must be 0 */
} osiv_geometry;

/* Iteration parameters.  osiv_default_params() fills the paper's values. */
typedef struct {
    double  beta;            /* TV weight against the blank-normalised log-likelihood (C6,C7); the
                                subset update uses beta/M ("multiplied by the thinning parameter") */
    int32_t n_subsets;       /* M; subset m holds views {v : v mod M == m}; M must divide n_views */
    int32_t n_iters;         /* number of SUBSET updates */
    double  mu0;             /* homogeneous initial image, default 0.005 /mm = 0.05 /cm */
    double  lambda0;         /* 0.01 */
    double  lambda_up;       /* 1e-4   (Eq. 4) */
    double  lambda_down;     /* 2e-4   (Eq. 5) */
    double  lambda_min;      /* floor of lambda, 1e-4 (C10) */
    double  kappa;           /* step scale, 100 (C6): tau_S = kappa*SAD*dgamma/(V_S*max(nx,ny)*pixel^3) */
    double  tv_eps;          /* TV smoothing, 1e-5 /mm (C9) */
    int32_t return_best;     /* 0: final iterate; 1: iterate with the smallest monitor D */
    int32_t monitor_mode;    /* which earlier D Eq. 4-5 compare D(n) with: 0 = D(n-1), the previous iteration (C10, default);
                                1 = D(n-M), the same subset one pass earlier (G3; lambda(n) = lambda0 for n < M) */
    /* Stack of slices (readings H1-H3): the `batch` slices of a call form one volume, slice 0 first. */
    int32_t view_shift;      /* H1: views the gantry advances per slice; view j of slice s was taken at angle
                                theta0 + 2*pi*(j + view_shift*s)/V.  0 = every slice at the same angles (default) */
    int32_t reserved;        /* must be 0 */
    double  tv_z;            /* H2: > 0 couples neighbouring slices through the 3-D smoothed TV
                                sum sqrt(eps^2 + dx^2 + dy^2 + (tv_z*(mu_{s+1} - mu_s))^2); 0 = 2-D TV per slice (default).
                                Every slice keeps its own monitor and step (H3).  With view_shift != 0 or tv_z > 0,
                                return_best and forced_lambda must be off. */
    const double* forced_lambda;  /* HOST pointer: NULL, or n_iters values used instead of Eq. 4-5 */
} osiv_params;

typedef struct osiv_handle osiv_handle;

/* Library version (major*10000 + minor*100 + patch). */
int osiv_version(void);

/* Text for a status code; never NULL; static storage. */
const char* osiv_strerror(int status);

/* Fill *p with the defaults listed above (beta = 0.005, n_subsets = 1, n_iters = 1). */
int osiv_default_params(osiv_params* p);

/* Create a reconstruction context on CUDA device `device` for up to `max_batch` slices per call:
 * builds the per-ray geometry tables in float64 on the host, stores them as float32 in HBM, and
 * allocates the per-slice workspace lazily.  The handle is not thread-safe; use one per thread. */
int osiv_create(const osiv_geometry* geom, int32_t max_batch, int32_t device, osiv_handle** out);

/* Release everything the handle owns (synchronises the device).  NULL is accepted. */
int osiv_destroy(osiv_handle* h);

/* A0 setup, host only (no GPU needed): the per-ray coefficients the kernels use.  Writes, for every ray
 * (v,c), four floats {alpha, beta, g0, h} to h_rays [V][C][4] and {cos th_v, sin th_v} to h_views [V][2]
 * (either may be NULL), such that the weight is
 *   a(v,c; ix,iy) = h * clamp( w - |alpha*(ix-(nx-1)/2) + beta*(iy-(ny-1)/2) + g0|, 0, 1 ),
 * with half-width w = (|alpha|+|beta|)/2 for the exact chord of reading C2 (model 0; one of alpha, beta is +-1, the
 * other has magnitude >= 1) and w = 1 for Joseph's model (model 1; one of alpha, beta is +-1, the other has
 * magnitude <= 1).  Computed in float64, rounded once to float32. */
int osiv_ray_table(const osiv_geometry* geom, float* h_rays, float* h_views);

/* Resolved channel pitch (after the dgamma_rad <= 0 rule) and step constant tau_S for M subsets. */
int osiv_get_dgamma(const osiv_handle* h, double* dgamma_rad);
int osiv_get_tau(const osiv_handle* h, int32_t n_subsets, double kappa, double* tau);

/* Forward projection ("reprojection"):  l_i = sum_r a(i,r) mu_r  for the rays of
 * subset `subset` of `n_subsets` (subset < 0: all views; then n_subsets is ignored), where a(i,r) is
 * the exact length of ray i inside square pixel r (C2).
 * d_img [batch][ny][nx] -> d_sino [batch][V_S][C].  Asynchronous on cuda_stream. */
int osiv_forward(osiv_handle* h, const float* d_img, float* d_sino, int32_t batch,
                 int32_t subset, int32_t n_subsets, void* cuda_stream);

/* Matched backprojection ("estimation"):  g_r = sum_{i in S} a(i,r) s_i  with the same
 * a(i,r), computed as an atomic-free gather per pixel (C3).
 * d_sino [batch][V_S][C] -> d_img [batch][ny][nx].  Asynchronous on cuda_stream. */
int osiv_backward(osiv_handle* h, const float* d_sino, float* d_img, int32_t batch,
                  int32_t subset, int32_t n_subsets, void* cuda_stream);

/* Gradient of the smoothed isotropic total variation (C8):  d_grad[b] = dTV_eps/dmu (d_img[b]).
 * Both [batch][ny][nx].  Asynchronous on cuda_stream. */
int osiv_tv_gradient(osiv_handle* h, const float* d_img, float* d_grad, int32_t batch, double tv_eps,
                     void* cuda_stream);

/* The same gradient (C8) for callers that may not allocate device memory (code under CUDA graph capture, serving
 * loops, harnesses that forbid cudaMalloc): this call makes no cudaMalloc / cudaFree / allocating library call, on the
 * first call or any later one.  The padded copy of the images, which osiv_tv_gradient keeps in the handle's lazily
 * allocated workspace, lives in a fixed array of OSIV_STATIC_SCRATCH_BYTES that is part of the library image: every GPU
 * that loads libosiv holds it until the process exits.  osiv_create resolves the array's device address once per
 * device.  Needs batch * (ny + 2) * (nx + 8) * 4 bytes of it (one 1016 x 1016 slice, or three 512 x 512 slices);
 * a larger request returns OSIV_ERR_SCRATCH_LIMIT before anything is enqueued and leaves d_grad untouched.
 * The array is shared by every handle and every call on a device and keeps the last call's contents: each call clears
 * the part it uses first (the zero border is part of the operation), so calls in one stream are safe back to back,
 * but two calls that overlap on the GPU (different streams, or different handles on different streams) race on it --
 * serialise them.  Same arguments, results and asynchrony as osiv_tv_gradient (bit-identical output). */
#define OSIV_STATIC_SCRATCH_BYTES (4u << 20)
int osiv_tv_gradient_static(osiv_handle* h, const float* d_img, float* d_grad, int32_t batch, double tv_eps,
                            void* cuda_stream);

/* The ordered-subset iteration (PAPER.md:74 Eq. 3, :100-108 Eq. 4-5, :114, :118, :63, :140):
 *   mu(0) = mu0;  for n = 0 .. n_iters-1, m = n mod M:
 *     l = A_m mu(n);  ybar = b exp(-l);  r = (ybar - y)/b_ref;  D(n) = sum_i (l_i - ln(b_i/max(y_i,1)))^2
 *     lambda(n) by Eq. 4-5 on D(n) vs D(n-1) (lambda(0) = lambda0; floor lambda_min)
 *     mu(n+1) = max(mu(n) + lambda(n) tau_S (A_m^T r - (beta/M) dTV_eps(mu(n))), 0)
 * for `batch` independent slices that share geometry and subset order but own lambda, D and best image.
 *   d_counts    [batch][V][C] measured counts y
 *   d_blank     [C] blank-scan counts b per channel, or NULL to use blank_scalar for every channel;
 *               b_ref = mean_c b_c
 *   d_img_out   [batch][ny][nx] result
 *   h_trace     HOST pointer: NULL, or [batch][n_iters][2] doubles receiving (D(n), lambda(n)).
 * All work is enqueued on cuda_stream with no host round-trip inside the loop.  If h_trace is NULL the
 * call returns without synchronising (a non-finite monitor then shows only in the image; use
 * osiv_reconstruct_host or a trace to have it reported); otherwise it synchronises the stream, fills h_trace
 * and returns OSIV_ERR_NOT_FINITE if any slice's monitor was not finite.  tv_eps must be > 0.  A failed kernel
 * launch ends the call at that launch with OSIV_ERR_CUDA. */
int osiv_reconstruct(osiv_handle* h, const float* d_counts, const float* d_blank, float blank_scalar,
                     const osiv_params* params, int32_t batch, float* d_img_out, double* h_trace,
                     void* cuda_stream);

/* Same reconstruction with HOST buffers (the end-to-end call): copies h_counts (and h_blank) to the
 * device, runs osiv_reconstruct, copies the images back to h_img_out and synchronises the stream.
 * Pinned host memory makes the copies asynchronous but is not required.  Returns OSIV_ERR_NOT_FINITE (image
 * still delivered) if any slice's monitor was not finite, with or without h_trace. */
int osiv_reconstruct_host(osiv_handle* h, const float* h_counts, const float* h_blank, float blank_scalar,
                          const osiv_params* params, int32_t batch, float* h_img_out, double* h_trace,
                          void* cuda_stream);

/* =====================================================================================================
 * DIAGNOSTICS -- not part of the method.  Launch accounting, A/B switches and per-kernel timing used by the
 * tests and by bench.py's roofline report; a caller who only reconstructs needs none of them.
 * ===================================================================================================== */

/* Number of CUDA kernels this handle has launched since osiv_create (for launch accounting). */
int64_t osiv_launch_count(const osiv_handle* h);

/* Quarter-turn symmetry.  When the grid is square with nx % 4 == 0, n_views % 4 == 0 and a subset holds whole
 * orbits {v, v+V/4, v+V/2, v+3V/4} (V_S % 4 == 0), the kernels evaluate each chord weight once for the four
 * rotated (ray, pixel) pairs.  It is on by default wherever it applies; enable = 0 forces
 * the general kernels (used by the tests to compare the two paths).  Results differ only by rounding. */
int osiv_set_symmetry(osiv_handle* h, int32_t enable);

/* Launch overlap inside osiv_reconstruct.  By default (enable = 1) K1 and K2 are chained with programmatic
 * dependent launches: the next kernel's blocks become resident and run their data-independent prologue while the
 * current kernel drains, and wait on the device for its completion before they read its output.  enable = 0 uses
 * plain stream order (same results bit for bit; used by the tests and for A/B timing). */
int osiv_set_overlap(osiv_handle* h, int32_t enable);

/* One CUDA graph per call.  By default (enable = 1) osiv_reconstruct captures its launch sequence (set-up, n_iters x
 * (K1, K2) with their programmatic dependent edges, result) into a CUDA graph when a call repeats the previous call's
 * arguments (pointers, parameters, batch) and replays it with a single cudaGraphLaunch while they keep repeating (the
 * graphs of the two most recent argument sets are kept) (SURVEY.md section 7 step
 * 7); calls with forced_lambda or with per-kernel profiling, and drivers that cannot capture the sequence, enqueue launch
 * by launch.  enable = 0 always enqueues launch by launch (same results bit for bit; used by the tests).
 * osiv_graph_replays counts the graph launches made so far. */
int osiv_set_graph(osiv_handle* h, int32_t enable);
int64_t osiv_graph_replays(const osiv_handle* h);

/* Which K2 runs.  On the quarter-turn path with one slice per block (batch < 4, no stack), grids whose side is a multiple
 * of 8 and fans below 90 degrees, K2 is the kernel that stages each block's ray-table, residual and interval windows in
 * shared memory (csrc/osiv_back_staged.cuh) -- mode 0 (default): when one staging round holds the whole subset (otherwise
 * the general gather kernel is the faster one); mode 1: never (used by the tests to compare the two kernels); mode 2:
 * whenever the geometry allows, in as many rounds as it takes.  Results differ only by rounding order. */
int osiv_set_back_kernel(osiv_handle* h, int32_t mode);
/* *staged = 1 if osiv_reconstruct / osiv_backward with `n_subsets` subsets (<= 0: all views) and `batch` slices would
 * run the staged K2, else 0.  Host only. */
int osiv_get_back_kernel(const osiv_handle* h, int32_t n_subsets, int32_t batch, int32_t* staged);

/* Launch plan osiv_reconstruct would use for `n_subsets` subsets (<= 0: all views) and `batch` slices:
 * (independent slices: a stack with view_shift or tv_z never pairs slices)
 * out8 = {K1 orbit size (1 or 4), K1 line segments per ray, K1 blocks, K1 threads per block,
 *         K2 orbit size, K2 view shares per tile, K2 blocks, K2 threads per block}; both kernels run one block per SM
 *         and slice (launches with >= 4 slices: per pair of slices, in half-size blocks).  Host only. */
int osiv_get_plan(const osiv_handle* h, int32_t n_subsets, int32_t batch, int32_t* out8);

/* Per-kernel device timing for the roofline report.  While enabled (enable != 0), osiv_reconstruct records a
 * CUDA event on cuda_stream before and after every K1 (forward + residual + monitor partials) and K2
 * (step rule + backprojection + TV + update) launch and synchronises the stream at the end of the call to accumulate the
 * elapsed times; use it on extra steps, not on the steps whose throughput is reported.
 * osiv_get_profile returns the sums since the last osiv_set_profiling call: milliseconds and launch counts. */
int osiv_set_profiling(osiv_handle* h, int32_t enable);
int osiv_get_profile(const osiv_handle* h, double* ms_forward, int64_t* n_forward, double* ms_back, int64_t* n_back);

/* Phase timeline of the two hot kernels (only in the build made with -DOSIV_TRACE, `python -m
 * paper_1903_10088_b200.build --trace` -> libosiv_trace.so; the regular library returns OSIV_ERR_INVALID_ARG).
 * Every block of slice group 0 stamps its SM's cycle counter at its phase boundaries; h_out receives
 * [4][256][16] uint64: first index = (iteration & 1) * 2 + kernel (0 = K1, 1 = K2) of the last two iterations run on
 * the current device, second = block, third = {block start, before the dependent-launch wait, after it, end of the
 * main loop (latest warp), after the block barrier, block end (latest warp) -- all in SM cycles --, SM id, a mark
 * inside the prologue [cycles], the GPU's global nanosecond timer read at block start, unused...}.  n_entries must be
 * 4*256*16.  Synchronises the device.  Driver: `python -m paper_1903_10088_b200.timeline`. */
int osiv_debug_timeline(uint64_t* h_out, int32_t n_entries);

/* Index checks of the two hot kernels (only in the build made with -DOSIV_CHECKED, `python -m paper_1903_10088_b200.build
 * --check` -> libosiv_check.so; the regular library returns OSIV_ERR_INVALID_ARG).  Every gather index that relies on
 * clamping, zero padding or slack behind a row is compared with its buffer's extent on the device; h_out3 receives
 * {violations since the library was loaded, site number of the first one, warp-level checks made}.  Synchronises the device. */
int osiv_debug_checks(uint64_t* h_out3);

/* Micro-probes of the units that bound the two hot kernels (csrc/osiv_probes.cu): saturating loops
 * of one instruction kind at full occupancy on `device`, CUDA-event timed, best of 5 (takes about 0.1 s).
 * out8 = { FP32 TFLOP/s with FFMA (three register operands), FP32 TFLOP/s with FFMA2 (fma.rn.f32x2),
 *          G warp-instructions/s issued (FMA-pipe and ALU-pipe instructions alternating),
 *          GB/s read out of L2 (ld.global.cg over a 64 MiB buffer, every block streaming all of it),
 *          GB/s shared-memory reads (conflict-free LDS.128), GB/s L1-hit reads with LDG.128, GB/s L1-hit reads with
 *          LDG.32 (one 128-byte wavefront per warp instruction), number of SMs }.  Synchronises the device. */
int osiv_probe_peaks(int32_t device, double* out8);

#ifdef __cplusplus
}
#endif
#endif /* OSIV_H */
