/*
 * toi.h -- C ABI of libtoi: the B200-native (sm_100a) hot path of the Transient-Oriented
 * Imager (TOI, 2-D mode) of arxiv 2512.06254.
 *
 * One call images one time sample ("snapshot") of a Measurement Set:
 *
 *   uvw (metres) --SVD plane fit, rotation (section 3.1)-->
 *   (r1, r2) in wavelengths per channel
 *   --flags/weights/parallel-hand average (section 3.5)-->
 *   --gridding, inverse 2-D C2C FFT-->
 *   --grid correction, crop, 1/(omega Wsum) (Eqs. 7-8)--> dirty image
 *
 * All arithmetic runs in CUDA kernels of this library (+ cuFFT for the transform); there is
 * no CPU fallback.  The paper is silent on the gridding kernel, padding, grid correction and
 * uniform weighting: the readings taken are listed in DESIGN.md section 3 (G1..G19).
 *
 * Conventions
 *   - every function returns an int status (TOI_OK = 0, errors < 0); nothing throws or aborts;
 *   - the caller owns every buffer it passes in; the library only reads them;
 *   - the plan owns every workspace, ring and returned image pointer; nothing is allocated
 *     after toi_plan_create returns;
 *   - toi_image_snapshot only ENQUEUES work on a CUDA stream unless `info` is non-NULL;
 *   - a plan is not thread-safe; different plans are independent;
 *   - image layout: float32 [N][N] row-major, row j = t2 axis, column i = t1 axis,
 *     t1(i) = -beta (i - N/2), t2(j) = +beta (j - N/2)  (Eq. 9, 0-based).
 */
#ifndef TOI_H_
#define TOI_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct toi_plan toi_plan; /* opaque */

enum {
    TOI_OK = 0,
    TOI_ERR_INVALID_ARG = -1,
    TOI_ERR_CUDA = -2,
    TOI_ERR_CUFFT = -3,
    TOI_ERR_NOMEM = -4,
    TOI_ERR_DEGENERATE_GEOMETRY = -5, /* collinear baselines or V33 < 1e-6: no visibility plane */
    TOI_ERR_CALLBACK = -6,
    TOI_ERR_UNSUPPORTED = -7
};

enum { TOI_WEIGHT_NATURAL = 0, TOI_WEIGHT_UNIFORM = 1 };
enum { TOI_MEM_HOST = 0, TOI_MEM_DEVICE = 1 };
/* gridding kernels: SLIDING is the product (sliding 8x8 register window on even cells, groups of 4
 * lanes with two columns per lane, k_grid_pair8.cu); ATOMIC (one thread per sample, 98 global
 * float atomics, k_grid_atomic.cu) is the ncu comparison point the design replaces and a second,
 * structurally different implementation for the parity tests.  Both give the same image within
 * the parity bars. */
enum { TOI_GRIDDER_SLIDING = 0, TOI_GRIDDER_ATOMIC = 1 };

/* The paper's inputs (Measurement Set, image size, cell size) plus the knobs the
 * paper leaves open.  Zero selects the default of every optional field. */
typedef struct {
    int32_t n_baselines;        /* rows of one time sample (cross-correlations only) */
    int32_t n_channels;         /* CHAN_FREQ length */
    int32_t n_pols;             /* 1, 2 or 4 correlations per sample */
    int32_t pol_a, pol_b;       /* the two parallel hands, e.g. (0,3); equal => one hand */
    const double *chan_freq_hz; /* HOST, [n_channels], copied by toi_plan_create */
    int32_t image_size;         /* N, even, >= 16 */
    double cell_size_deg;       /* beta of Eq. 9, degrees */
    int32_t weighting;          /* TOI_WEIGHT_* */
    int32_t grid_size;          /* G: 0 -> 2N; even, >= N, <= 32768 */
    int32_t kernel_support;     /* W: 0 -> 7; only 7 is built */
    int32_t apply_jacobian;     /* 0 -> 1: divide by omega (Eq. 7); 2 -> do not */
    int32_t input_location;     /* TOI_MEM_*: where toi_image_snapshot's pointers live */
    int32_t image_ring_depth;   /* 0 -> 5; the image returned stays valid for
                                   depth-1 further snapshots */
    int32_t device;             /* CUDA ordinal */
    int32_t gridder;            /* TOI_GRIDDER_* */
    int32_t enable_3d;          /* 1: also allocate what toi_image_snapshot_3d needs (N*N complex
                                   accumulator, Bessel table, r3 range) */
    int32_t debug_keep_grid;    /* 1: also allocate the copies toi_debug_copy_grid / _density read */
    int32_t reserved[5];        /* must be 0 */
} toi_config;

/* Filled when `info` is passed (forces a stream synchronise). */
typedef struct {
    double V[9];                /* row-major transform, R = B V^T */
    double omega;               /* |V11 V22 - V21 V12| (Eq. 8) */
    double sing[3];             /* singular values of the centred baseline matrix */
    double wsum;                /* sum_q f_q w_I,q over gridded samples: Eq. 7's N_vis */
    int64_t n_gridded, n_off_grid, n_flagged;
    float ms_h2d, ms_planefit, ms_weight, ms_grid, ms_fft, ms_crop, ms_total;
    float ms_clear;             /* sparse clear of the gridding grid: only the 128x8-cell tiles this
                                   snapshot touched are zeroed again, after the first FFT pass has
                                   read the grid; not included in ms_fft */
    float ms_clear_density;     /* uniform weighting: the same for the density map (the rectangles
                                   under and opposite the marked tiles), a launch of its own in a
                                   call that asks for this info; 0 otherwise; not included in ms_fft */
} toi_snapshot_info;

/* Allocate everything: device input slots, gridding grid, FFT workspace, tile maps, image ring,
 * density, cuFFT plans, correction tables, streams and events (and, behind cfg.enable_3d /
 * cfg.debug_keep_grid, the buffers of the 3-D mode / of the debug exports).  Nothing is allocated
 * by any later call except toi_stream_set_output.  *out is NULL on failure. */
int toi_plan_create(const toi_config *cfg, toi_plan **out);
int toi_plan_destroy(toi_plan *plan);

/*
 * Image one snapshot.
 *   uvw_m    float64 [n_baselines][3]  UVW column, metres
 *   vis      complex64 [n_baselines][n_channels][n_pols]  DATA column (interleaved re, im)
 *   weights  float32 same shape, or NULL for unit weights (WEIGHT_SPECTRUM)
 *   flags    uint8 same shape (non-zero = flagged), or NULL (FLAG)
 *            all four live where cfg.input_location says (host: copied H2D on the stream;
 *            the host buffers must stay untouched until the stream reaches that point --
 *            pass `info` or call toi_plan_sync to be sure)
 *   cuda_stream  a cudaStream_t, or NULL for the plan's own compute stream
 *   d_image_out  receives a DEVICE pointer to float32 [N][N] inside the plan's image ring
 *   info     NULL, or filled after synchronising the stream.  Only calls with info != NULL record the
 *            timed events the ms_* fields are read from (a timed event between two kernels costs
 *            1-2 us of the stream's time: about 0.02 ms per snapshot)
 * Returns TOI_ERR_DEGENERATE_GEOMETRY only when it synchronises (info != NULL); otherwise a
 * degenerate snapshot yields a zero image and the status is reported by toi_plan_sync.
 * An all-flagged snapshot is TOI_OK with a zero image and wsum = 0.
 */
int toi_image_snapshot(toi_plan *plan, const double *uvw_m, const void *vis, const float *weights,
                       const uint8_t *flags, void *cuda_stream, float **d_image_out,
                       toi_snapshot_info *info);

/* Wait for everything the plan enqueued; returns the first deferred status since the last
 * sync (e.g. TOI_ERR_DEGENERATE_GEOMETRY, TOI_ERR_CUDA). */
int toi_plan_sync(toi_plan *plan);

/* Copy an image of the ring (as returned through d_image_out) to host memory; synchronous. */
int toi_copy_image_to_host(toi_plan *plan, const float *d_image, float *h_image);

/*
 * Streamed run (section 4): a depth-2 pinned host ring feeds a depth-2 device
 * input ring on a copy stream while the compute stream images the previous snapshot; events
 * chain the slots, the host never waits for compute.
 *
 * fill: called for idx = 0, 1, ...; `slot` holds plan-owned PINNED host buffers to write the
 *   snapshot into.  The callback may instead REPLACE any of the four pointers with its own
 *   host buffers (pinned for full speed), which must then stay valid and unchanged until
 *   the fill call for idx + 2 is made or the stream run returns.  weights/flags may be set to NULL.
 *   Return 0 = ok, 1 = end of data (no snapshot produced), < 0 = error (TOI_ERR_CALLBACK).
 * sink: called after snapshot idx has been ENQUEUED; d_image is valid in stream order on
 *   `cuda_stream` and stays valid for ring_depth-1 further snapshots.  info is NULL unless
 *   the stream was started with want_info != 0 (which synchronises every snapshot).
 */
typedef struct {
    double *uvw_m;
    void *vis;
    float *weights;
    uint8_t *flags;
} toi_snapshot_buffers;

typedef int (*toi_fill_fn)(void *user, int64_t idx, toi_snapshot_buffers *slot);
typedef int (*toi_sink_fn)(void *user, int64_t idx, const float *d_image, void *cuda_stream,
                           const toi_snapshot_info *info);

typedef struct {
    int64_t n_done;             /* snapshots imaged */
    double wall_s;              /* host wall clock of the whole run */
    double gpu_ms;              /* first H2D start -> last image done, CUDA events */
    double h2d_bytes;           /* total bytes copied host -> device */
    double h2d_ms_sum;          /* sum of per-snapshot H2D durations (events) */
    double compute_ms_sum;      /* sum of per-snapshot imaging durations (events) */
    double d2h_bytes;           /* total bytes copied device -> host (toi_stream_set_output.to_host) */
    double d2h_ms_sum;          /* sum of per-image D2H durations (events) */
} toi_stream_stats;

/*
 * Output side of the streamed run (the paper's `interpolate` and `copy_cpu` stages, PAPER.md:302-304,
 * 345, 355): what toi_image_stream delivers for every snapshot.
 *   product     TOI_OUT_TILTED: the dirty image on the tilted plane (default);
 *               TOI_OUT_REPROJECT_EXACT / _PAPER: that image re-projected to the (l, m) grid (see
 *               toi_reproject) with the snapshot's own V, into a second device ring of the plan's
 *               image_ring_depth (the interpolate stage owns the image ring)
 *   difference  1: deliver product(n) - product(n-1) instead; snapshot 0 has no
 *               predecessor and delivers its product to the device sink and nothing to the host sink
 *   to_host     1: copy every delivered image device -> host on a third stream through a depth-2
 *               PINNED ring (cudaMemcpyAsync only, events between the streams) and
 *               call host_sink(user, idx, h_image) once it has landed -- in index order, from the
 *               thread running toi_image_stream, up to two snapshots after idx was enqueued (all
 *               before toi_image_stream returns).  h_image is valid until the callback returns.
 *               Needs image_ring_depth >= 3 (the slot a D2H reads is never the one the next two
 *               snapshots write).  A negative return aborts the run (TOI_ERR_CALLBACK).
 * The device sink of toi_image_stream receives the delivered image (difference or product).
 * Everything this needs is allocated HERE, not in the loop.  NULL restores the default.
 */
enum { TOI_OUT_TILTED = 0, TOI_OUT_REPROJECT_EXACT = 1, TOI_OUT_REPROJECT_PAPER = 2 };
typedef int (*toi_host_sink_fn)(void *user, int64_t idx, const float *h_image);
typedef struct {
    int32_t product;
    int32_t difference;
    int32_t to_host;
    int32_t reserved[5];        /* must be 0 */
    toi_host_sink_fn host_sink; /* required when to_host */
    void *host_user;
} toi_stream_output;
int toi_stream_set_output(toi_plan *plan, const toi_stream_output *out);

int toi_image_stream(toi_plan *plan, int64_t n_snapshots, toi_fill_fn fill, void *fill_user,
                     toi_sink_fn sink, void *sink_user, int32_t want_info, toi_stream_stats *stats);

/*
 * Near-coplanar ("3-D") mode, PAPER.md:202-269 (section 3.4, Eqs. 17-27): the residual coordinate
 * r3 = rho3 s_c (third row of R = B V^T) is kept.  Its range is cut into n_slab equal slabs; inside
 * a slab the residual phase is expanded in K Chebyshev polynomials (Jacobi-Anger), so the image is
 *   I(t1,t2) = Re{ sum_p exp(i 2 pi r3_p t3) sum_k c_k(2 pi Delta_r3 t3) M_pk(t1,t2) } / (omega Wsum)
 * with t3(t1,t2) of Eq. 17, c_0 = J_0, c_k = 2 i^k J_k (Eq. 22) and each Chebyshev moment M_pk one
 * gridding (samples of slab p times T_k(s_q), Eq. 19) + inverse FFT + correction/crop -- n_slab * K
 * passes of the 2-D machinery.  Pixels outside the sphere constraint of Eq. 17 are NaN.
 *   n_slab, K   0 = chosen from the snapshot as the paper prescribes (Eqs. 25-27: alpha_target = 10;
 *               smallest K in {8, 16, 24, 32} whose sampled expansion error is below 1e-2), else
 *               taken as given (1 <= n_slab <= 1024, 1 <= K <= 64)
 *   info3       NULL or filled; info NULL or filled (counts, V, wsum; stage times are not split)
 * This call SYNCHRONISES the stream once (the slab layout needs the snapshot's r3 range and V on
 * the host).  Needs a plan created with cfg.enable_3d = 1 (TOI_ERR_UNSUPPORTED otherwise): nothing
 * is allocated here.  Readings G24-G26 of DESIGN.md.
 * Other arguments and the returned image as toi_image_snapshot.
 */
typedef struct {
    int32_t n_slab, K, n_passes, reserved;
    double phi_max;             /* Eq. 26 */
    double t3_max;              /* Eq. 25 over the image */
    double r3_min, r3_max;      /* wavelengths */
    double alpha_slab;          /* phi_max / n_slab */
    double expansion_error;     /* sampled max |exp(i a s) - sum_k c_k T_k| for the K used */
    float ms_total;
} toi_3d_info;
int toi_image_snapshot_3d(toi_plan *plan, const double *uvw_m, const void *vis, const float *weights,
                          const uint8_t *flags, void *cuda_stream, int32_t n_slab, int32_t K,
                          float **d_image_out, toi_3d_info *info3, toi_snapshot_info *info);

/*
 * Re-projection ("interpolate" stage, section 3.3 Eqs. 9-16, Appendix A): resample
 * a dirty image from the tilted (t1, t2) plane it was reconstructed on to the standard (l, m) grid
 * of the same size and cell size.  GATHER: output pixel (i, j) is the direction
 * l = -beta (i - N/2), m = +beta (j - N/2); its place on the tilted image is (Eq. 16)
 * p1' = N/2 - t1/beta, p2' = N/2 + t2/beta with
 *   TOI_REPROJECT_EXACT  t = V s, s = (l, m, n - 1), n = sqrt(1 - l^2 - m^2)      (Eqs. 3-4)
 *   TOI_REPROJECT_PAPER  t1 = l + xi z, t2 = m + eta z, z = 1 - n (Eq. 13),
 *                        xi = V31/V33, eta = V32/V33 (Eqs. 14-15; sign reading DESIGN.md G16),
 *                        the small-tilt reduction the paper evaluates
 * and the value is the bilinear interpolation of the four neighbouring pixels (fp64 coordinates,
 * fp32 values).  A position more than 1e-6 pixel outside [0, N-1]^2, or a direction outside the
 * SIN domain (l^2 + m^2 > 1), gives NaN.  Readings G20-G23 of DESIGN.md.
 *   d_image  DEVICE float32 [N][N], e.g. the pointer toi_image_snapshot returned
 *   V        HOST row-major 3x3, or NULL = the transform of the snapshot most recently enqueued
 *            by this plan (read on the device in stream order: enqueue on the same stream, before
 *            the next snapshot).  With NULL a degenerate snapshot gives an all-NaN image.
 *            A non-NULL V is staged in one plan-owned device buffer: use one stream for such calls.
 *   d_out    DEVICE float32 [N][N], caller-owned, must not alias d_image
 * Enqueues one kernel on cuda_stream (NULL = the plan's compute stream); does not synchronise.
 */
enum { TOI_REPROJECT_EXACT = 0, TOI_REPROJECT_PAPER = 1 };
int toi_reproject(toi_plan *plan, const float *d_image, const double *V, int32_t mode, void *cuda_stream,
                  float *d_out);

/* Difference image d_out = d_a - d_b of two snapshots (what the downstream transient search
 * consumes); DEVICE float32 [N][N] each, d_out may alias either input.  One kernel on
 * cuda_stream (NULL = the plan's compute stream); does not synchronise. */
int toi_difference(toi_plan *plan, const float *d_a, const float *d_b, void *cuda_stream, float *d_out);

/* Human-readable description of the last error of this plan (or of plan creation when plan is
 * NULL); the string is owned by the library. */
const char *toi_last_error(const toi_plan *plan);

/* Number of kernel launches (own kernels + cuFFT execs + memsets) the last snapshot enqueued. */
int toi_last_launch_count(const toi_plan *plan);

/* ---- debug / parity exports: not on the timed path --------------------------------------- */
/* Inject V (row-major 3x3, host) for subsequent snapshots instead of fitting it; NULL clears.
 * Index-parity protocol G5 of DESIGN.md. */
int toi_debug_set_transform(toi_plan *plan, const double *V);
/* Centre cells of the LAST snapshot's samples, recomputed from its (still resident) uvw:
 * int32 [n_baselines][n_channels] each, DEVICE pointers. */
int toi_debug_cell_indices(toi_plan *plan, int32_t *d_iu, int32_t *d_iv);
/* The LAST snapshot's grid before the FFT, complex64 [G][G], signed cell (kv, ku) stored CENTRED at
 * [kv + G/2][ku + G/2] (the layout the gridder writes; the (-1)^(n+m) this gives the FFT output is
 * undone in the correction kernel); DEVICE pointer.  Needs a plan created with cfg.debug_keep_grid = 1
 * and capture switched on with toi_debug_keep_grid(plan, 1) before imaging (costs one extra G*G copy
 * per snapshot, and one of the density map under uniform weighting). */
int toi_debug_keep_grid(toi_plan *plan, int32_t on);
int toi_debug_copy_grid(toi_plan *plan, void *d_grid_c64);
/* Uniform-weighting density of the LAST snapshot, float32 [G][G], same index convention. */
int toi_debug_copy_density(toi_plan *plan, float *d_density);

/* ---- allocation-free entry point ------------------------------------------------------------ */
/* Steps a1-a3 (DESIGN.md section 3 steps 1-5) without a plan and WITHOUT ANY ALLOCATION,
 * for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): plane fit of the snapshot's baselines, rotation, and the centre cell of every
 * (baseline, channel) sample -- bit-identical to what a plan computes (toi_debug_cell_indices).
 *   d_uvw_m       DEVICE, f64 [n_baselines][3], metres
 *   chan_freq_hz  HOST, f64 [n_channels], Hz, positive; n_channels <= TOI_STATIC_MAX_CHANNELS
 *                 (TOI_ERR_UNSUPPORTED beyond it: the scratch is a fixed-size array)
 *   grid_size     G in [2, 32768]; cell_size_deg the image cell, degrees
 *   cuda_stream   cudaStream_t or NULL; the work is enqueued on it, the call does not synchronise
 *                 (the copy of the channel table from pageable host memory may wait for the stream's
 *                 earlier work)
 *   d_iu, d_iv    DEVICE out, int32 [n_baselines][n_channels]: signed centre cells (TOI off-grid
 *                 samples keep their out-of-range index, as in toi_debug_cell_indices)
 *   d_fit_out     DEVICE out or NULL: 13 doubles, V[9] row-major, omega (Eq. 8), singular values[3]
 *   err, err_len  NULL / 0, or a buffer the error text is written to
 * The scratch (snapshot state + channel scale table, 256 B + 8 B x TOI_STATIC_MAX_CHANNELS) is a
 * file-scope __device__ array: every GPU that loads the library holds it until the process exits.
 * All calls share it and it keeps the last call's contents (nothing in it needs to start at zero: each
 * call rewrites what it reads).  Calls that OVERLAP ON THE GPU -- different streams, or several host
 * threads on one device -- race on it; calls on one stream are ordered by the stream.
 * Calls no cudaMalloc / cudaFree / allocating library routine.  Returns TOI_OK or an error < 0. */
#define TOI_STATIC_MAX_CHANNELS 32768
int toi_cell_indices_static(const double *d_uvw_m, int32_t n_baselines, const double *chan_freq_hz,
                            int32_t n_channels, int32_t grid_size, double cell_size_deg, void *cuda_stream,
                            int32_t *d_iu, int32_t *d_iv, double *d_fit_out, char *err, int32_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* TOI_H_ */
