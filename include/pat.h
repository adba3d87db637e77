/*
 * pat.h -- C-ABI of the B200-native phase-corrected back projection
 * (Wang & Jing, arxiv 1501.03869; hot path = Eq. 7).
 *
 * One GPU (sm_100a), fp32, no CPU fallback: on a machine without a usable
 * sm_100 device every call that needs the device returns PAT_ERR_UNSUPPORTED
 * or PAT_ERR_CUDA -- nothing is ever computed on the host in its place.
 *
 * Conventions
 *   - every entry point returns a pat_status; nothing throws, aborts or prints;
 *   - *out is written only on PAT_OK;
 *   - all arrays are caller-owned and only BORROWED: host arrays until the call
 *     returns, the device workspace until pat_destroy, traces/images until the
 *     work enqueued on `stream` has completed;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - a plan is not thread-safe; different plans may be used concurrently;
 *   - grids are node-centred, x fastest: linear index = ix + n[0]*(iy + n[1]*iz),
 *     node coordinates = origin + index*h.
 */
#ifndef PAT_H_
#define PAT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pat_plan pat_plan;               /* opaque, host-side */

typedef enum {
    PAT_OK = 0,
    PAT_ERR_INVALID_ARG = 1,
    PAT_ERR_BAD_STATE = 2,      /* e.g. pat_backproject before every sensor row was set */
    PAT_ERR_CUDA = 3,           /* CUDA runtime failure; text in pat_last_error */
    PAT_ERR_NOMEM = 4,          /* host allocation failed or workspace too small */
    PAT_ERR_UNSUPPORTED = 5     /* device is not sm_100 (no fallback path exists) */
} pat_status;

/* BP weighting b = wp*p - wd*t*dp/dt applied to the traces (reading R1). */
typedef enum {
    PAT_W_DELAY_SUM = 0,        /* p                         (plain delay-and-sum)          */
    PAT_W_PAPER = 1,            /* p - t*dp/dt               (Eq. 7 as printed) */
    PAT_W_UBP = 2,              /* 2p - 2t*dp/dt             (universal BP, ref. [5])        */
    /* Eq. 7 read literally ("p_i(t_ij) - t_ij * dp_i(t_ij)/dt"):
     * p AND dp/dt are each interpolated at the arrival time and the factor t is t_ij itself,
     *     term = wp*[(1-a)*p[k] + a*p[k+1]] - wd*(u + t0*fs)*[(1-a)*D[k] + a*D[k+1]],
     * which differs from modes 1, 2 by wd*a(1-a)*(D[k+1] - D[k]) per term (second order in 1/fs).
     * The pre-pass then writes TWO channels per frame (wp*p and -wd*D), so a frame occupies two
     * frame slots of the plan: nframes <= max_batch/2. */
    PAT_W_PAPER_EXACT = 3,      /* p(t_ij) - t_ij*dp/dt(t_ij)                                */
    PAT_W_UBP_EXACT = 4         /* 2 x PAT_W_PAPER_EXACT                                     */
} pat_weighting;

/* Regular grid of the speed-of-sound map / FMM domain. */
typedef struct {
    int32_t ndim;               /* 2 or 3 */
    int32_t n[3];               /* nodes per axis, x fastest; n[2] = 1 in 2-D */
    float   h;                  /* isotropic spacing [m] (paper: 0.195e-3 / 0.39e-3) */
    float   origin[3];          /* coordinates of node (0,0,0) [m] */
} pat_grid;

/* ---- device memory ---------------------------------------------------------------------------------------------
 * The library never owns device memory it did not get from the caller.  Two channels:
 *   1. the WORKSPACE of pat_plan_create: everything whose size follows from (nsens, npix, nt, max_batch) -- the
 *      re-tiled table, the weighted traces (three buffers), staging for host-side inputs;
 *   2. a PROVIDER installed with pat_set_device_allocator, for what depends on the data or on optional features:
 *        - the work list of every frame-count class used (built at the first call of the class): per class about
 *          16 bytes x (R + 1)/R per (tile, sensor) row that holds a valid pixel, R = rows per chunk (6 .. 24) -- 0.7 MB
 *          for configs[1] (43 008 rows), ~0.6 GB for configs[4] (33.5 M rows);
 *        - pat_set_pixel_weights / pat_compute_solid_angle_weights: a table of the size of the travel-time table;
 *        - pat_backproject_conventional: 12 bytes per tile slot + 12 per sensor, and 8 bytes per (tile, sensor) row of
 *          scratch while the row ranges of a new c0 are computed;
 *        - pat_set_roi_mask: 4 bytes per tile slot;  pat_compute_solid_angle_weights: 24 bytes per tile slot of scratch;
 *        - pat_eikonal_travel_times_device: one fp64 field per concurrently solved sensor (see there).
 *      alloc(bytes, user) must return DEVICE memory, 256-byte aligned, valid until release(ptr, bytes, user), or NULL
 *      (the call then fails with PAT_ERR_NOMEM).  Both are called on the calling thread, never from inside a stream
 *      capture (nothing is allocated on the call path once a class's work list exists).  The provider is
 *      process-wide; a plan keeps the one that was installed when it was created.  With no provider installed the
 *      library's shim (csrc/alloc.cu) uses cudaMalloc / cudaFree.  pat_get_stats reports what a plan holds. */
typedef void *(*pat_alloc_fn)(size_t bytes, void *user);
typedef void (*pat_free_fn)(void *ptr, size_t bytes, void *user);
pat_status pat_set_device_allocator(pat_alloc_fn alloc, pat_free_fn release, void *user);   /* both NULL: built-in shim */

typedef struct {
    int64_t workspace_bytes;        /* what pat_plan_workspace_bytes returned for this plan */
    int64_t provider_bytes;         /* device memory currently held through the provider */
    int64_t provider_bytes_peak;
    int64_t work_list_bytes;        /* part of provider_bytes: the work lists built so far */
    int64_t work_lists;             /* how many */
    double  work_list_build_seconds;/* host time spent building them (first call of a frame-count class) */
    int64_t kernel_launches, chained_calls;
} pat_stats;
pat_status pat_get_stats(const pat_plan *plan, pat_stats *out);

/* Bytes of DEVICE workspace a plan with these sizes needs (0 on invalid sizes).
 * Layout: re-tiled table (the dominant term, 4*nsens*npix rounded up to whole
 * 256-pixel tiles), per-row sample ranges, THREE buffers of weighted traces for max_batch frames (rounded up to
 * the frame-count class; consecutive calls rotate through them, see pat_backproject), staging for host-side
 * inputs, pixel permutation, counters. */
size_t pat_plan_workspace_bytes(const pat_grid *grid, int32_t nsens, int64_t npix,
                                int32_t nt, int32_t max_batch);

/* pat_plan_create -- the paper's problem statement.
 *   grid        FMM / c-map grid.
 *   c_map       HOST fp32 [n0*n1*n2] speed of sound [m/s]; copied into the plan for
 *               pat_compute_travel_times; may be NULL if the caller supplies tau itself.
 *               Every entry must be finite and > 0.
 *   sensor_xyz  HOST fp32 [nsens*3] sensor positions [m]; copied; may be NULL (as c_map).
 *   roi_index   HOST int64 [npix] strictly ascending linear node indices of the pixels to
 *               reconstruct ("the area within the skull"); NULL => all nodes
 *               (npix must then equal n0*n1*n2).
 *   nt, fs, t0  trace sampling: sample n is at time t0 + n/fs; nt >= 2, fs > 0.
 *   weighting   pat_weighting.
 *   max_batch   largest nframes a pat_backproject call will pass (>= 1).
 *   workspace   DEVICE memory, 256-byte aligned, >= pat_plan_workspace_bytes(...), owned by
 *               the caller (e.g. a torch tensor) and borrowed until pat_destroy.
 * Errors: NULL out/grid/workspace, bad sizes, non-ascending or out-of-grid roi_index,
 * bad c_map entry, misaligned or too small workspace -> PAT_ERR_INVALID_ARG (argument checks
 * run before any CUDA call); no sm_100 device -> PAT_ERR_UNSUPPORTED; CUDA failure -> PAT_ERR_CUDA. */
pat_status pat_plan_create(pat_plan **out, const pat_grid *grid, const float *c_map,
                           const float *sensor_xyz, int32_t nsens,
                           const int64_t *roi_index, int64_t npix,
                           int32_t nt, float fs, float t0,
                           int32_t weighting, int32_t max_batch,
                           void *workspace, size_t workspace_bytes);

/* pat_set_travel_times -- hand the plan rows of the tau table.
 *   tau   fp32 seconds, row-major [count][npix] (pixel order = roi_index order) for sensors
 *         [sensor_begin, sensor_begin+count).  HOST or DEVICE pointer (detected).
 * Converts to sample units u = fl32(fl32(tau - t0)*fs) and re-tiles the rows into the workspace
 * (spatially compact 256-pixel tiles) on `stream`; a host source is staged in pieces, so the call
 * returns after the host buffer has been consumed.  The call that completes the table (every
 * sensor row set) also reduces each (tile, sensor) row to its sample range and synchronises.  May be called repeatedly with disjoint sensor ranges (the 34 GB 3-D table).
 * Values that are negative, NaN, +-inf or beyond the record are LEGAL and contribute 0. */
pat_status pat_set_travel_times(pat_plan *plan, const float *tau, int32_t sensor_begin,
                                int32_t count, void *stream);

/* pat_backproject -- Eq. 7 for nframes frames:
 *     images[f][j] = sum_i (1-a)*b_fi[k] + a*b_fi[k+1],   u = fl32(fl32(tau_ij - t0)*fs),
 *     k = floor(u), a = u - k, terms with !(0 <= u < nt-1) contribute 0,
 *     b_fi[n] = wp*p_fi[n] - wd*(n + t0*fs)*D_fi[n]   (central differences, one-sided ends).
 *   traces  fp32 [nframes][nsens][nt]     images  fp32 [nframes][npix] (roi_index order)
 * Both DEVICE (16-byte aligned) or both HOST pointers (detected; host buffers should be
 * pinned for the copies to be asynchronous).  Enqueues weighting pre-pass + gather (+ the
 * copies for host buffers) on `stream` and returns without synchronising -- except for the first
 * call with a given frame-count class (1, 2, 3-4, 5-8, 9-16, 17+) after the table changed, which
 * builds that class's work list on the host (memory from the device-memory provider, size under "device memory"
 * above: 0.7 MB for configs[1], ~0.6 GB and 0.7 s for the 34 GB table of configs[4]) and uploads it synchronously;
 * that first call must therefore not happen inside a stream capture.
 * A plan is driven from ONE stream at a time, with the device it was created on current (another current device ->
 * PAT_ERR_INVALID_ARG); traces and images must not overlap.  HOST traces must be complete in memory when the call is
 * made: their copy runs on the plan's own copy stream and is NOT ordered behind work already enqueued on `stream`
 * (a pinned buffer still being filled by an earlier stream-ordered copy or callback would be read too early).
 * Consecutive calls (cross-call overlap).  Inside a stream capture -- the way to run a ~10 us frame without paying
 * a launch gap per kernel -- consecutive calls with DEVICE buffers are captured with explicit graph edges instead of
 * a linear chain: the gather of call j hangs on the gather of call j-1 by a programmatic edge (its CTAs take over
 * the SM slots that gather frees one by one) and the pre-pass of call j only on the gather of call j-3, so it runs
 * while the two gathers before it are still busy (the plan rotates through three buffers of weighted traces).
 * The library does this only when it can prove it safe at capture time: the capture's dependency set at the call
 * is exactly the previous call's gather (nothing foreign in between), and the images/traces of the call do not
 * overlap the images of the previous call (if they overlap those of the call before that -- a caller alternating
 * between two image buffers -- the pre-pass waits for that gather instead).  In every other case, and always outside
 * a capture, the call is ordered the ordinary way behind everything enqueued before it.  Work captured AFTER a call
 * depends on that call's gather, whose completion implies the completion of every earlier call of the run.
 * The results never depend on which way a call was captured.  pat_chained_calls counts the calls captured this way.
 * HOST buffers (the paper's timings include the transfers): the traces are copied on a
 * copy stream owned by the plan into one of two staging buffers and `stream` waits for that copy, so
 * the transfer of one call runs under the kernels of the previous call; everything is complete when
 * `stream` is (the host traces must stay untouched until then).  Inside a stream capture, or with
 * PAT_NO_PIPE=1, the copy is simply enqueued on `stream`.  Only the samples the table can touch are
 * transferred (pat_get_trace_window).
 * With PAT_W_PAPER_EXACT / PAT_W_UBP_EXACT the term is the one stated at pat_weighting (two channels per
 * frame through the same kernels) and nframes <= max_batch/2.
 * nframes = 0 is a no-op; nframes > max_batch (> max_batch/2 for the _EXACT weightings) ->
 * PAT_ERR_INVALID_ARG; tau rows missing -> PAT_ERR_BAD_STATE. */
pat_status pat_backproject(pat_plan *plan, const float *traces, float *images,
                           int32_t nframes, void *stream);

/* pat_backproject_conventional -- SURVEY.md 8(f) NEXT-3: the conventional back projection the paper
 * compares with ("t_ij is calculated analytically by assuming a constant speed"; PAPER.md:79:
 * c0 = 1560 m/s): Eq. 7 exactly as pat_backproject, but with tau_ij = |r_j - s_i| / c0 computed inside the
 * gather instead of read from the table (no 4*S*P-byte stream: the kernel is arithmetic-bound).  r_j is the
 * position of ROI node j on the plan's grid, s_i the plan's sensor position; fp32, one IEEE operation per
 * step: x_d = origin_d + i_d*h, e_d = x_d - s_d, d2 = (e_0^2 + e_1^2) + e_2^2, tau = sqrt(d2) * (1/c0).
 * The plan needs sensor_xyz but no travel-time table; tables and conventional calls may be mixed.
 * The first call for a given c0 (and frame-count class) builds work lists and synchronises `stream`.
 * Errors as pat_backproject; c0 not finite or <= 0 -> PAT_ERR_INVALID_ARG; no sensor_xyz -> PAT_ERR_BAD_STATE. */
pat_status pat_backproject_conventional(pat_plan *plan, const float *traces, float *images,
                                        int32_t nframes, float c0, void *stream);

/* pat_backproject_conventional_sweep -- SURVEY.md 8(f) NEXT-3, "a c0 sweep (autofocus-style)": the paper picks the
 * conventional BP's speed, c0 = 1560 m/s, "by an automatic sound speed selection", i.e. by reconstructing
 * with many candidate speeds.  One call reconstructs ONE frame with nc0 speeds:
 *     images[q][j] = pat_backproject_conventional(traces, c0[q])[j]        q = 0 .. nc0-1
 * bit-for-bit the same delays (tau = sqrt(d2) * (1/c0[q]), then the time -> sample map), but the distance of a
 * (pixel, sensor) pair is formed once for all speeds and the trace windows -- sized for the envelope of the delays
 * over [min c0, max c0] -- are staged once: the speeds play the role of the frame axis.
 *   traces  DEVICE fp32 [nsens][nt] (one frame)      images  DEVICE fp32 [nc0][npix]
 *   c0      HOST fp32 [nc0], finite and > 0, 1 <= nc0 <= PAT_MAX_SWEEP; read before the call returns
 * The first call with a new (min c0, max c0) builds row ranges and a work list (synchronises `stream`).
 * Errors as pat_backproject_conventional; host buffers, _EXACT weightings, pixel weights -> PAT_ERR_UNSUPPORTED. */
#define PAT_MAX_SWEEP 16
pat_status pat_backproject_conventional_sweep(pat_plan *plan, const float *traces, float *images,
                                              const float *c0, int32_t nc0, void *stream);

/* pat_set_roi_mask -- PAPER.md:81: "a specific region of interest can be selected for reconstruction to
 * further reduce the reconstruction time" -- without touching the uploaded table.
 *   mask   HOST uint8 [npix] in roi_index order, non-zero = reconstruct; NULL = all pixels again.
 * Subsequent pat_backproject / pat_backproject_conventional calls skip every 256-pixel tile that holds no
 * selected pixel (its part of the table is not read at all) and write 0 to unselected pixels; selected
 * pixels get exactly the values of an unmasked call.  Synchronises the device and drops the work lists
 * (rebuilt at the next call). */
pat_status pat_set_roi_mask(pat_plan *plan, const uint8_t *mask);

/* pat_set_pixel_weights -- SURVEY.md 8(f) NEXT-4: optional per-(sensor, pixel) factors w_ij that multiply every
 * term of Eq. 7,  images[f][j] = sum_i w_ij * [(1-a)*b_fi[k] + a*b_fi[k+1]]  (Eq. 7 "can be viewed
 * as an approximation to the exact BP algorithm [5]", whose terms carry the solid-angle factor
 * dOmega_ij / Omega0_j; any other apodisation or directivity table goes the same way).
 *   w   fp32 row-major [count][npix] (roi_index order) for sensors [sensor_begin, +count); HOST or DEVICE.
 * The first call allocates a library-owned table of the size of the travel-time table (4*nsens*npix bytes,
 * freed by pat_destroy), initialised to 1, and synchronises the device; rows not set stay 1.  From then on
 * pat_backproject and pat_backproject_conventional stream the weight rows next to the delays.
 * w = NULL with count = 0 removes the weights again (synchronises).
 * Errors: bad range / NULL with count > 0 -> PAT_ERR_INVALID_ARG; a plan with an _EXACT weighting ->
 * PAT_ERR_UNSUPPORTED; CUDA failure -> PAT_ERR_CUDA. */
pat_status pat_set_pixel_weights(pat_plan *plan, const float *w, int32_t sensor_begin, int32_t count,
                                 void *stream);

/* pat_compute_solid_angle_weights -- fills the weight table with the universal BP's factors [5] computed on the
 * device from the plan's geometry (fp64 from the fp32 inputs):
 *     w_ij = dOmega_ij / sum_i' dOmega_i'j ,   dOmega_ij = n_i . (s_i - r_j) / |s_i - r_j|^3   (3-D)
 *                                                          n_i . (s_i - r_j) / |s_i - r_j|^2   (2-D: subtended angle)
 * with r_j = origin + index*h the ROI node, s_i the plan's sensor position and n_i the unit normal of the
 * detection surface pointing away from the imaged region; a detector facing away (n.e <= 0) or sitting on the
 * node gets 0, a node no detector faces gets all zeros (R27).  With weighting PAT_W_UBP this is the
 * discretised universal back projection; for a ring much larger than the region w_ij -> 1/nsens.
 *   normals  HOST fp32 [nsens*3], finite; read before the call returns (synchronises `stream`).
 * Errors: NULL / non-finite normals -> PAT_ERR_INVALID_ARG; plan without sensor_xyz -> PAT_ERR_BAD_STATE;
 * _EXACT weighting -> PAT_ERR_UNSUPPORTED. */
pat_status pat_compute_solid_angle_weights(pat_plan *plan, const float *normals, void *stream);

/* Frees the host-side plan; never frees caller memory.  NULL is allowed. */
pat_status pat_destroy(pat_plan *plan);

/* ---- helpers ------------------------------------------------------------------------ */

/* Last error text of a plan (or of the last failed pat_plan_create when plan == NULL).
 * Never NULL; owned by the library. */
const char *pat_last_error(const pat_plan *plan);

/* The part of every trace the uploaded table can touch: samples [first, first+count) hold b[k], b[k+1] of every valid
 * (sensor, pixel) pair plus the +-1 halo of the central difference (rounded to whole 16-byte quads).  A
 * pat_backproject call with HOST buffers transfers only this part of every trace (one strided copy) when it is at
 * most 80 % of the record -- the paper's frame times include the transfers, and on configs[1] a pixel
 * inside the skull can only be reached by about a quarter of the 2048 samples; otherwise, or with
 * PAT_FULL_H2D=1, first = 0 and count = nt.  PAT_ERR_BAD_STATE until every tau row has been set. */
pat_status pat_get_trace_window(const pat_plan *plan, int32_t *first, int32_t *count);

/* Number of kernels of this library launched through `plan` so far (monotone counter). */
int64_t pat_kernel_launches(const pat_plan *plan);

/* Number of pat_backproject / pat_backproject_conventional calls on `plan` whose pre-pass was chained behind the
 * previous call's gather with a programmatic edge (see pat_backproject, "Consecutive calls"). */
int64_t pat_chained_calls(const pat_plan *plan);

/* Override the gather's shared-memory geometry (tuning / test hook; 0 = choose automatically):
 *   wr      longest trace window one (tile, sensor) row may occupy in shared memory, a power of two in
 *           [8, 4096] (clipped to the frame-count class's limit): a row whose pixels span more than
 *           wr-4 samples is processed in several segments;
 *   rows    (tile, sensor) rows per pipeline stage, 1..30;   stages  pipeline depth, 2..8.
 * A request that does not fit one CTA's shared memory for a given frame-count class is shrunk
 * (rows, then stages).  Takes effect at the next pat_backproject (the work lists are rebuilt).
 * Results do not depend on the tuning beyond fp32 summation order. */
pat_status pat_set_gather_tuning(pat_plan *plan, int32_t wr, int32_t rows, int32_t stages);

/* Measurement helper (bench.py's roofline leg).  mode 0 = off; 1 = pat_backproject brackets the
 * pre-pass and the gather with CUDA events on `stream` (this disables their programmatic overlap and
 * adds event overhead); 2 = pat_backproject launches ONLY the gather (b is whatever the last full
 * call left; the images are not zeroed -- timing only); 3 = only the pre-pass; 4 = neither: ONE kernel
 * that merely streams the step's footprint (u table + b in, images out; the images are garbage) -- the
 * "what does a plain read of these bytes cost here" line beside the roofline.  pat_get_profile
 * (mode 1) waits for the recorded events and returns the number of profiled calls and the summed
 * device milliseconds of each kernel since the last reset; any out pointer may be NULL.  At most
 * 65536 calls are recorded between resets. */
pat_status pat_set_profiling(pat_plan *plan, int32_t enable);
pat_status pat_get_profile(pat_plan *plan, int32_t reset, int64_t *calls, double *prepass_ms,
                           double *gather_ms);

/* pat_fmm_travel_times -- UNTIMED input preparation, HOST only: the
 * first-order upwind, heap-ordered narrow-band fast marching solve of |grad T| = 1/c from
 * each sensor (reciprocity); order = 2 uses the paper's Eq. 6 stencil with
 * first-order fallback.  Rows for sensors [sensor_begin, sensor_begin+count) of sensor_xyz:
 *   tau_out  HOST fp32 [count][npix], T computed in double and rounded once.
 *   nthreads OpenMP threads over sensors (<= 0: all cores).
 * A sensor outside the grid -> PAT_ERR_INVALID_ARG. */
pat_status pat_fmm_travel_times(const pat_grid *grid, const float *c_map,
                                const float *sensor_xyz, int32_t nsens,
                                const int64_t *roi_index, int64_t npix,
                                int32_t sensor_begin, int32_t count, int32_t order,
                                float *tau_out, int32_t nthreads);

/* Convenience: run pat_fmm_travel_times on the plan's own grid / c_map / sensors (both must
 * have been given to pat_plan_create) in chunks and feed every row to pat_set_travel_times. */
pat_status pat_compute_travel_times(pat_plan *plan, int32_t order, int32_t nthreads, void *stream);

/* pat_eikonal_travel_times_device -- SURVEY.md 8(f) NEXT-2: the same first-order upwind system
 * solved on the GPU, one CTA per sensor, many sensors at once, fp64 (csrc/eikonal.cu).
 * Default: a block-ordered fast iterative method -- the grid is cut into 8x8x8 (2-D: 16x16) blocks, the active
 * block with the smallest arrival time on its boundary is solved next (fast marching's causal order applied to
 * blocks) with Jacobi iterations in shared memory until nothing in it changes, and every face that changed wakes the
 * neighbour behind it; the solve ends when no block is active.  PAT_EIK_ALGO=sweep selects round 1's level-by-level
 * fast sweeping (also used when the grid has more blocks than one CTA's shared memory can track).  Either way the
 * fixed point is what fast marching computes; rows agree with pat_fmm_travel_times(order = 1) to fp32 rounding.
 *   c_map, sensor_xyz, roi_index   HOST, as for pat_fmm_travel_times.
 *   tau_out      DEVICE fp32 [count][npix], written on `stream`; the call synchronises `stream`.
 *   max_rounds   cap per sensor, in rounds (<= 0: 64).  A round is as much work as one visit of every block
 *                (sweeping: 2^ndim passes over the grid); every solve takes more than one.
 *   rounds_out   HOST, may be NULL: the largest number of rounds any sensor needed.
 * Temporary device memory (one fp64 field per concurrent sensor) comes from the device-memory provider and is
 * returned inside.  A sensor outside the grid / bad c_map -> PAT_ERR_INVALID_ARG; a sensor that did not converge
 * within max_rounds -> PAT_ERR_BAD_STATE (tau_out then holds upper bounds). */
pat_status pat_eikonal_travel_times_device(const pat_grid *grid, const float *c_map,
                                           const float *sensor_xyz, int32_t nsens,
                                           const int64_t *roi_index, int64_t npix,
                                           int32_t sensor_begin, int32_t count, float *tau_out,
                                           int32_t max_rounds, int32_t *rounds_out, void *stream);

/* Work counters of this thread's latest pat_eikonal_travel_times_device call (block-ordered solver; zeros after a
 * sweeping solve): blocks solved, Jacobi iterations, node updates, summed over the call's sensors.  Any pointer may be NULL. */
pat_status pat_eikonal_last_stats(int64_t *block_visits, int64_t *jacobi_iterations, int64_t *node_updates);

/* Convenience: pat_eikonal_travel_times_device on the plan's own grid / c_map / sensors, in chunks
 * through the plan's staging buffer, every row handed to pat_set_travel_times on the device. */
pat_status pat_compute_travel_times_gpu(pat_plan *plan, int32_t max_rounds, int32_t *rounds_out,
                                        void *stream);

/* pat_pixel_order -- host only, no CUDA call: the slot order of the tile-major table pat_plan_create builds for this
 * region.  perm_out[slot] = position in roi_index (0 .. npix-1), or -1 for the padding slots that fill the last tile;
 * perm_out holds ceil(npix/256)*256 entries.  A tile is 256 consecutive slots, a warp of the gather takes 32 of them.
 * The order is a recursive coordinate bisection (tiles, then halves down to groups of 8, Morton order inside), so that
 * tiles and warps are spatially compact whatever the region's shape (a region that cuts the blocks of a plain Morton
 * order -- the paper's "area within the skull", PAPER.md:79 -- would otherwise spread them over distant blocks);
 * plain_morton != 0 gives round 1's plain Morton order (what PAT_PLAIN_MORTON=1 selects at plan creation).
 * Errors: NULL / bad grid / index outside the grid -> PAT_ERR_INVALID_ARG. */
pat_status pat_pixel_order(const pat_grid *grid, const int64_t *roi_index, int64_t npix, int32_t plain_morton,
                           int32_t *perm_out);

/* ---- the entry point that allocates nothing -------------------------------------------------------------
 * Eq. 7 with the sample-time weightings, for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it): no plan, no workspace, no allocator.  The only
 * scratch of the path -- the weighted traces b the pre-pass writes and the gather reads -- is a file-scope
 * __device__ array of PAT_STATIC_MAX_SAMPLES floats (4 MiB) that every GPU holds from the moment it loads the
 * library until the process exits.  The call enqueues two kernels on `stream` and returns; it calls no cudaMalloc,
 * cudaFree or other allocating routine, copies nothing, and does not synchronise.
 *   tau      DEVICE fp32 [nsens][npix], seconds, row-major as pat_set_travel_times takes it (not retained)
 *   traces   DEVICE fp32 [nframes][nsens][nt]
 *   images   DEVICE fp32 [nframes][npix], written (not accumulated): needs no zeroing
 *   u = fl32(fl32(tau - t0)*fs), k = floor(u), a = u - k, terms with !(0 <= u < nt-1) contribute 0 -- the index rule
 *   and the per-term arithmetic of pat_backproject; the sum over sensors runs in another order (fp32), so the two
 *   agree within the tolerance of DESIGN.md section 3, not bit for bit.  A plain variant of the kernels: the tuned
 *   table layout and pipeline of the plan path are not here (expect a few times pat_backproject's step time).
 * Limit: nframes*nsens*nt <= PAT_STATIC_MAX_SAMPLES (the paper-scale frame, 512 x 2048, fits exactly); beyond it ->
 * PAT_ERR_INVALID_ARG with the numbers in the error text.  The array is shared by all calls on a device and keeps
 * the last call's contents; every call overwrites the part it reads, nothing in it must start at zero.  Calls that
 * OVERLAP on the GPU (different streams) race on the array; calls on one stream are ordered.
 * Errors: NULL / host pointers, sizes <= 0, nt < 2, non-finite fs or t0 -> PAT_ERR_INVALID_ARG; _EXACT weightings
 * -> PAT_ERR_UNSUPPORTED; not an sm_100 device -> PAT_ERR_UNSUPPORTED; CUDA failure -> PAT_ERR_CUDA.  The text is
 * returned by pat_backproject_static_last_error (per thread; never NULL). */
#define PAT_STATIC_MAX_SAMPLES (1 << 20)
pat_status pat_backproject_static(const float *tau, const float *traces, float *images, int32_t nsens,
                                  int64_t npix, int32_t nt, int32_t nframes, float fs, float t0,
                                  pat_weighting weighting, void *stream);
int64_t pat_backproject_static_max_samples(void);
const char *pat_backproject_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PAT_H_ */
