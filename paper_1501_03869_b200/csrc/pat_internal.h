// pat_internal.h -- shared declarations of the product library (NOT part of the ABI).
#ifndef PAT_INTERNAL_H_
#define PAT_INTERNAL_H_

#include "../../include/pat.h"

#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

// ---- compile-time layout constants ---------------------------------------------------
// A "tile" is 256 spatially compact (Morton-ordered) ROI pixels; the tau table is stored
// tile-major, tau_t[tile][sensor][256], so that one (tile, sensor-range) block is a single
// contiguous run that a 1-D bulk async copy (TMA) can fetch.
constexpr int kTilePix = 256;

struct PatDims {
    int32_t nsens = 0;
    int64_t npix = 0;
    int32_t nt = 0;
    int32_t max_batch = 0;
    int64_t ntiles = 0;
};

struct PatLayout {            // byte offsets into the caller's workspace
    size_t tau = 0;           // float  [ntiles][nsens][256]   u = fl32(fl32(tau - t0)*fs), tile-major
    size_t meta = 0;          // int2   [ntiles*nsens]         {kmin, kmax} of each row
    size_t bd = 0;            // float  weighted traces b: [g][nsens][nt4][Bp] (Bp <= 2) or blocked [g][nsens][ntb][Bp][32]
    size_t bd2 = 0, bd3 = 0;  // float  two more b buffers: consecutive calls rotate, so the pre-pass of call j may run while
                              //        the gathers of calls j-1 and j-2 still read theirs (cross-call overlap, pat_api.cu)
    size_t sync = 0;          // uint32 [3][64] per b buffer: [0] pre-pass blocks done, [1] gather CTAs done, [32] b-ready flag
    size_t perm = 0;          // int32  [ntiles*256]  slot -> position in roi list, -1 = pad
    size_t traces = 0;        // float  [max_batch][nsens][nt]    staging for host traces
    size_t traces2 = 0;       // float  second staging buffer: the copy of call i+1 overlaps the kernels of call i
    size_t images = 0;        // float  [max_batch][npix]         staging for host images
    size_t tau_stage = 0;     // float  [stage_rows][npix]        staging for host tau rows
    int64_t stage_rows = 0;
    size_t total = 0;
};

PatLayout pat_layout(const PatDims &d);

// Shared-memory geometry of the gather for Bp frames per launch group (gather.cu).
struct PatGatherConfig {
    int bp = 0;               // frames per group: 1, 2, 4, ..., 64
    int wr = 0;               // longest window of one slot, samples (longer rows are split)
    int step = 0;             // longest k-range of one slot (longer rows are split into segments of this)
    int cap = 0;              // window units one stage holds for all its slots (samples; 32-sample blocks for Bp >= 4)
    int R = 0;                // slots per stage
    int stages = 0;
    uint32_t hdr_bytes = 0, stage_bytes = 0;
    bool onfly = false;       // work list of the conventional BP (k-ranges from the geometry, no table)
    bool exact = false;       // PAT_W_*_EXACT: the bp "frames" are channel pairs {wp*p, -wd*D} of bp/2 frames
    bool weighted = false;    // pat_set_pixel_weights: a stage holds R weight rows after its R u rows
    bool fastu = false;       // conventional BP, one frame, fast delays (gather.cu onfly_u_fast2d): its own instantiation
};

// Tuning / diagnostic knobs, read from the environment ONCE, in pat_plan_create (never on a call path):
// PAT_WR, PAT_R, PAT_STAGES, PAT_CAP, PAT_BUDGET_KB (shared-memory geometry), PAT_CHUNK_COST, PAT_SLOW_COST (cost
// model of the work-list dealer), PAT_DEBUG=1 (schedule summary on stderr), PAT_SCHED_DUMP=<file>.
struct PatTune {
    int wr = 0, R = 0, stages = 0, cap = 0, budget_kb = 0;
    int chunk_cost = 6, slow_cost = 5;
    bool debug = false;
    int chain_depth = 3;          // PAT_CHAIN_DEPTH (A/B): 3 = the pre-pass of call j hangs on the gather of call j-3, 2 = on j-2
    bool old_blocked_prepass = false;   // PAT_OLD_BLOCKED_PREPASS=1 (A/B)
    bool no_fast_delays = false;  // PAT_NO_FAST_DELAYS=1 (A/B): conventional BP always with the generic delay arithmetic
    std::string sched_dump;
};

// Conventional BP: tau = |r - s| / c0 computed inside the gather.
struct PatOnfly {
    const float *pix = nullptr;     // device [3][pix_stride] node coordinates per tile slot
    const float *sens = nullptr;    // device [nsens][3]
    int64_t pix_stride = 0;
    float inv_c0 = 0, t0 = 0, fs = 0;
    int32_t ndim = 2;
    int32_t nsweep = 0;                 // > 0: pat_backproject_conventional_sweep, one image per speed
    bool fast2d = false;                // 2-D, t0 = 0, every |r - s|^2 in [1e-30, 1e30]: the gather may use onfly_u_fast2d
    float sweep_inv_c0[PAT_MAX_SWEEP] = {};
};

// Device memory the library asks for on its own goes through the caller's provider (alloc.cu).
struct PatAllocator { pat_alloc_fn alloc = nullptr; pat_free_fn release = nullptr; void *user = nullptr; };
struct PatDevBuf { void *p = nullptr; size_t bytes = 0; };
PatAllocator pat_current_allocator();
bool pat_dev_alloc(const PatAllocator &a, size_t bytes, PatDevBuf *out, int64_t *held = nullptr, int64_t *peak = nullptr);
void pat_dev_free(const PatAllocator &a, PatDevBuf *buf, int64_t *held = nullptr);

// Host-built work list of one PatGatherConfig (built lazily; device memory from the caller's provider).
struct PatSchedule {
    PatGatherConfig cfg;
    int grid_x = 0;
    int64_t nchunks = 0;
    PatDevBuf buf;                    // one block: the three arrays below
    void *d_sched = nullptr;          // int4 [nchunks][R + 1]
    void *d_first = nullptr;          // int4 [grid_x][R + 1]: every CTA's first chunk again, indexed by CTA
    int32_t *d_cta_chunk = nullptr;   // int32 [grid_x + 1]
};

struct pat_plan {
    PatDims dims;
    PatLayout lay;
    pat_grid grid{};
    float fs = 0, t0 = 0;
    int32_t nt4 = 0;
    int32_t weighting = 1;
    float wp = 1, wd = 1;
    bool exact = false;       // PAT_W_PAPER_EXACT / PAT_W_UBP_EXACT: weight taken at t_ij, two channels per frame
    char *ws = nullptr;       // device workspace base (borrowed)
    int device = 0;
    int num_sms = 0;
    int prio_high = 0;                // greatest stream priority of the device (cudaDeviceGetStreamPriorityRange)
    int tune_wr = 0, tune_R = 0, tune_stages = 0;   // pat_set_gather_tuning overrides (0 = automatic)
    PatTune env;                                    // environment knobs as they were at pat_plan_create
    bool use_pdl = true;
    bool probes = false;              // PAT_ENABLE_PROBES=1 at create: pat_set_profiling's kernel-only modes 2-4 allowed
    int b_slot = 0;                   // which of the three b buffers the next call writes
    bool sync_dirty = false;          // a launch failed between pre-pass and gather: re-zero the counters first
    bool window_prepass = true;       // H1 only over the samples the table can touch (PAT_FULL_PREPASS=1: all)
    bool window_h2d = true;           // host traces: copy only the samples the table can touch (PAT_FULL_H2D=1: all)
    std::vector<uint8_t> row_set;     // per sensor: tau row uploaded?
    int64_t rows_set = 0;
    bool meta_valid = false;          // host_meta matches the uploaded table
    std::vector<int32_t> host_meta;   // {kmin, kmax} per row, host copy
    std::vector<PatSchedule> schedules;
    std::vector<float> c_map;         // host copies for pat_compute_travel_times
    std::vector<float> sensors;
    std::vector<int64_t> roi;         // empty => all nodes
    int64_t launches = 0;
    int64_t chained = 0;              // calls whose pre-pass was launched with a programmatic edge (launch chain)
    bool trace_file = false;                   // PAT_TRACE_FILE was set at create
    std::string trace_file_name;
    PatAllocator alloc;                        // the device-memory provider as it was at pat_plan_create
    int64_t dev_bytes = 0, dev_bytes_peak = 0; // device memory currently / at most held through it
    int64_t sched_builds = 0;                  // work lists built so far, and the host seconds that took
    double sched_build_seconds = 0.0;
    PatDevBuf trace_buf, onfly_buf, w_buf, mask_buf;
    unsigned long long *trace_dev = nullptr;   // PAT_TRACE_FILE diagnostic: timeline of the last gather launch
    int trace_ctas = 0;
    // host-buffer calls: H2D on an own copy stream into alternating staging buffers, so that the transfer
    // of one call runs under the kernels of the previous one
    void *copy_stream = nullptr;
    void *ev_h2d[2] = {nullptr, nullptr}, *ev_read[2] = {nullptr, nullptr};
    uint64_t host_calls = 0;
    // samples [need_lo, need_hi) of a trace are all the table can touch (k-ranges of every row plus the
    // derivative's +-1 halo, rounded to 4 samples): host-buffer calls transfer only that part of every trace
    int32_t need_lo = 0, need_hi = 0;        // table path; valid when meta_valid
    int32_t onfly_lo = 0, onfly_hi = 0;      // conventional BP, for onfly_c0
    // conventional BP (pat_backproject_conventional): geometry on the device, k-ranges for the current c0
    std::vector<int32_t> host_perm;   // tile slot -> ROI position (-1 = padding)
    float *d_pix = nullptr, *d_sens = nullptr;
    bool onfly_d2_in_range = false;         // every |r - s|^2 of the plan is inside [1e-30, 1e30] (onfly_meta_kernel)
    float onfly_c0 = 0, onfly_c0_hi = 0;   // speed (range, for a sweep) the row ranges below were computed for
    std::vector<int32_t> onfly_meta;
    // pat_set_pixel_weights / pat_compute_solid_angle_weights: per-(sensor, pixel) factors, tile-major like u_t
    float *d_w_t = nullptr;           // library-owned [ntiles][nsens][256], NULL = no weights
    // pat_set_roi_mask: tiles without a selected pixel leave the work lists; unselected pixels are not written
    std::vector<uint8_t> tile_active;   // empty = everything
    int32_t *d_perm_masked = nullptr;   // [ntiles*256] perm with the unselected pixels set to -1
    int profiling = 0;        // pat_set_profiling mode
    std::vector<void *> prof_events;  // cudaEvent_t triples: before pre-pass, between, after gather
    std::string err;
};

// ---- kernel launchers (defined in the .cu files; all enqueue on `stream`) -------------
struct PatLaunchCtx {
    void *stream;
    int num_sms;
    bool use_pdl;
    unsigned long long *pre_trace = nullptr;   // PAT_TRACE_FILE diagnostic: {pre-pass block 0 start, flag raised}
    int high_priority = 0;                     // the device's greatest stream priority (pre-pass launches)
    bool old_blocked_prepass = false;          // PAT_OLD_BLOCKED_PREPASS=1 at plan creation (A/B): round 1's blocked pre-pass kernel
};

// tau rows [sensor_begin, +count) from src[count][npix] (device) -> u_t (tile-major, u = (tau-t0)*fs).
int pat_launch_retile(const PatLaunchCtx &ctx, const float *src, float *u_t, const int32_t *perm,
                      int32_t nsens, int64_t npix, int64_t ntiles, int32_t sensor_begin, int32_t count,
                      float fs, float t0);

// {kmin, kmax} of every row of u_t (int2 [nrows]).
int pat_launch_row_meta(const PatLaunchCtx &ctx, const float *u_t, void *meta, int64_t nrows, int32_t nt);

// H1: weighting pre-pass (Eq. 7 integrand at the sample times):
//   traces[f][s][n] (fp32) -> b[((g*nsens + s)*nt4 + n)*bp + fl],  f = g*bp + fl; rows n >= nt and
//   frames f >= nframes are zero.  Also zeroes images[nframes*npix] (the gather accumulates into it).
// bp >= 4 writes the blocked layout b[((g*nsens + s)*ntb + n/32)*bp + fl][n%32] (ntb = ceil(nt/32)).
// exact (PAT_W_*_EXACT): bp counts CHANNELS, frame f owns channels 2f = wp*p[n] and 2f+1 = -wd*D[n].
int pat_launch_prepass(const PatLaunchCtx &ctx, const float *traces, float *b, float *images,
                       int32_t nsens, int32_t nt, int32_t nt4, int32_t nframes, int32_t bp,
                       int64_t npix, float wp, float wd, float t0fs, bool exact = false,
                       int32_t n_lo = 0, int32_t n_hi = INT32_MAX,    // only samples [n_lo, n_hi) of b are needed
                       uint32_t *ready = nullptr,                     // [0]: every block counts itself when its part of b / images is
                                                                      // written, the last one raises the flag [32]
                       int64_t nzero = -1);                           // image floats to zero (-1: nframes*npix)

// Measurement only (pat_set_profiling mode 4): stream a_bytes + c_bytes in, nout floats out.
int pat_launch_stream_probe(const PatLaunchCtx &ctx, const void *a, int64_t a_bytes, const void *c, int64_t c_bytes,
                            float *out, int64_t nout);

// H2-H4: the gather (gather.cu).
int pat_frames_per_group(int32_t nframes);
bool pat_gather_blocked(int bp);       // trace layout [sensor][n/32][frame][32] instead of [sensor][n][frame]
int pat_gather_wrmax(int bp);          // default / largest slot window for this frame-count class
PatGatherConfig pat_gather_config(int bp, int wr, int R, int stages, bool onfly, bool exact, bool weighted,
                                  const PatTune &env);      // 0 = choose automatically
size_t pat_gather_smem_bytes(const PatGatherConfig &c);
int pat_gather_occupancy(const PatGatherConfig &c, int *per_sm);
int pat_launch_gather(const PatLaunchCtx &ctx, const PatGatherConfig &c, const float *u_t, const float *b,
                      const void *sched, const void *first, const int32_t *cta_chunk, int grid_x, const int32_t *perm,
                      float *images, int32_t nsens, int64_t npix, int32_t nt, int32_t nt4, int32_t nframes,
                      unsigned long long *trace = nullptr,    // trace: per-CTA timeline, 8 x u64 per CTA, or NULL
                      const PatOnfly *onfly = nullptr,        // conventional BP: u computed in the kernel
                      float t0fs = 0.0f,                      // exact-time weightings: t0*fs
                      const float *w_t = nullptr,             // pixel weights [ntiles][nsens][256] (cfg.weighted)
                      uint32_t *ready = nullptr);             // counters of this call's b buffer: [0] pre-pass blocks done, [1] CTAs of
                                                              // this grid done, [32] "b ready" flag (NULL: b is already there)

// Set-up kernels of the pixel weights (weights.cu).
int pat_launch_fill(const PatLaunchCtx &ctx, float *dst, int64_t n, float value);
// Universal-BP solid-angle weights dOmega_ij / Omega0_j straight into the tile-major table: pix = double
// [3][slots] node coordinates per tile slot, sens / nrm = float [nsens][3] (all device).
int pat_launch_solid_angle(const PatLaunchCtx &ctx, const double *pix, int64_t slots, const float *sens,
                           const float *nrm, int32_t nsens, int32_t ndim, float *w_t);
int pat_launch_onfly_meta(const PatLaunchCtx &ctx, const PatOnfly &o, int32_t nsens, void *meta, int64_t nrows, int32_t nt,
                          int32_t *d2_out_of_range = nullptr);

#endif  // PAT_INTERNAL_H_
