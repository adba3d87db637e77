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

// The value written into tau_t for padding lanes: u = tau*fs is negative => contributes 0.
#define PAT_TAU_PAD (-1.0f)

struct PatDims {
    int32_t nsens = 0;
    int64_t npix = 0;
    int32_t nt = 0;
    int32_t max_batch = 0;
    int64_t ntiles = 0;
};

struct PatLayout {            // byte offsets into the caller's workspace
    size_t tau = 0;           // float  [ntiles][nsens][256]
    size_t bd = 0;            // float2 [nsens][nt][nframes]      {b[n], b[n+1]-b[n]}
    size_t perm = 0;          // int32  [ntiles*256]  slot -> position in roi list, -1 = pad
    size_t traces = 0;        // float  [max_batch][nsens][nt]    staging for host traces
    size_t images = 0;        // float  [max_batch][npix]         staging for host images
    size_t tau_stage = 0;     // float  [stage_rows][npix]        staging for host tau rows
    int64_t stage_rows = 0;
    size_t total = 0;
};

PatLayout pat_layout(const PatDims &d);

struct pat_plan {
    PatDims dims;
    PatLayout lay;
    pat_grid grid{};
    float fs = 0, t0 = 0;
    int32_t weighting = 1;
    float wp = 1, wd = 1;
    char *ws = nullptr;       // device workspace base (borrowed)
    int device = 0;
    int num_sms = 0;
    int variant = 0;          // 0 auto, 1 pixel-lane, 2 frame-lane
    bool use_pdl = true;
    std::vector<uint8_t> row_set;     // per sensor: tau row uploaded?
    int64_t rows_set = 0;
    std::vector<float> c_map;         // host copies for pat_compute_travel_times
    std::vector<float> sensors;
    std::vector<int64_t> roi;         // empty => all nodes
    int64_t launches = 0;
    bool profiling = false;
    std::vector<void *> prof_events;  // cudaEvent_t triples: before pre-pass, between, after gather
    std::string err;
};

// ---- kernel launchers (defined in the .cu files; all enqueue on `stream`) -------------
struct PatLaunchCtx {
    void *stream;
    int num_sms;
    bool use_pdl;
};

// tau rows [sensor_begin, +count) from src[count][npix] (device) into tau_t.
int pat_launch_retile(const PatLaunchCtx &ctx, const float *src, float *tau_t, const int32_t *perm,
                      int32_t nsens, int64_t npix, int64_t ntiles, int32_t sensor_begin, int32_t count);

// H1: weighting pre-pass (Eq. 7 integrand at the sample times):
//   traces[f][s][n] (fp32) -> bd[(s*nt + n)*nframes + f] = { b[n], b[n+1]-b[n] } (float2),
//   entry n = nt-1 is {0,0}.  Also zeroes images[nframes*npix] (the gather accumulates into it).
int pat_launch_prepass(const PatLaunchCtx &ctx, const float *traces, float *bd, float *images,
                       int32_t nsens, int32_t nt, int32_t nframes, int64_t npix,
                       float wp, float wd, float t0fs);

// H2-H4: the gather, pixel-lane variant (one thread per pixel, FB frames in registers).
int pat_launch_gather_pixel(const PatLaunchCtx &ctx, const float *tau_t, const float *bd,
                            const int32_t *perm, float *images, int32_t nsens, int64_t npix,
                            int64_t ntiles, int32_t nt, int32_t nframes, float fs, float t0);

#endif  // PAT_INTERNAL_H_
