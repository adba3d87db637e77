// static_bp.cu -- pat_backproject_static: Eq. 7 for callers that must not allocate.
//
// Some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it) and cannot hand the library a workspace either.  This ONE entry point needs no plan, no
// workspace and no allocator: the only scratch the path has -- the weighted traces b = wp*p - wd*t*dp/dt
// that the pre-pass (H1) writes and the gather (H2-H4) reads -- lives in a file-scope __device__ array of
// PAT_STATIC_MAX_SAMPLES floats (4 MiB; every GPU that loads the library holds it until the process exits).
// The caller passes the inputs (tau, traces) and the output (images) as device pointers.
//
// It is a plain variant of the two kernels (thread-per-sample pre-pass, thread-per-(pixel, sensor quarter)
// gather reading tau rows as they are uploaded, [sensor][pixel] in seconds): the arithmetic of every term is
// the product path's (same fp32 operations for u, k, a, b and the interpolation; only the order of the sum
// over sensors differs), the tuned table layout, work lists and TMA pipeline of pat_backproject are not here.
// No existing code path is touched.
//
// The array is shared by every call on a device and keeps the last call's contents.  Nothing in it has to
// start at zero: a call overwrites all nframes*nsens*nt entries it later reads, and the images are written,
// not accumulated.  Two calls that overlap on the GPU (different streams, or one graph replayed on two
// streams) race on the array; calls on one stream are ordered.
#include "../../include/pat.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <mutex>

namespace {

constexpr int64_t kMaxSamples = PAT_STATIC_MAX_SAMPLES;

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: the address the
// kernels get comes from cudaGetSymbolAddress (resolve_scratch), once per device.
static __device__ __align__(256) float g_static_b[kMaxSamples];

thread_local char g_static_err[256] = "";

pat_status fail(pat_status st, const char *fmt, const char *a = "", long long x = 0, long long y = 0) {
    snprintf(g_static_err, sizeof(g_static_err), fmt, a, x, y);
    return st;
}

constexpr int kMaxDevices = 64;
float *g_scratch_ptr[kMaxDevices];                       // device address of g_static_b on device d
std::atomic<bool> g_scratch_ok[kMaxDevices];
std::mutex g_scratch_mutex;

// Once per device, with that device current: the device address of the array (and that the device is sm_100).
pat_status resolve_scratch(float **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(PAT_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(PAT_ERR_UNSUPPORTED, "%sdevice ordinal %lld is beyond %lld", "", dev, kMaxDevices - 1);
    if (!g_scratch_ok[dev].load(std::memory_order_acquire)) {
        std::lock_guard<std::mutex> lock(g_scratch_mutex);
        if (!g_scratch_ok[dev].load(std::memory_order_relaxed)) {
            int major = 0;
            e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
            if (e != cudaSuccess) return fail(PAT_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
            if (major != 10) return fail(PAT_ERR_UNSUPPORTED, "%sthe device is sm_%lldx, this library holds sm_100a code only (no fallback)", "", major);
            float *ptr = nullptr;
            e = cudaGetSymbolAddress((void **)&ptr, g_static_b);
            if (e != cudaSuccess || ptr == nullptr)
                return fail(PAT_ERR_CUDA, "cudaGetSymbolAddress(static scratch): %s", cudaGetErrorString(e));
            g_scratch_ptr[dev] = ptr;
            g_scratch_ok[dev].store(true, std::memory_order_release);
        }
    }
    *out = g_scratch_ptr[dev];
    return PAT_OK;
}

// ---- H1: b[f][i][n] = wp*p[n] - wd*(n + t0*fs)*D[n], D = central difference, one-sided at both ends
// (the operations of prepass.cu's weight_at, restated) ----------------------------------
__global__ void __launch_bounds__(256)
static_prepass_kernel(const float *__restrict__ traces, float *__restrict__ b, int64_t total, int32_t nt,
                      float wp, float wd, float t0fs) {
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int32_t n = (int32_t)(idx % nt);
    const float pn = __ldg(traces + idx);
    float out;
    if (wd == 0.0f) {
        out = wp * pn;
    } else {
        float D;
        if (n == 0)            D = __fsub_rn(__ldg(traces + idx + 1), pn);
        else if (n == nt - 1)  D = __fsub_rn(pn, __ldg(traces + idx - 1));
        else                   D = 0.5f * __fsub_rn(__ldg(traces + idx + 1), __ldg(traces + idx - 1));
        const float tn = __fadd_rn((float)n, t0fs);
        out = wp * __fmaf_rn(-tn, D, pn);                  // wp = wd is 1 or 2: the product is exact
    }
    b[idx] = out;
}

// ---- H2-H4: image[f][j] = sum_i (1-a)*b[f][i][k] + a*b[f][i][k+1], u = fl32(fl32(tau - t0)*fs), k = floor(u),
// a = u - k, terms with !(0 <= u < nt-1) skipped (R7, R8) ------------------
// Block = 64 pixels x 4 sensor quarters; a quarter takes sensors q, q+4, ...; the four partial sums meet in
// shared memory and ONE thread per pixel writes the image (no atomics, nothing to zero).
constexpr int kPix = 64, kParts = 4;

__global__ void __launch_bounds__(kPix * kParts)
static_gather_kernel(const float *__restrict__ tau, const float *__restrict__ b, float *__restrict__ images,
                     int32_t nsens, int64_t npix, int32_t nt, float fs, float t0) {
    __shared__ float part[kParts][kPix];
    const int lane_pix = threadIdx.x % kPix, q = threadIdx.x / kPix;
    const int64_t j = (int64_t)blockIdx.x * kPix + lane_pix;
    const int32_t f = blockIdx.y;
    const float *bf = b + (size_t)f * nsens * nt;
    const float ulim = (float)(nt - 1);
    float acc = 0.0f;
    if (j < npix) {
        for (int32_t i = q; i < nsens; i += kParts) {
            const float u = __fmul_rn(__fsub_rn(__ldg(tau + (size_t)i * npix + j), t0), fs);
            if (!(u >= 0.0f && u < ulim)) continue;       // NaN, +-inf, negative, beyond the record
            const float kf = floorf(u);
            const float a = __fsub_rn(u, kf);              // exact
            const float *row = bf + (size_t)i * nt + (int32_t)kf;
            acc = __fmaf_rn(a, row[1], __fmaf_rn(__fsub_rn(1.0f, a), row[0], acc));
        }
    }
    part[q][lane_pix] = acc;
    __syncthreads();
    if (q == 0 && j < npix)
        images[(size_t)f * npix + j] = __fadd_rn(__fadd_rn(part[0][lane_pix], part[1][lane_pix]),
                                                 __fadd_rn(part[2][lane_pix], part[3][lane_pix]));
}

bool on_device(const void *p) {
    cudaPointerAttributes at{};
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" {

int64_t pat_backproject_static_max_samples(void) { return kMaxSamples; }

const char *pat_backproject_static_last_error(void) { return g_static_err; }

pat_status pat_backproject_static(const float *tau, const float *traces, float *images, int32_t nsens, int64_t npix,
                                  int32_t nt, int32_t nframes, float fs, float t0, pat_weighting weighting,
                                  void *stream) {
    g_static_err[0] = 0;
    if (!tau || !traces || !images) return fail(PAT_ERR_INVALID_ARG, "%stau, traces and images must not be NULL");
    if (nsens <= 0 || npix <= 0 || nt < 2 || nframes <= 0)
        return fail(PAT_ERR_INVALID_ARG, "%sneed nsens > 0, npix > 0, nt >= 2, nframes > 0");
    if (!(fs > 0.0f) || !(fs < 3.0e38f) || !(t0 == t0) || !(t0 > -3.0e38f && t0 < 3.0e38f))
        return fail(PAT_ERR_INVALID_ARG, "%sfs must be finite and > 0, t0 finite");
    if (weighting != PAT_W_DELAY_SUM && weighting != PAT_W_PAPER && weighting != PAT_W_UBP)
        return fail(PAT_ERR_UNSUPPORTED, "%sonly the sample-time weightings PAT_W_DELAY_SUM, PAT_W_PAPER, PAT_W_UBP");
    if (nt > (1 << 23)) return fail(PAT_ERR_INVALID_ARG, "%snt beyond 2^23");
    const long long total = (long long)nframes * nsens * nt;
    if ((long long)nframes * nsens > kMaxSamples || total > kMaxSamples)
        return fail(PAT_ERR_INVALID_ARG,
                    "%snframes*nsens*nt = %lld samples exceed the static scratch of %lld floats "
                    "(PAT_STATIC_MAX_SAMPLES): fewer frames per call, or use a plan (pat_backproject)",
                    "", total, (long long)kMaxSamples);
    if (((uintptr_t)tau | (uintptr_t)traces | (uintptr_t)images) & 3u)
        return fail(PAT_ERR_INVALID_ARG, "%spointers must be 4-byte aligned");
    if (!on_device(tau) || !on_device(traces) || !on_device(images))
        return fail(PAT_ERR_INVALID_ARG, "%stau, traces and images must be DEVICE pointers (this entry point copies nothing)");
    const long long pix_blocks = (npix + kPix - 1) / kPix;
    if (pix_blocks > 0x7fffffffLL || nframes > 65535)
        return fail(PAT_ERR_INVALID_ARG, "%stoo many pixels or frames for one launch");
    float *scratch = nullptr;
    const pat_status st = resolve_scratch(&scratch);
    if (st != PAT_OK) return st;

    const float wp = weighting == PAT_W_UBP ? 2.0f : 1.0f;
    const float wd = weighting == PAT_W_DELAY_SUM ? 0.0f : wp;
    const float t0fs = (float)((double)t0 * (double)fs);
    cudaStream_t s = (cudaStream_t)stream;
    static_prepass_kernel<<<(unsigned)((total + 255) / 256), 256, 0, s>>>(traces, scratch, total, nt, wp, wd, t0fs);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PAT_ERR_CUDA, "pre-pass launch: %s", cudaGetErrorString(e));
    static_gather_kernel<<<dim3((unsigned)pix_blocks, (unsigned)nframes), kPix * kParts, 0, s>>>(
        tau, scratch, images, nsens, npix, nt, fs, t0);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PAT_ERR_CUDA, "gather launch: %s", cudaGetErrorString(e));
    return PAT_OK;
}

}  // extern "C"
