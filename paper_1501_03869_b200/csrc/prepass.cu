// prepass.cu -- tau re-tiling (set-up) and the H1 weighting pre-pass (sm_100a).
//
// H1 (Eq. 7): the integrand p_i(t) - t*dp_i/dt evaluated at the sample times,
//   b[n] = wp*p[n] - wd*(n + t0*fs)*D[n],  D = central difference (one-sided at the ends),
// stored together with its forward difference so that the gather's linear interpolation
// (1-a)*b[k] + a*b[k+1] = b[k] + a*(b[k+1]-b[k]) is ONE 8-byte load and two FP ops.
#include "pat_internal.h"

#include <cuda_runtime.h>

namespace {

// ---- tau re-tiling: row-major [count][npix] -> tile-major [tile][sensor][256] -----------
__global__ void __launch_bounds__(256)
retile_kernel(const float *__restrict__ src, float *__restrict__ tau_t,
              const int32_t *__restrict__ perm, int32_t nsens, int64_t npix,
              int32_t sensor_begin, int32_t count) {
    const int64_t tile = blockIdx.x;
    const int32_t slot = perm[tile * kTilePix + threadIdx.x];
    for (int32_t r = blockIdx.y; r < count; r += gridDim.y) {
        float v = PAT_TAU_PAD;
        if (slot >= 0) v = __ldg(src + (int64_t)r * npix + slot);
        tau_t[(tile * nsens + sensor_begin + r) * kTilePix + threadIdx.x] = v;
    }
}

// ---- H1 -------------------------------------------------------------------------------
// b[n] for one trace (fp32).  p points at sample 0 of the trace.
__device__ __forceinline__ float weight_at(const float *__restrict__ p, int32_t n, int32_t nt,
                                           float wp, float wd, float t0fs) {
    const float pn = __ldg(p + n);
    if (wd == 0.0f) return wp * pn;
    float D;
    if (n == 0)            D = __fsub_rn(__ldg(p + 1), pn);
    else if (n == nt - 1)  D = __fsub_rn(pn, __ldg(p + n - 1));
    else                   D = 0.5f * __fsub_rn(__ldg(p + n + 1), __ldg(p + n - 1));
    const float tn = __fadd_rn((float)n, t0fs);
    // wp*(p - tn*D): one rounding in the fma; wp = wd is 1 or 2 (exact scaling).
    return wp * __fmaf_rn(-tn, D, pn);
}

// Single-frame layout: thread per sample, fully coalesced 4-byte reads / 8-byte writes.
__global__ void __launch_bounds__(256)
prepass_b1_kernel(const float *__restrict__ traces, float2 *__restrict__ bd,
                  float *__restrict__ images, int64_t total /* nsens*nt */, int32_t nt,
                  int64_t npix, float wp, float wd, float t0fs) {
#if __CUDA_ARCH__ >= 900
    asm volatile("griddepcontrol.launch_dependents;");
#endif
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (int64_t q = gid; q < npix; q += stride) images[q] = 0.0f;
    for (int64_t q = gid; q < total; q += stride) {
        const int64_t s = q / nt;
        const int32_t n = (int32_t)(q - s * nt);
        const float *p = traces + s * nt;
        float2 out = make_float2(0.0f, 0.0f);
        if (n < nt - 1) {
            const float b0 = weight_at(p, n, nt, wp, wd, t0fs);
            const float b1 = weight_at(p, n + 1, nt, wp, wd, t0fs);
            out = make_float2(b0, __fsub_rn(b1, b0));
        }
        bd[q] = out;
    }
}

// Batched layout bd[(s*nt + n)*B + f]: a block handles 32 samples x all frames of one sensor;
// frames are the fastest thread index so the 8-byte stores of a (s, n) row are contiguous.
__global__ void __launch_bounds__(256)
prepass_batch_kernel(const float *__restrict__ traces, float2 *__restrict__ bd,
                     float *__restrict__ images, int32_t nsens, int32_t nt, int32_t nframes,
                     int64_t npix, float wp, float wd, float t0fs) {
#if __CUDA_ARCH__ >= 900
    asm volatile("griddepcontrol.launch_dependents;");
#endif
    {
        const int64_t stride = (int64_t)gridDim.x * gridDim.y * blockDim.x;
        const int64_t gid = ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * blockDim.x + threadIdx.x;
        for (int64_t q = gid; q < npix * nframes; q += stride) images[q] = 0.0f;
    }
    const int32_t s = blockIdx.y;
    const int64_t row_elems = (int64_t)nt * nframes;
    for (int64_t e0 = (int64_t)blockIdx.x * blockDim.x; e0 < row_elems; e0 += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = e0 + threadIdx.x;
        if (e >= row_elems) break;
        const int32_t n = (int32_t)(e / nframes);
        const int32_t f = (int32_t)(e - (int64_t)n * nframes);
        const float *p = traces + ((int64_t)f * nsens + s) * nt;
        float2 out = make_float2(0.0f, 0.0f);
        if (n < nt - 1) {
            const float b0 = weight_at(p, n, nt, wp, wd, t0fs);
            const float b1 = weight_at(p, n + 1, nt, wp, wd, t0fs);
            out = make_float2(b0, __fsub_rn(b1, b0));
        }
        bd[(int64_t)s * row_elems + e] = out;
    }
}

}  // namespace

int pat_launch_retile(const PatLaunchCtx &ctx, const float *src, float *tau_t, const int32_t *perm,
                      int32_t nsens, int64_t npix, int64_t ntiles, int32_t sensor_begin, int32_t count) {
    if (count <= 0 || ntiles <= 0) return 0;
    dim3 grid((unsigned)ntiles, (unsigned)(count < 64 ? count : 64));
    retile_kernel<<<grid, kTilePix, 0, (cudaStream_t)ctx.stream>>>(src, tau_t, perm, nsens, npix,
                                                                  sensor_begin, count);
    return (int)cudaGetLastError();
}

int pat_launch_prepass(const PatLaunchCtx &ctx, const float *traces, float *bd, float *images,
                       int32_t nsens, int32_t nt, int32_t nframes, int64_t npix,
                       float wp, float wd, float t0fs) {
    cudaStream_t st = (cudaStream_t)ctx.stream;
    if (nframes == 1) {
        const int64_t total = (int64_t)nsens * nt;
        int64_t blocks = (total + 255) / 256;
        const int64_t cap = (int64_t)ctx.num_sms * 8;
        if (blocks > cap) blocks = cap;
        if (blocks < 1) blocks = 1;
        prepass_b1_kernel<<<(unsigned)blocks, 256, 0, st>>>(traces, (float2 *)bd, images, total, nt,
                                                            npix, wp, wd, t0fs);
    } else {
        const int64_t row_elems = (int64_t)nt * nframes;
        int64_t bx = (row_elems + 255) / 256;
        int64_t cap = ((int64_t)ctx.num_sms * 8 + nsens - 1) / nsens;
        if (cap < 1) cap = 1;
        if (bx > cap) bx = cap;
        dim3 grid((unsigned)bx, (unsigned)nsens);
        prepass_batch_kernel<<<grid, 256, 0, st>>>(traces, (float2 *)bd, images, nsens, nt, nframes,
                                                   npix, wp, wd, t0fs);
    }
    return (int)cudaGetLastError();
}
