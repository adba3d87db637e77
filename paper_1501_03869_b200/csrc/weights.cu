// weights.cu -- set-up kernels of the per-(sensor, pixel) weights (sm_100a; not part of the timed step).
//
// "Eq. 7 can be viewed as an approximation to the exact BP algorithm [5]" -- the universal back
// projection weights the term of detector i at point r_j by the solid angle the detector element subtends
// there, normalised by the total:  w_ij = dOmega_ij / Omega0_j,  dOmega_ij = n_i.(s_i - r_j) / |s_i - r_j|^3
// (n.e/|e|^2 in 2-D; <= 0 or |e| = 0 -> 0; R27).  The gather's WEIGHTED instantiations multiply
// every term by the table these kernels fill.
#include "pat_internal.h"

#include <cuda_runtime.h>

namespace {

__global__ void __launch_bounds__(256) fill_kernel(float *__restrict__ dst, int64_t n, float v) {
    for (int64_t q = (int64_t)blockIdx.x * 256 + threadIdx.x; q < n; q += (int64_t)gridDim.x * 256) dst[q] = v;
}

// One CTA per tile, thread = tile slot (padding slots repeat the tile's first pixel).  fp64 from the fp32 sensor
// data and the fp64 node coordinates, sensors in ascending order in both passes (the order the oracle sums in).
__device__ __forceinline__ double omega_term(const double (&r)[3], const float *__restrict__ s,
                                             const float *__restrict__ n, int ndim) {
    double dot = 0.0, d2 = 0.0;
    for (int d = 0; d < ndim; ++d) {
        const double e = __dsub_rn((double)__ldg(s + d), r[d]);
        dot = __dadd_rn(dot, __dmul_rn((double)__ldg(n + d), e));
        d2 = __dadd_rn(d2, __dmul_rn(e, e));
    }
    if (!(dot > 0.0) || !(d2 > 0.0)) return 0.0;
    return ndim == 3 ? __ddiv_rn(dot, __dmul_rn(d2, __dsqrt_rn(d2))) : __ddiv_rn(dot, d2);
}

__global__ void __launch_bounds__(kTilePix)
solid_angle_kernel(const double *__restrict__ pix, int64_t slots, const float *__restrict__ sens,
                   const float *__restrict__ nrm, int32_t nsens, int32_t ndim, float *__restrict__ w_t) {
    const int64_t tile = blockIdx.x, slot = tile * kTilePix + threadIdx.x;
    const double r[3] = {pix[slot], pix[slots + slot], pix[2 * slots + slot]};
    double total = 0.0;
    for (int32_t i = 0; i < nsens; ++i) total = __dadd_rn(total, omega_term(r, sens + 3 * i, nrm + 3 * i, ndim));
    for (int32_t i = 0; i < nsens; ++i) {
        const double om = omega_term(r, sens + 3 * i, nrm + 3 * i, ndim);
        w_t[(tile * nsens + i) * kTilePix + threadIdx.x] = total > 0.0 ? (float)__ddiv_rn(om, total) : 0.0f;
    }
}

}  // namespace

int pat_launch_fill(const PatLaunchCtx &ctx, float *dst, int64_t n, float value) {
    if (n <= 0) return 0;
    int64_t blocks = (n + 255) / 256;
    if (blocks > (int64_t)ctx.num_sms * 32) blocks = (int64_t)ctx.num_sms * 32;
    fill_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)ctx.stream>>>(dst, n, value);
    return (int)cudaGetLastError();
}

int pat_launch_solid_angle(const PatLaunchCtx &ctx, const double *pix, int64_t slots, const float *sens,
                           const float *nrm, int32_t nsens, int32_t ndim, float *w_t) {
    if (slots <= 0 || nsens <= 0) return 0;
    solid_angle_kernel<<<(unsigned)(slots / kTilePix), kTilePix, 0, (cudaStream_t)ctx.stream>>>(pix, slots, sens, nrm,
                                                                                              nsens, ndim, w_t);
    return (int)cudaGetLastError();
}
