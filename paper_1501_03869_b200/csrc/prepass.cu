// prepass.cu -- table re-tiling (set-up) and the H1 weighting pre-pass (sm_100a).
//
// H1 (Eq. 7): the integrand p_i(t) - t*dp_i/dt evaluated at the sample times,
//   b[n] = wp*p[n] - wd*(n + t0*fs)*D[n],  D = central difference (one-sided at the ends),
// written so that the window of samples a pixel tile can touch is ONE contiguous run for all frames of a
// group (a single bulk async copy in gather.cu): [group][sensor][sample][Bp] for Bp <= 2, blocked
// [group][sensor][sample/32][Bp][32] for Bp >= 4.
#include "pat_internal.h"

#include <cuda_runtime.h>

namespace {

// ---- table re-tiling: tau row-major [count][npix] -> u tile-major [tile][sensor][256] --------
// u = fl32(fl32(tau - t0)*fs): H2's time -> sample mapping, two fp32 roundings (R8),
// done once here instead of once per frame in the gather.
__global__ void __launch_bounds__(256)
retile_kernel(const float *__restrict__ src, float *__restrict__ u_t,
              const int32_t *__restrict__ perm, int32_t nsens, int64_t npix,
              int32_t sensor_begin, int32_t count, float fs, float t0) {
    const int64_t tile = blockIdx.x;
    const int32_t slot = perm[tile * kTilePix + threadIdx.x], first = perm[tile * kTilePix];
    for (int32_t r = blockIdx.y; r < count; r += gridDim.y) {
        // padding lanes of the last tile repeat the tile's first pixel: the row stays "all valid" (no
        // test in the gather's fast path) and the lane's sum is simply never written (perm = -1)
        const int32_t from = slot >= 0 ? slot : first;
        const float v = __fmul_rn(__fsub_rn(__ldg(src + (int64_t)r * npix + from), t0), fs);
        u_t[(tile * nsens + sensor_begin + r) * kTilePix + threadIdx.x] = v;
    }
}

// ---- H1 -----------------------------------------------------------------------------------
// b[n] from the staged samples p[n-1], p[n], p[n+1] (t points at p[n-1]).
__device__ __forceinline__ float weight_at(const float *t, int32_t n, int32_t nt, float wp, float wd, float t0fs) {
    const float pm = t[0], pn = t[1], pp = t[2];
    if (wd == 0.0f) return wp * pn;
    float D;
    if (n == 0)            D = __fsub_rn(pp, pn);
    else if (n == nt - 1)  D = __fsub_rn(pn, pm);
    else                   D = 0.5f * __fsub_rn(pp, pm);
    const float tn = __fadd_rn((float)n, t0fs);
    return wp * __fmaf_rn(-tn, D, pn);                     // wp*(p - tn*D); wp = wd is 1 or 2 (exact)
}

// Bp = 32 (interleaved layout [sensor][sample][32]): transposition through shared memory.
// Block = (sample chunk, sensor, frame group).  The chunk of every frame of the group is read
// coalesced along time into shared memory (+1 halo each side), then written frame-fastest.
__global__ void __launch_bounds__(256)
prepass_kernel(const float *__restrict__ traces, float *__restrict__ b, float *__restrict__ images,
               int32_t nsens, int32_t nt, int32_t nt4, int32_t nframes, int32_t log2_bp, int32_t ns,
               int64_t npix, float wp, float wd, float t0fs) {
    asm volatile("griddepcontrol.launch_dependents;");
    extern __shared__ float tile[];                        // [bp][ns + 3]
    const int32_t bp = 1 << log2_bp, pitch = ns + 3;
    const int32_t s = blockIdx.y, grp = blockIdx.z;
    const int32_t n_begin = blockIdx.x * ns;
    {
        const int64_t nblk = (int64_t)gridDim.x * gridDim.y * gridDim.z;
        const int64_t blk = ((int64_t)grp * gridDim.y + s) * gridDim.x + blockIdx.x;
        const int64_t tot = npix * nframes;
        for (int64_t q = blk * 256 + threadIdx.x; q < tot; q += nblk * 256) images[q] = 0.0f;
    }
    const int64_t obase = (((int64_t)grp * nsens + s) * nt4 + n_begin) * bp;
    // Interior block (full frame group, central differences everywhere, 16-byte aligned rows):
    // vector loads, no bounds tests, one thread per (sample, 4 frames) with a 16-byte store.
    const bool interior = bp >= 4 && (nt & 3) == 0 && n_begin >= 1 && n_begin + ns <= nt - 1 &&
                          (grp + 1) * bp <= nframes;
    if (interior) {
        const int32_t log2_q = 31 - __clz(ns >> 2);                 // ns is a power of two >= 4
        const float *base = traces + ((int64_t)(grp * bp) * nsens + s) * nt + n_begin;
        const int64_t fstride = (int64_t)nsens * nt;
        for (int32_t e = threadIdx.x; e < (bp << log2_q); e += 256) {
            const int32_t fl = e >> log2_q, q = e & ((1 << log2_q) - 1);
            const float4 v = __ldg(reinterpret_cast<const float4 *>(base + fl * fstride) + q);
            float *t = tile + fl * pitch + 1 + 4 * q;
            t[0] = v.x; t[1] = v.y; t[2] = v.z; t[3] = v.w;
        }
        if (threadIdx.x < 2 * bp) {
            const int32_t fl = threadIdx.x >> 1, side = threadIdx.x & 1;
            tile[fl * pitch + (side ? ns + 1 : 0)] = __ldg(base + fl * fstride + (side ? ns : -1));
        }
        __syncthreads();
        const int32_t log2_fq = log2_bp - 2;
        float4 *out4 = reinterpret_cast<float4 *>(b + obase);
        for (int32_t idx = threadIdx.x; idx < (ns << log2_fq); idx += 256) {
            const int32_t nl = idx >> log2_fq, fq = idx & ((1 << log2_fq) - 1);
            const float tn = __fadd_rn((float)(n_begin + nl), t0fs);
            const float *t = tile + (4 * fq) * pitch + nl;
            float o[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float pm = t[j * pitch], pn = t[j * pitch + 1], pp = t[j * pitch + 2];
                o[j] = wd == 0.0f ? wp * pn : wp * __fmaf_rn(-tn, 0.5f * __fsub_rn(pp, pm), pn);
            }
            out4[idx] = make_float4(o[0], o[1], o[2], o[3]);
        }
        return;
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int32_t fl = warp; fl < bp; fl += 8) {
        const int32_t f = grp * bp + fl;
        const float *p = traces + ((int64_t)f * nsens + s) * nt;
        for (int32_t j = lane; j < ns + 2; j += 32) {
            const int32_t n = n_begin - 1 + j;
            tile[fl * pitch + j] = (f < nframes && n >= 0 && n < nt) ? __ldg(p + n) : 0.0f;
        }
    }
    __syncthreads();
    const int32_t nloc = min(ns, nt4 - n_begin);
    for (int32_t idx = threadIdx.x; idx < (nloc << log2_bp); idx += 256) {
        const int32_t nl = idx >> log2_bp, fl = idx & (bp - 1);
        const int32_t n = n_begin + nl;
        float v = 0.0f;
        if (n < nt && grp * bp + fl < nframes) v = weight_at(tile + fl * pitch + nl, n, nt, wp, wd, t0fs);
        b[obase + idx] = v;
    }
}

// Bp = 4, 8, 16: the BLOCKED layout b[g][sensor][n/32][frame][32] (gather.cu, PPL == 3).  One thread per
// (frame, sensor, 4 consecutive samples): reads straight from the traces (coalesced along time, the +-1
// neighbours come from L1) and writes one 16-byte piece of a 128-byte block -- no transposition at all.
__global__ void __launch_bounds__(256)
prepass_blocked_kernel(const float *__restrict__ traces, float *__restrict__ b, float *__restrict__ images,
                       int32_t nsens, int32_t nt, int32_t ntb, int32_t nframes, int32_t log2_bp, int32_t groups,
                       int64_t npix, float wp, float wd, float t0fs) {
    asm volatile("griddepcontrol.launch_dependents;");
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x, nthr = (int64_t)gridDim.x * 256;
    for (int64_t q = gid; q < npix * nframes; q += nthr) images[q] = 0.0f;
    const int32_t bp = 1 << log2_bp, quads = ntb * 8;
    const int64_t per_frame = (int64_t)nsens * quads, total = per_frame * ((int64_t)groups << log2_bp);
    for (int64_t q = gid; q < total; q += nthr) {
        const int32_t f = (int32_t)(q / per_frame);
        const int64_t r = q - (int64_t)f * per_frame;
        const int32_t s = (int32_t)(r / quads), n0 = (int32_t)(r - (int64_t)s * quads) << 2;
        float4 o = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (f < nframes && n0 < nt) {
            const float *p = traces + ((int64_t)f * nsens + s) * nt;
            float w[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};    // p[n0-1 .. n0+4]
            if ((nt & 3) == 0) {                           // rows are 16-byte aligned: one vector load + 2 halo
                const float4 v = __ldg(reinterpret_cast<const float4 *>(p + n0));
                w[1] = v.x; w[2] = v.y; w[3] = v.z; w[4] = v.w;
                if (n0 > 0) w[0] = __ldg(p + n0 - 1);
                if (n0 + 4 < nt) w[5] = __ldg(p + n0 + 4);
            } else {
#pragma unroll
                for (int j = 0; j < 6; ++j) {
                    const int32_t n = n0 - 1 + j;
                    if (n >= 0 && n < nt) w[j] = __ldg(p + n);
                }
            }
            float *ov = reinterpret_cast<float *>(&o);
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if (n0 + j < nt) ov[j] = weight_at(w + j, n0 + j, nt, wp, wd, t0fs);
        }
        const int32_t g = f >> log2_bp, fl = f & (bp - 1);
        float *dst = b + (((((int64_t)g * nsens + s) * ntb + (n0 >> 5)) << log2_bp) + fl) * 32 + (n0 & 31);
        *reinterpret_cast<float4 *>(dst) = o;
    }
}

// Bp <= 2 (layout [sensor][sample][Bp]): one thread per 4 consecutive samples of all BP frames,
// straight from global memory (the +-1 neighbours come from L1), BP 16-byte stores.
template <int BP>
__global__ void __launch_bounds__(256)
prepass_small_kernel(const float *__restrict__ traces, float *__restrict__ b, float *__restrict__ images,
                     int32_t nsens, int32_t nt, int32_t nt4, int32_t nframes, int64_t npix, float wp, float wd,
                     float t0fs) {
    asm volatile("griddepcontrol.launch_dependents;");
    const int64_t gid = (int64_t)blockIdx.x * 256 + threadIdx.x, nthr = (int64_t)gridDim.x * 256;
    for (int64_t q = gid; q < npix * nframes; q += nthr) images[q] = 0.0f;
    const int32_t quads = nt4 >> 2;
    for (int64_t q = gid; q < (int64_t)nsens * quads; q += nthr) {
        const int32_t s = (int32_t)(q / quads), n0 = (int32_t)(q - (int64_t)s * quads) << 2;
        float o[4][BP];
#pragma unroll
        for (int f = 0; f < BP; ++f) {
            const float *p = traces + ((int64_t)f * nsens + s) * nt;
            float w[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};    // p[n0-1 .. n0+4]
            if (f < nframes) {
                if ((nt & 3) == 0) {                       // rows are 16-byte aligned: one vector load + 2 halo
                    const float4 v = __ldg(reinterpret_cast<const float4 *>(p + n0));
                    w[1] = v.x; w[2] = v.y; w[3] = v.z; w[4] = v.w;
                    if (n0 > 0) w[0] = __ldg(p + n0 - 1);
                    if (n0 + 4 < nt) w[5] = __ldg(p + n0 + 4);
                } else {
#pragma unroll
                    for (int j = 0; j < 6; ++j) {
                        const int32_t n = n0 - 1 + j;
                        if (n >= 0 && n < nt) w[j] = __ldg(p + n);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j)
                o[j][f] = (f < nframes && n0 + j < nt) ? weight_at(w + j, n0 + j, nt, wp, wd, t0fs) : 0.0f;
        }
        float4 *dst = reinterpret_cast<float4 *>(b + ((int64_t)s * nt4 + n0) * BP);
        const float *flat = &o[0][0];                      // [sample][frame] = the output order
#pragma unroll
        for (int v = 0; v < BP; ++v) dst[v] = make_float4(flat[4 * v], flat[4 * v + 1], flat[4 * v + 2], flat[4 * v + 3]);
    }
}

}  // namespace

int pat_launch_retile(const PatLaunchCtx &ctx, const float *src, float *u_t, const int32_t *perm,
                      int32_t nsens, int64_t npix, int64_t ntiles, int32_t sensor_begin, int32_t count,
                      float fs, float t0) {
    if (count <= 0 || ntiles <= 0) return 0;
    dim3 grid((unsigned)ntiles, (unsigned)(count < 64 ? count : 64));
    retile_kernel<<<grid, kTilePix, 0, (cudaStream_t)ctx.stream>>>(src, u_t, perm, nsens, npix,
                                                                  sensor_begin, count, fs, t0);
    return (int)cudaGetLastError();
}

int pat_launch_prepass(const PatLaunchCtx &ctx, const float *traces, float *b, float *images,
                       int32_t nsens, int32_t nt, int32_t nt4, int32_t nframes, int32_t bp,
                       int64_t npix, float wp, float wd, float t0fs) {
    if (bp <= 2) {
        const int64_t work = (int64_t)nsens * (nt4 >> 2);
        int64_t blocks = (work + 255) / 256;
        if (blocks > (int64_t)ctx.num_sms * 16) blocks = (int64_t)ctx.num_sms * 16;
        cudaStream_t st = (cudaStream_t)ctx.stream;
        if (bp == 1)
            prepass_small_kernel<1><<<(unsigned)blocks, 256, 0, st>>>(traces, b, images, nsens, nt, nt4, nframes, npix, wp, wd, t0fs);
        else
            prepass_small_kernel<2><<<(unsigned)blocks, 256, 0, st>>>(traces, b, images, nsens, nt, nt4, nframes, npix, wp, wd, t0fs);
        return (int)cudaGetLastError();
    }
    int log2_bp = 0;
    while ((1 << log2_bp) < bp) ++log2_bp;
    if (pat_gather_blocked(bp)) {
        const int32_t groups = (nframes + bp - 1) / bp, ntb = (nt + 31) / 32;
        const int64_t work = (int64_t)groups * bp * nsens * ntb * 8;
        int64_t blocks = (work + 255) / 256;
        if (blocks > (int64_t)ctx.num_sms * 32) blocks = (int64_t)ctx.num_sms * 32;
        prepass_blocked_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)ctx.stream>>>(traces, b, images, nsens, nt, ntb,
                                                                                      nframes, log2_bp, groups, npix, wp,
                                                                                      wd, t0fs);
        return (int)cudaGetLastError();
    }
    int32_t ns = 8192 / bp;                                // samples per block (a power of two)
    if (ns > 1024) ns = 1024;
    while (ns > 4 && ns > nt4) ns >>= 1;
    const int32_t groups = (nframes + bp - 1) / bp;
    dim3 grid((unsigned)((nt4 + ns - 1) / ns), (unsigned)nsens, (unsigned)groups);
    const size_t smem = (size_t)bp * (ns + 3) * sizeof(float);
    prepass_kernel<<<grid, 256, smem, (cudaStream_t)ctx.stream>>>(traces, b, images, nsens, nt, nt4, nframes,
                                                                log2_bp, ns, npix, wp, wd, t0fs);
    return (int)cudaGetLastError();
}
