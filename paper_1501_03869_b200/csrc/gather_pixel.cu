// gather_pixel.cu -- H2-H4 of the hot path, "pixel-lane" variant (sm_100a).
//
// Eq. 7: P(r_j) = sum_i b_i(t_ij), with t_ij the FMM arrival time.
//   H2  u = fl32(fl32(tau - t0)*fs), k = floor(u), a = u - k, valid iff 0 <= u < nt-1
//   H3  v = b[k] + a*(b[k+1]-b[k])                (one 8-byte load of the {b, d} pair)
//   H4  acc += v over the sensors; partial sums over sensor ranges meet in fp32 atomics.
//
// Mapping: one thread per pixel of a 256-pixel tile, FB frames in registers.  The tau table
// (the dominant HBM stream, 4 B per pixel*sensor) is NOT loaded through registers: each CTA
// owns a contiguous range of (tile, sensor) rows of the tile-major table and streams it into a
// shared-memory ring with 1-D bulk async copies (TMA, cp.async.bulk + mbarrier complete_tx),
// evict-first in L2, so the bytes in flight per SM are set by the ring depth and not by
// occupancy.  The weighted traces (L2-resident) are gathered through L1: the 32 pixels of a
// warp are a compact Morton block, so one warp-wide gather touches 1-3 cache lines.
#include "pat_internal.h"

#include <cuda_runtime.h>

namespace {

constexpr int kRowsPerChunk = 16;      // sensors per TMA chunk: 16 KB
constexpr int kStages = 3;             // ring depth: 48 KB in flight per CTA
constexpr int kThreads = kTilePix;

__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}

struct Chunk { int64_t row; int32_t nrows; };   // rows [row, row+nrows) of the (tile, sensor) space

// Next chunk starting at `cur`: at most kRowsPerChunk rows, never crossing a tile or `end`.
__device__ __forceinline__ Chunk next_chunk(int64_t cur, int64_t end, int32_t nsens) {
    const int64_t tile = cur / nsens;
    const int64_t tile_end = (tile + 1) * nsens;
    int64_t lim = end < tile_end ? end : tile_end;
    int64_t n = lim - cur;
    Chunk c;
    c.row = cur;
    c.nrows = (int32_t)(n < kRowsPerChunk ? n : kRowsPerChunk);
    return c;
}

template <int FB>
__global__ void __launch_bounds__(kThreads)
gather_pixel_kernel(const float *__restrict__ tau_t, const float2 *__restrict__ bd,
                    const int32_t *__restrict__ perm, float *__restrict__ images,
                    int32_t nsens, int64_t npix, int64_t total_rows, int32_t nt, int32_t nframes,
                    float fs, float t0) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *ring = reinterpret_cast<float *>(smem_raw);                       // [kStages][16][256]
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + (size_t)kStages * kRowsPerChunk * kTilePix * 4);

    const int tid = threadIdx.x;
    const int64_t row_begin = total_rows * blockIdx.x / gridDim.x;
    const int64_t row_end = total_rows * (blockIdx.x + 1) / gridDim.x;
    const int32_t f0 = blockIdx.y * FB;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // producer state (thread 0 only)
    int64_t pcur = row_begin;
    uint64_t policy = 0;
    if (tid == 0) {
        policy = policy_evict_first();
        for (int s = 0; s < kStages && pcur < row_end; ++s) {
            Chunk c = next_chunk(pcur, row_end, nsens);
            const uint32_t bytes = (uint32_t)c.nrows * kTilePix * 4;
            mbar_arrive_expect_tx(&full[s], bytes);
            bulk_g2s(ring + (size_t)s * kRowsPerChunk * kTilePix, tau_t + c.row * kTilePix, bytes, &full[s], policy);
            pcur += c.nrows;
        }
    }
#if __CUDA_ARCH__ >= 900
    // tau does not depend on the pre-pass; everything below reads bd / accumulates into images.
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif

    float acc[FB];
#pragma unroll
    for (int r = 0; r < FB; ++r) acc[r] = 0.0f;

    const uint32_t klim = (uint32_t)(nt - 1);
    int64_t cur = row_begin;
    int64_t cur_tile = row_begin < row_end ? row_begin / nsens : -1;
    int stage = 0;
    uint32_t phase = 0;

    auto flush = [&](int64_t tile) {
        const int32_t slot = __ldg(perm + tile * kTilePix + tid);
        if (slot >= 0) {
#pragma unroll
            for (int r = 0; r < FB; ++r)
                if (f0 + r < nframes) atomicAdd(images + (int64_t)(f0 + r) * npix + slot, acc[r]);
        }
#pragma unroll
        for (int r = 0; r < FB; ++r) acc[r] = 0.0f;
    };

    while (cur < row_end) {
        const Chunk c = next_chunk(cur, row_end, nsens);
        const int64_t tile = c.row / nsens;
        if (tile != cur_tile) { flush(cur_tile); cur_tile = tile; }
        const int32_t s0 = (int32_t)(c.row - tile * nsens);

        mbar_wait(&full[stage], phase);
        const float *st = ring + (size_t)stage * kRowsPerChunk * kTilePix + tid;
        const float2 *bd_s = bd + (int64_t)s0 * nt * nframes + f0;

#pragma unroll 4
        for (int j = 0; j < c.nrows; ++j) {
            const float tau = st[j * kTilePix];
            const float u = __fmul_rn(__fsub_rn(tau, t0), fs);           // ONE fp32 multiply
            const float t = __fadd_rd(u, 8388608.0f);                    // floor(u) + 2^23 for 0 <= u < 2^23
            const uint32_t k = (uint32_t)(__float_as_int(t) - 0x4B000000);
            const float a = __fsub_rn(u, __fsub_rn(t, 8388608.0f));      // u - floor(u), exact
            if (k < klim) {
                const float2 *src = bd_s + ((int64_t)j * nt + k) * nframes;
#pragma unroll
                for (int r = 0; r < FB; ++r) {
                    if (FB > 1 && f0 + r >= nframes) break;
                    const float2 v = __ldg(src + r);
                    acc[r] = __fmaf_rn(a, v.y, __fadd_rn(acc[r], v.x));
                }
            }
        }
        cur += c.nrows;
        __syncthreads();                                   // everyone is done with this stage
        if (tid == 0 && pcur < row_end) {
            Chunk pc = next_chunk(pcur, row_end, nsens);
            const uint32_t bytes = (uint32_t)pc.nrows * kTilePix * 4;
            mbar_arrive_expect_tx(&full[stage], bytes);
            bulk_g2s(ring + (size_t)stage * kRowsPerChunk * kTilePix, tau_t + pc.row * kTilePix, bytes,
                     &full[stage], policy);
            pcur += pc.nrows;
        }
        if (++stage == kStages) { stage = 0; phase ^= 1u; }
    }
    if (cur_tile >= 0) flush(cur_tile);
}

constexpr size_t kSmemBytes = (size_t)kStages * kRowsPerChunk * kTilePix * 4 + kStages * sizeof(uint64_t);

template <int FB>
int launch_fb(const PatLaunchCtx &ctx, const float *tau_t, const float *bd, const int32_t *perm,
              float *images, int32_t nsens, int64_t npix, int64_t ntiles, int32_t nt, int32_t nframes,
              float fs, float t0) {
    auto kern = gather_pixel_kernel<FB>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
    if (e != cudaSuccess) return (int)e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, kSmemBytes);
    if (e != cudaSuccess) return (int)e;
    if (per_sm < 1) per_sm = 1;
    const int64_t total_rows = ntiles * nsens;
    const int32_t groups = (nframes + FB - 1) / FB;
    int64_t gx = (int64_t)ctx.num_sms * per_sm / groups;
    if (gx < ctx.num_sms) gx = ctx.num_sms;
    const int64_t max_gx = (total_rows + 3) / 4;          // at least ~4 rows per CTA
    if (gx > max_gx) gx = max_gx;
    if (gx < 1) gx = 1;

    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)gx, (unsigned)groups);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
    cfg.stream = (cudaStream_t)ctx.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = ctx.use_pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelEx(&cfg, kern, tau_t, (const float2 *)bd, perm, images, nsens, npix, total_rows,
                           nt, nframes, fs, t0);
    return (int)e;
}

}  // namespace

int pat_launch_gather_pixel(const PatLaunchCtx &ctx, const float *tau_t, const float *bd,
                            const int32_t *perm, float *images, int32_t nsens, int64_t npix,
                            int64_t ntiles, int32_t nt, int32_t nframes, float fs, float t0) {
    if (nframes == 1) return launch_fb<1>(ctx, tau_t, bd, perm, images, nsens, npix, ntiles, nt, nframes, fs, t0);
    if (nframes == 2) return launch_fb<2>(ctx, tau_t, bd, perm, images, nsens, npix, ntiles, nt, nframes, fs, t0);
    return launch_fb<4>(ctx, tau_t, bd, perm, images, nsens, npix, ntiles, nt, nframes, fs, t0);
}
