// eikonal.cu -- SURVEY.md 8(f) NEXT-2: the off-line travel-time solve on the GPU (sm_100a).
//
// T(r) from |grad T| = 1/c with the first-order upwind (Godunov) discretisation,
// one solve per sensor (reciprocity); "the off-line process needs to be repeated ... if
// the sensor positions are changed" (184.28 s on the paper's CPU).  The heap-ordered
// fast marching of fmm.cpp is serial per sensor; here the SAME discrete equations are solved by fast
// sweeping: Gauss-Seidel passes over the grid in the 2^ndim axis orderings, each pass run level by
// level (i' + j' (+ k') = const: the nodes of a level do not depend on one another), one CTA per
// sensor, many sensors at once.  Updates only ever lower T, so the iteration ends exactly when a
// whole round of 2^ndim passes changes nothing; the fixed point is the unique solution of the
// upwind system, i.e. the values fast marching produces.  Arithmetic: fp64, the update written with
// explicit round-to-nearest operations in the order fmm.cpp uses (no contraction), T rounded to
// fp32 once at the end -- the rows agree with pat_fmm_travel_times to the last bit or two.
// Only order = 1 (the `north_star` scheme); the paper's Eq. 6 second-order option stays on the CPU.
#include "pat_internal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <limits>
#include <vector>

namespace {

struct EikParams {
    int32_t n[3];
    int64_t stride[3];
    int64_t N;
    const double *sh;          // [N] slowness * h
    double *T;                 // [gridDim.x][N] one field per CTA
    const double *seed_val;    // [count][8]
    const int32_t *seed_node;  // [count][8], -1 = unused
    const int64_t *roi;        // [npix] or NULL (all nodes)
    int64_t npix;
    float *tau_out;            // [count][npix]
    int32_t count, max_rounds;
    int32_t *info;             // [0] = largest number of rounds any sensor took, [1] = sensors not converged
};

// Godunov update from the sorted upwind values a0 <= a1 <= a2 (inf = absent): the smallest root that
// is causal (same case analysis and operation order as fmm.cpp's solve_first_order).
template <int ND>
__device__ __forceinline__ double godunov(double a0, double a1, double a2, double sh) {
    const double T1 = __dadd_rn(a0, sh);
    if (ND < 2 || !(T1 > a1)) return T1;
    const double d = __dsub_rn(a0, a1);
    const double r2 = __dsub_rn(__dmul_rn(__dmul_rn(2.0, sh), sh), __dmul_rn(d, d));
    const double T2 = __dmul_rn(0.5, __dadd_rn(__dadd_rn(a0, a1), __dsqrt_rn(r2)));
    if (ND < 3 || !(T2 > a2)) return T2;
    const double S = __dadd_rn(__dadd_rn(a0, a1), a2);
    const double Q = __dadd_rn(__dadd_rn(__dmul_rn(a0, a0), __dmul_rn(a1, a1)), __dmul_rn(a2, a2));
    const double disc = __dsub_rn(__dmul_rn(S, S), __dmul_rn(3.0, __dsub_rn(Q, __dmul_rn(sh, sh))));
    if (disc < 0.0) return T2;
    return __ddiv_rn(__dadd_rn(S, __dsqrt_rn(disc)), 3.0);
}

template <int ND>
__device__ __forceinline__ bool relax(const EikParams &P, double *T, int32_t i, int32_t j, int32_t k) {
    const int64_t q = i + P.stride[1] * j + P.stride[2] * k;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    double a[3] = {inf, inf, inf};
    const int32_t idx[3] = {i, j, k};
#pragma unroll
    for (int d = 0; d < ND; ++d) {
        if (idx[d] > 0) a[d] = T[q - P.stride[d]];
        if (idx[d] + 1 < P.n[d]) a[d] = fmin(a[d], T[q + P.stride[d]]);
    }
    if (ND >= 2 && a[1] < a[0]) { const double t = a[0]; a[0] = a[1]; a[1] = t; }
    if (ND >= 3) {
        if (a[2] < a[1]) { const double t = a[1]; a[1] = a[2]; a[2] = t; }
        if (a[1] < a[0]) { const double t = a[0]; a[0] = a[1]; a[1] = t; }
    }
    if (!(a[0] < inf)) return false;
    const double Tn = godunov<ND>(a[0], a[1], a[2], P.sh[q]);
    if (Tn < T[q]) { T[q] = Tn; return true; }
    return false;
}

template <int ND>
__global__ void __launch_bounds__(1024)
eikonal_sweep_kernel(const EikParams P) {
    double *T = P.T + (int64_t)blockIdx.x * P.N;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const int32_t n0 = P.n[0], n1 = P.n[1], n2 = ND == 3 ? P.n[2] : 1;
    for (int32_t sidx = blockIdx.x; sidx < P.count; sidx += gridDim.x) {
        for (int64_t q = threadIdx.x; q < P.N; q += blockDim.x) T[q] = inf;
        __syncthreads();
        if (threadIdx.x < (1 << ND)) {
            const int32_t node = P.seed_node[sidx * 8 + threadIdx.x];
            if (node >= 0) T[node] = P.seed_val[sidx * 8 + threadIdx.x];
        }
        __syncthreads();
        int32_t round = 0;
        bool converged = false;
        while (round < P.max_rounds) {
            int changed = 0;
            for (int dir = 0; dir < (1 << ND); ++dir) {
                const bool r0 = dir & 1, r1 = dir & 2, r2 = dir & 4;
                const int32_t levels = n0 + n1 + n2 - 2;
                for (int32_t L = 0; L < levels; ++L) {
                    if (ND == 2) {
                        const int32_t lo = max(0, L - (n1 - 1)), hi = min(n0 - 1, L);
                        for (int32_t ip = lo + threadIdx.x; ip <= hi; ip += blockDim.x) {
                            const int32_t jp = L - ip;
                            changed |= relax<ND>(P, T, r0 ? n0 - 1 - ip : ip, r1 ? n1 - 1 - jp : jp, 0);
                        }
                    } else {
                        const int32_t klo = max(0, L - (n0 - 1) - (n1 - 1)), khi = min(n2 - 1, L);
                        const int32_t cnt = (khi - klo + 1) * n1;
                        for (int32_t e = threadIdx.x; e < cnt; e += blockDim.x) {
                            const int32_t kp = klo + e / n1, jp = e - (kp - klo) * n1, ip = L - kp - jp;
                            if (ip < 0 || ip >= n0) continue;
                            changed |= relax<ND>(P, T, r0 ? n0 - 1 - ip : ip, r1 ? n1 - 1 - jp : jp,
                                                 r2 ? n2 - 1 - kp : kp);
                        }
                    }
                    __syncthreads();
                }
            }
            ++round;
            if (!__syncthreads_or(changed)) { converged = true; break; }
        }
        if (threadIdx.x == 0) {
            atomicMax(P.info, round);
            if (!converged) atomicAdd(P.info + 1, 1);
        }
        float *row = P.tau_out + (int64_t)sidx * P.npix;
        for (int64_t j = threadIdx.x; j < P.npix; j += blockDim.x) row[j] = (float)T[P.roi ? P.roi[j] : j];
        __syncthreads();
    }
}

}  // namespace

extern "C" pat_status pat_eikonal_travel_times_device(const pat_grid *grid, const float *c_map,
                                                      const float *sensor_xyz, int32_t nsens,
                                                      const int64_t *roi_index, int64_t npix,
                                                      int32_t sensor_begin, int32_t count, float *tau_out,
                                                      int32_t max_rounds, int32_t *rounds_out, void *stream) {
    if (!grid || !c_map || !sensor_xyz || !tau_out) return PAT_ERR_INVALID_ARG;
    if (grid->ndim != 2 && grid->ndim != 3) return PAT_ERR_INVALID_ARG;
    if (!(grid->h > 0.0f)) return PAT_ERR_INVALID_ARG;
    if (nsens <= 0 || sensor_begin < 0 || count < 0 || sensor_begin > nsens - count) return PAT_ERR_INVALID_ARG;
    if (max_rounds <= 0) max_rounds = 64;
    const int nd = grid->ndim;
    EikParams P{};
    const double h = (double)grid->h;
    double org[3];
    P.N = 1;
    for (int d = 0; d < 3; ++d) {
        P.n[d] = d < nd ? grid->n[d] : 1;
        if (d < nd && P.n[d] < 2) return PAT_ERR_INVALID_ARG;
        org[d] = (double)grid->origin[d];
        P.stride[d] = P.N;
        P.N *= P.n[d];
    }
    if (P.N > (int64_t)std::numeric_limits<int32_t>::max()) return PAT_ERR_INVALID_ARG;
    if (npix < 0 || (!roi_index && npix != P.N)) return PAT_ERR_INVALID_ARG;
    if (rounds_out) *rounds_out = 0;
    if (count == 0 || npix == 0) return PAT_OK;

    std::vector<double> slow, sh, seed_val;
    std::vector<int32_t> seed_node;
    try {
        slow.resize((size_t)P.N); sh.resize((size_t)P.N);
        seed_val.assign((size_t)count * 8, 0.0); seed_node.assign((size_t)count * 8, -1);
    } catch (...) { return PAT_ERR_NOMEM; }
    for (int64_t q = 0; q < P.N; ++q) {
        const float c = c_map[q];
        if (!(c > 0.0f) || !std::isfinite(c)) return PAT_ERR_INVALID_ARG;
        slow[(size_t)q] = 1.0 / (double)c;
        sh[(size_t)q] = slow[(size_t)q] * h;
    }
    if (roi_index)
        for (int64_t j = 0; j < npix; ++j)
            if (roi_index[j] < 0 || roi_index[j] >= P.N) return PAT_ERR_INVALID_ARG;
    // source initialisation as in fmm.cpp: the corners of the sensor's cell get distance * slowness of the
    // node nearest to the sensor
    for (int32_t i = 0; i < count; ++i) {
        const float *sf = sensor_xyz + 3 * (int64_t)(sensor_begin + i);
        int64_t i0[3] = {0, 0, 0}, inr[3] = {0, 0, 0};
        double src[3] = {(double)sf[0], (double)sf[1], (double)sf[2]};
        for (int d = 0; d < nd; ++d) {
            const double g = (src[d] - org[d]) / h;
            if (!(g >= 0.0 && g <= (double)(P.n[d] - 1))) return PAT_ERR_INVALID_ARG;
            i0[d] = std::min<int64_t>((int64_t)std::floor(g), P.n[d] - 2);
            inr[d] = std::min<int64_t>((int64_t)std::floor(g + 0.5), P.n[d] - 1);
        }
        const double s_near = slow[(size_t)(inr[0] + P.stride[1] * inr[1] + P.stride[2] * inr[2])];
        for (int cn = 0; cn < (1 << nd); ++cn) {
            int64_t q = 0;
            double d2 = 0;
            for (int d = 0; d < nd; ++d) {
                const int64_t id = i0[d] + ((cn >> d) & 1);
                const double x = org[d] + (double)id * h - src[d];
                d2 += x * x;
                q += id * P.stride[d];
            }
            seed_node[(size_t)i * 8 + cn] = (int32_t)q;
            seed_val[(size_t)i * 8 + cn] = std::sqrt(d2) * s_near;
        }
    }

    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return PAT_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PAT_ERR_CUDA;
    const int threads = nd == 2 ? std::min(1024, std::max(128, (std::min(P.n[0], P.n[1]) + 31) / 32 * 32)) : 1024;
    const int per_sm = std::max(1, 2048 / threads);
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    int64_t slots = std::min<int64_t>(count, (int64_t)sms * per_sm);
    const int64_t mem_cap = (int64_t)(free_b / 2) / (P.N * 8);
    slots = std::max<int64_t>(1, std::min(slots, mem_cap));
    if (const char *ev = std::getenv("PAT_EIK_SLOTS")) slots = std::max<int64_t>(1, std::min<int64_t>(slots, std::atoi(ev)));

    cudaStream_t st = (cudaStream_t)stream;
    // scratch: one block from the caller's device-memory provider (alloc.cu), carved into
    // [slowness*h][T fields of the concurrent sensors][seed values][seed nodes][info][roi indices]
    const PatAllocator alloc = pat_current_allocator();
    auto up = [](size_t v) { return (v + 255) / 256 * 256; };
    const size_t o_sh = 0, o_T = o_sh + up((size_t)P.N * 8), o_sv = o_T + up((size_t)slots * P.N * 8),
                 o_sn = o_sv + up(seed_val.size() * 8), o_info = o_sn + up(seed_node.size() * 4), o_roi = o_info + 256,
                 total_bytes = o_roi + (roi_index ? up((size_t)npix * 8) : 0);
    PatDevBuf buf;
    if (!pat_dev_alloc(alloc, total_bytes, &buf)) return PAT_ERR_NOMEM;
    char *base = (char *)buf.p;
    double *d_sh = (double *)(base + o_sh), *d_T = (double *)(base + o_T), *d_sv = (double *)(base + o_sv);
    int32_t *d_sn = (int32_t *)(base + o_sn), *d_info = (int32_t *)(base + o_info);
    int64_t *d_roi = roi_index ? (int64_t *)(base + o_roi) : nullptr;
    auto cleanup = [&]() { pat_dev_free(alloc, &buf); };
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_sh, sh.data(), (size_t)P.N * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_sv, seed_val.data(), seed_val.size() * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_sn, seed_node.data(), seed_node.size() * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && roi_index)
        e = cudaMemcpyAsync(d_roi, roi_index, (size_t)npix * 8, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_info, 0, 8, st);
    if (e != cudaSuccess) { cudaStreamSynchronize(st); cleanup(); return PAT_ERR_CUDA; }
    P.sh = d_sh; P.T = d_T; P.seed_val = d_sv; P.seed_node = d_sn; P.roi = d_roi; P.npix = npix;
    P.tau_out = tau_out; P.count = count; P.max_rounds = max_rounds; P.info = d_info;
    if (nd == 2) eikonal_sweep_kernel<2><<<(unsigned)slots, threads, 0, st>>>(P);
    else         eikonal_sweep_kernel<3><<<(unsigned)slots, threads, 0, st>>>(P);
    e = cudaGetLastError();
    int32_t info[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpyAsync(info, d_info, 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cleanup();
    if (e != cudaSuccess) return PAT_ERR_CUDA;
    if (rounds_out) *rounds_out = info[0];
    return info[1] ? PAT_ERR_BAD_STATE : PAT_OK;       // a sensor hit max_rounds without converging
}
