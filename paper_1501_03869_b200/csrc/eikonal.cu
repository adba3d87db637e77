// eikonal.cu -- SURVEY.md 8(f) NEXT-2: the off-line travel-time solve on the GPU (sm_100a).
//
// T(r) from |grad T| = 1/c with the first-order upwind (Godunov) discretisation,
// one solve per sensor (reciprocity); "the off-line process needs to be repeated ... if
// the sensor positions are changed" (184.28 s on the paper's CPU).  The heap-ordered
// fast marching of fmm.cpp is serial per sensor; here the SAME discrete equations are solved by fast
// sweeping: Gauss-Seidel passes over the grid in the 2^ndim axis orderings, each pass run level by
// level (i' + j' (+ k') = const: the nodes of a level do not depend on one another), one CTA per
// sensor, many sensors at once (round 1; kept for A/B, PAT_EIK_ALGO=sweep) -- and, since round 2, by a
// block-ordered fast iterative method (further down) that only works where the front is.  Updates only
// ever lower T, so either iteration ends exactly when nothing can change any more; the fixed point is the
// unique solution of the upwind system, i.e. the values fast marching produces.  Arithmetic: fp64, the update written with
// explicit round-to-nearest operations in the order fmm.cpp uses (no contraction), T rounded to
// fp32 once at the end -- the rows agree with pat_fmm_travel_times to the last bit or two.
// Only order = 1 (the `north_star` scheme); the paper's Eq. 6 second-order option stays on the CPU.
#include "pat_internal.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <string>
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


// ---- block-ordered fast iterative method (round 2) -----------------------------------------------------------
// The sweeping kernel above visits every node in every pass (configs[4]: 26 rounds x 8 passes over 4.3 M nodes per
// sensor, each level a strided walk through a 34 MB field: 119 s for 4096 sensors, HBM-sector-bound).  The same
// discrete system -- T = min(seed, godunov(upwind neighbours)) at every node, updates only ever lower T, unique
// fixed point -- is solved here with work where the front is.  The grid is cut into blocks (8 x 8 x 8 nodes in 3-D,
// 16 x 16 in 2-D); a block is ACTIVE when a value on the far side of one of its faces changed since it was last
// solved, and carries as KEY the smallest such value.  One CTA per sensor repeatedly picks the active block with
// the smallest key (parallel arg-min over the keys in shared memory; ties go to the lower block index, so the order
// is deterministic) -- fast marching's causal order, applied to blocks instead of nodes, so that a block is mostly
// solved once its upwind neighbours are final -- stages the block and its one-node halo in shared memory, relaxes it
// with Jacobi iterations (read phase / write phase, a barrier between) until nothing in it changes, writes it back
// and hands every face on which a value changed to the neighbour behind it (key = min(key, smallest changed value)).
// The solve ends when no block is active.  Same fp64 update (godunov<ND>, explicit rn operations), same seeds,
// T rounded to fp32 once.
template <int ND> struct FimGeo {
    static constexpr int BX = ND == 3 ? 8 : 16, BY = ND == 3 ? 8 : 16, BZ = ND == 3 ? 8 : 1;
    static constexpr int NODES = BX * BY * BZ, THREADS = 256, NPT = NODES / THREADS;
    static constexpr int HX = BX + 2, HY = BY + 2, HZ = ND == 3 ? BZ + 2 : 1, HALO = HX * HY * HZ;
    static constexpr int MAX_ITERS = 96;                  // Jacobi iterations per visit; a block that hits it stays active
};

struct FimParams {
    EikParams e;
    int32_t nb[3];             // blocks per axis
    int32_t nblocks;
    int32_t max_iters;         // Jacobi iterations per visit; a block that hits the cap stays active
    unsigned long long *stat;  // [0] block visits, [1] Jacobi iterations, [2] node updates (diagnostic, PAT_EIK_STATS)
};

thread_local int64_t g_last_stats[3] = {0, 0, 0};        // of this thread's latest pat_eikonal_travel_times_device call

constexpr uint32_t kKeyInf = 0x7f800000u;                // +inf as float bits: keys are non-negative floats, ordered as integers

template <int ND>
__global__ void __launch_bounds__(256, ND == 3 ? 3 : 6)
eikonal_fim_kernel(const FimParams FP) {
    using G = FimGeo<ND>;
    const EikParams &P = FP.e;
    extern __shared__ __align__(16) unsigned char fim_smem[];
    double *Ts = reinterpret_cast<double *>(fim_smem);                            // [HALO]
    uint32_t *keys = reinterpret_cast<uint32_t *>(fim_smem + G::HALO * sizeof(double));   // [nblocks]
    __shared__ unsigned long long s_facemin[6], s_wbest[8];
    double *T = P.T + (int64_t)blockIdx.x * P.N;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const unsigned long long inf_bits = 0x7ff0000000000000ULL;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t n0 = P.n[0], n1 = P.n[1], n2 = ND == 3 ? P.n[2] : 1;
    const int32_t nbx = FP.nb[0], nby = FP.nb[1], nbz = ND == 3 ? FP.nb[2] : 1;
    // this thread's nodes inside a block (the same for every block)
    int lx[G::NPT], ly[G::NPT], lz[G::NPT], sidx_[G::NPT];
#pragma unroll
    for (int m = 0; m < G::NPT; ++m) {
        const int n = tid + G::THREADS * m;
        lx[m] = n % G::BX; ly[m] = (n / G::BX) % G::BY; lz[m] = n / (G::BX * G::BY);
        sidx_[m] = ND == 3 ? ((lz[m] + 1) * G::HY + (ly[m] + 1)) * G::HX + lx[m] + 1 : (ly[m] + 1) * G::HX + lx[m] + 1;
    }
    const unsigned long long visit_cap = (unsigned long long)P.max_rounds * (unsigned long long)FP.nblocks;
    for (int32_t sidx = blockIdx.x; sidx < P.count; sidx += gridDim.x) {
        for (int64_t q = tid; q < P.N; q += G::THREADS) T[q] = inf;
        for (int32_t b = tid; b < FP.nblocks; b += G::THREADS) keys[b] = kKeyInf;
        if (tid < 6) s_facemin[tid] = inf_bits;
        __syncthreads();
        if (tid == 0) {
            for (int c = 0; c < (1 << ND); ++c) {
                const int32_t node = P.seed_node[sidx * 8 + c];
                if (node < 0) continue;
                const double v = P.seed_val[sidx * 8 + c];
                T[node] = v;
                const uint32_t key = __float_as_uint(__double2float_rd(v));
                const int32_t i = node % n0, j = (node / n0) % n1, k = node / (n0 * n1);
                const int32_t bx = i / G::BX, by = j / G::BY, bz = ND == 3 ? k / G::BZ : 0;
                const int32_t self = bx + nbx * (by + nby * bz);
                // the seed's block and its face neighbours (a seed never changes, so nothing else would wake them)
                keys[self] = min(keys[self], key);
                if (bx > 0) keys[self - 1] = min(keys[self - 1], key);
                if (bx + 1 < nbx) keys[self + 1] = min(keys[self + 1], key);
                if (by > 0) keys[self - nbx] = min(keys[self - nbx], key);
                if (by + 1 < nby) keys[self + nbx] = min(keys[self + nbx], key);
                if (ND == 3 && bz > 0) keys[self - nbx * nby] = min(keys[self - nbx * nby], key);
                if (ND == 3 && bz + 1 < nbz) keys[self + nbx * nby] = min(keys[self + nbx * nby], key);
            }
        }
        __syncthreads();
        unsigned long long visits = 0, iters = 0, nups = 0;
        bool converged = false;
        while (visits < visit_cap) {
            // ---- the active block with the smallest key ----
            unsigned long long best = ~0ULL;
            for (int32_t b = tid; b < FP.nblocks; b += G::THREADS) {
                const uint32_t k = keys[b];
                if (k < kKeyInf) best = min(best, ((unsigned long long)k << 32) | (uint32_t)b);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, o));
            if (lane == 0) s_wbest[warp] = best;
            __syncthreads();
#pragma unroll
            for (int w = 0; w < 8; ++w) best = min(best, s_wbest[w]);
            if (best == ~0ULL) { converged = true; break; }
            const int32_t self = (int32_t)(uint32_t)best;
            const uint32_t self_key = (uint32_t)(best >> 32);
            const int32_t cbx = self % nbx, cby = (self / nbx) % nby, cbz = self / (nbx * nby);
            // ---- stage the block and its halo ----
            const int32_t gx0 = cbx * G::BX - 1, gy0 = cby * G::BY - 1, gz0 = ND == 3 ? cbz * G::BZ - 1 : 0;
            for (int s = tid; s < G::HALO; s += G::THREADS) {
                const int hx = s % G::HX, hy = (s / G::HX) % G::HY, hz = s / (G::HX * G::HY);
                const int32_t gx = gx0 + hx, gy = gy0 + hy, gz = gz0 + hz;
                const bool in = gx >= 0 && gx < n0 && gy >= 0 && gy < n1 && gz >= 0 && gz < n2;
                Ts[s] = in ? T[gx + P.stride[1] * gy + P.stride[2] * gz] : inf;
            }
            int64_t gq[G::NPT];
            double shv[G::NPT], cur[G::NPT], orig[G::NPT];
            bool valid[G::NPT];
#pragma unroll
            for (int m = 0; m < G::NPT; ++m) {
                const int32_t gx = gx0 + 1 + lx[m], gy = gy0 + 1 + ly[m], gz = ND == 3 ? gz0 + 1 + lz[m] : 0;
                valid[m] = gx < n0 && gy < n1 && gz < n2;
                gq[m] = gx + P.stride[1] * gy + P.stride[2] * gz;
                shv[m] = valid[m] ? P.sh[gq[m]] : 0.0;
            }
            __syncthreads();
#pragma unroll
            for (int m = 0; m < G::NPT; ++m) orig[m] = cur[m] = Ts[sidx_[m]];
            // ---- Jacobi iterations inside the block ----
            int it = 0, nup = 0;
            for (; it < FP.max_iters; ++it) {
                double nxt[G::NPT];
                int ch = 0;
#pragma unroll
                for (int m = 0; m < G::NPT; ++m) {
                    nxt[m] = cur[m];
                    if (!valid[m]) continue;
                    const int s = sidx_[m];
                    double a0 = fmin(Ts[s - 1], Ts[s + 1]);
                    double a1 = ND >= 2 ? fmin(Ts[s - G::HX], Ts[s + G::HX]) : inf;
                    double a2 = ND >= 3 ? fmin(Ts[s - G::HX * G::HY], Ts[s + G::HX * G::HY]) : inf;
                    if (ND >= 2 && a1 < a0) { const double t_ = a0; a0 = a1; a1 = t_; }
                    if (ND >= 3) {
                        if (a2 < a1) { const double t_ = a1; a1 = a2; a2 = t_; }
                        if (a1 < a0) { const double t_ = a0; a0 = a1; a1 = t_; }
                    }
                    if (!(a0 < cur[m])) continue;                     // T_new > a0 always: nothing upwind of this node
                    const double Tn = godunov<ND>(a0, a1, a2, shv[m]);
                    ++nup;
                    if (Tn < cur[m]) { nxt[m] = Tn; ch = 1; }
                }
                __syncthreads();                                          // every read of this iteration is done
#pragma unroll
                for (int m = 0; m < G::NPT; ++m)
                    if (nxt[m] < cur[m]) { cur[m] = nxt[m]; Ts[sidx_[m]] = nxt[m]; }
                if (!__syncthreads_or(ch)) break;
            }
            // ---- write back; every face on which a value changed wakes the neighbour behind it ----
#pragma unroll
            for (int m = 0; m < G::NPT; ++m) {
                if (valid[m] && cur[m] < orig[m]) {
                    T[gq[m]] = cur[m];
                    const unsigned long long vb = (unsigned long long)__double_as_longlong(cur[m]);   // >= 0: ordered as integers
                    if (lx[m] == 0) atomicMin(&s_facemin[0], vb);
                    if (lx[m] == G::BX - 1) atomicMin(&s_facemin[1], vb);
                    if (ly[m] == 0) atomicMin(&s_facemin[2], vb);
                    if (ly[m] == G::BY - 1) atomicMin(&s_facemin[3], vb);
                    if (ND == 3 && lz[m] == 0) atomicMin(&s_facemin[4], vb);
                    if (ND == 3 && lz[m] == G::BZ - 1) atomicMin(&s_facemin[5], vb);
                }
            }
            nups += (unsigned)nup;
            __syncthreads();
            if (tid == 0) {
                keys[self] = it >= FP.max_iters ? self_key : kKeyInf;
                const int32_t nbr[6] = {self - 1, self + 1, self - nbx, self + nbx, self - nbx * nby, self + nbx * nby};
                const bool has[6] = {cbx > 0, cbx + 1 < nbx, cby > 0, cby + 1 < nby, ND == 3 && cbz > 0, ND == 3 && cbz + 1 < nbz};
#pragma unroll
                for (int f = 0; f < 2 * ND; ++f) {
                    const unsigned long long vb = s_facemin[f];
                    s_facemin[f] = inf_bits;
                    if (vb != inf_bits && has[f])
                        keys[nbr[f]] = min(keys[nbr[f]], __float_as_uint(__double2float_rd(__longlong_as_double((long long)vb))));
                }
            }
            visits += 1;
            iters += (unsigned)min(it + 1, FP.max_iters);
            __syncthreads();
        }
        if (FP.stat) {
            if (tid == 0) { atomicAdd(FP.stat, visits); atomicAdd(FP.stat + 1, iters); }
            atomicAdd(FP.stat + 2, nups);
        }
        if (tid == 0) {
            atomicMax(P.info, 1 + (int32_t)(visits / (unsigned long long)FP.nblocks));   // "rounds": visits per block, rounded up
            if (!converged) atomicAdd(P.info + 1, 1);
        }
        float *row = P.tau_out + (int64_t)sidx * P.npix;
        for (int64_t j = tid; j < P.npix; j += G::THREADS) row[j] = (float)T[P.roi ? P.roi[j] : j];
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
    // algorithm: the block-structured fast iterative method unless PAT_EIK_ALGO=sweep asks for the level-by-level
    // fast sweeping of round 1 (kept for A/B) or the activity flags of the grid do not fit one CTA's shared memory
    const char *algo_env = std::getenv("PAT_EIK_ALGO");
    bool use_fim = !(algo_env && std::string(algo_env) == "sweep");
    const bool default_rounds = max_rounds <= 0;
    if (default_rounds) max_rounds = 64;
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
    FimParams FP{};
    size_t fim_smem = 0;
    {
        const int bx = nd == 3 ? FimGeo<3>::BX : FimGeo<2>::BX, by = nd == 3 ? FimGeo<3>::BY : FimGeo<2>::BY,
                  bz = nd == 3 ? FimGeo<3>::BZ : 1;
        FP.nb[0] = (P.n[0] + bx - 1) / bx; FP.nb[1] = (P.n[1] + by - 1) / by; FP.nb[2] = nd == 3 ? (P.n[2] + bz - 1) / bz : 1;
        const int64_t nblocks = (int64_t)FP.nb[0] * FP.nb[1] * FP.nb[2];
        const size_t halo = (size_t)(nd == 3 ? FimGeo<3>::HALO : FimGeo<2>::HALO);
        fim_smem = halo * sizeof(double) + (size_t)((nblocks + 3) / 4 * 4) * sizeof(uint32_t);
        if (fim_smem > (size_t)200 * 1024) use_fim = false;
        FP.nblocks = (int32_t)nblocks;
    }
    // block-ordered solver: a "round" is nblocks block visits (every block is visited at least once)
    const int threads = use_fim ? 256
                      : nd == 2 ? std::min(1024, std::max(128, (std::min(P.n[0], P.n[1]) + 31) / 32 * 32)) : 1024;
    int per_sm = std::max(1, 2048 / threads);
    if (use_fim) {               // what really fits (registers, shared memory): a CTA that is not resident only holds a field
        cudaError_t ee = nd == 2 ? cudaFuncSetAttribute(eikonal_fim_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fim_smem)
                                 : cudaFuncSetAttribute(eikonal_fim_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fim_smem);
        if (ee == cudaSuccess)
            ee = nd == 2 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, eikonal_fim_kernel<2>, threads, fim_smem)
                         : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, eikonal_fim_kernel<3>, threads, fim_smem);
        if (ee != cudaSuccess || per_sm < 1) return PAT_ERR_CUDA;
    }
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
    if (e == cudaSuccess) e = cudaMemsetAsync(d_info, 0, 64, st);
    if (e != cudaSuccess) { cudaStreamSynchronize(st); cleanup(); return PAT_ERR_CUDA; }
    P.sh = d_sh; P.T = d_T; P.seed_val = d_sv; P.seed_node = d_sn; P.roi = d_roi; P.npix = npix;
    P.tau_out = tau_out; P.count = count; P.max_rounds = max_rounds; P.info = d_info;
    if (use_fim) {
        FP.e = P;
        const char *it_env = std::getenv("PAT_EIK_ITERS");
        FP.max_iters = it_env && std::atoi(it_env) > 0 ? std::atoi(it_env) : (nd == 3 ? FimGeo<3>::MAX_ITERS : FimGeo<2>::MAX_ITERS);
        FP.stat = (unsigned long long *)(d_info + 4);         // three counters, read back with the round count
        e = nd == 2 ? cudaFuncSetAttribute(eikonal_fim_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fim_smem)
                    : cudaFuncSetAttribute(eikonal_fim_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fim_smem);
        if (e == cudaSuccess) {
            if (nd == 2) eikonal_fim_kernel<2><<<(unsigned)slots, threads, fim_smem, st>>>(FP);
            else         eikonal_fim_kernel<3><<<(unsigned)slots, threads, fim_smem, st>>>(FP);
            e = cudaGetLastError();
        }
    } else {
        if (nd == 2) eikonal_sweep_kernel<2><<<(unsigned)slots, threads, 0, st>>>(P);
        else         eikonal_sweep_kernel<3><<<(unsigned)slots, threads, 0, st>>>(P);
        e = cudaGetLastError();
    }
    int32_t info[16] = {0};
    if (e == cudaSuccess) e = cudaMemcpyAsync(info, d_info, 64, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cleanup();
    if (e != cudaSuccess) return PAT_ERR_CUDA;
    g_last_stats[0] = g_last_stats[1] = g_last_stats[2] = 0;
    if (use_fim) {
        unsigned long long stv[3];
        std::memcpy(stv, info + 4, sizeof(stv));
        for (int q = 0; q < 3; ++q) g_last_stats[q] = (int64_t)stv[q];
        if (std::getenv("PAT_EIK_STATS"))
            std::fprintf(stderr, "[pat] eikonal: %d sensors, %d blocks each, block visits %llu (%.2f per block), Jacobi iterations "
                         "%llu (%.2f per visit), node updates %llu (%.2f per node)\n", count, FP.nblocks, stv[0],
                         (double)stv[0] / ((double)count * FP.nblocks), stv[1], (double)stv[1] / (double)std::max<unsigned long long>(1, stv[0]),
                         stv[2], (double)stv[2] / ((double)count * (double)P.N));
    }
    if (rounds_out) *rounds_out = info[0];
    return info[1] ? PAT_ERR_BAD_STATE : PAT_OK;       // a sensor hit max_rounds without converging
}

extern "C" pat_status pat_eikonal_last_stats(int64_t *block_visits, int64_t *jacobi_iterations, int64_t *node_updates) {
    if (block_visits) *block_visits = g_last_stats[0];
    if (jacobi_iterations) *jacobi_iterations = g_last_stats[1];
    if (node_updates) *node_updates = g_last_stats[2];
    return PAT_OK;
}
