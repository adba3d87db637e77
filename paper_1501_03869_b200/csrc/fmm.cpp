// fmm.cpp -- production CPU fast marching solver (UNTIMED input preparation).
//
// PAPER.md:49-58 (Sec. II.B): |grad T|^2 = 1/c^2 solved by heap-ordered front
// propagation from each SENSOR (reciprocity), first-order upwind
// (BASELINE north_star) or the paper's second-order one-sided stencil Eq. 6
// with first-order fallback.  OpenMP over sensors; each solve
// stops as soon as every ROI node is frozen.
//
// Written independently of oracle/pat_oracle.c (different heap: indexed 4-ary
// with decrease-key; closed-form local solves); the two are only compared in tests.
#include "pat_internal.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr double kInf = std::numeric_limits<double>::infinity();

struct Front {                       // indexed 4-ary min-heap keyed (T, node)
    std::vector<int32_t> heap;       // node ids
    std::vector<int32_t> pos;        // node -> slot in heap, -1 = not queued
    const double *key = nullptr;

    bool less(int32_t a, int32_t b) const {
        return key[a] < key[b] || (key[a] == key[b] && a < b);
    }
    void up(size_t i) {
        int32_t v = heap[i];
        while (i > 0) {
            size_t p = (i - 1) >> 2;
            if (!less(v, heap[p])) break;
            heap[i] = heap[p]; pos[heap[i]] = (int32_t)i; i = p;
        }
        heap[i] = v; pos[v] = (int32_t)i;
    }
    void down(size_t i) {
        int32_t v = heap[i];
        const size_t n = heap.size();
        for (;;) {
            size_t c0 = 4 * i + 1;
            if (c0 >= n) break;
            size_t best = c0;
            size_t ce = std::min(c0 + 4, n);
            for (size_t c = c0 + 1; c < ce; ++c) if (less(heap[c], heap[best])) best = c;
            if (!less(heap[best], v)) break;
            heap[i] = heap[best]; pos[heap[i]] = (int32_t)i; i = best;
        }
        heap[i] = v; pos[v] = (int32_t)i;
    }
    void push_or_decrease(int32_t v) {
        if (pos[v] < 0) { heap.push_back(v); up(heap.size() - 1); }
        else up((size_t)pos[v]);
    }
    int32_t pop() {
        int32_t top = heap[0];
        pos[top] = -1;
        int32_t last = heap.back();
        heap.pop_back();
        if (!heap.empty()) { heap[0] = last; down(0); }
        return top;
    }
};

struct Domain {
    int ndim;
    int64_t n[3], stride[3], N;
    double h, org[3];
};

// One axis' upwind information at a node.
struct Upwind { double a, a2; };     // nearest frozen value, and the one behind it (or inf)

inline double solve_first_order(int ndim, double a0, double a1, double a2, double sh) {
    // a0 <= a1 <= a2 (inf = absent)
    double T = a0 + sh;
    if (ndim < 2 || !(T > a1)) return T;
    double d = a0 - a1;
    double T2 = 0.5 * (a0 + a1 + std::sqrt(2.0 * sh * sh - d * d));
    if (ndim < 3 || !(T2 > a2)) return T2;
    double S = a0 + a1 + a2, Q = a0 * a0 + a1 * a1 + a2 * a2;
    double disc = S * S - 3.0 * (Q - sh * sh);
    if (disc < 0.0) return T2;
    return (S + std::sqrt(disc)) / 3.0;
}

// Second-order variant: per axis use (3T - 4a + a2)/(2h) when a2 is usable.
inline double solve_mixed_order(int ndim, const Upwind *u, double s, double h) {
    int idx[3] = {0, 1, 2};
    auto cswap = [&](int i, int j) { if (u[idx[j]].a < u[idx[i]].a) std::swap(idx[i], idx[j]); };
    if (ndim == 3) { cswap(0, 1); cswap(1, 2); cswap(0, 1); }
    else if (ndim == 2) cswap(0, 1);
    double best = kInf;
    double A = 0, B = 0, C = -s * s;          // A T^2 - 2 B T + C = 0
    double A1 = 0, B1 = 0, C1 = -s * s;       // same, all axes first order
    for (int m = 0; m < ndim; ++m) {
        const Upwind &w = u[idx[m]];
        if (!std::isfinite(w.a)) break;
        double al = 1.0 / h, be = w.a / h;
        A1 += al * al; B1 += al * be; C1 += be * be;
        if (std::isfinite(w.a2) && w.a2 <= w.a) { al = 1.5 / h; be = (4.0 * w.a - w.a2) / (2.0 * h); }
        A += al * al; B += al * be; C += be * be;
        double disc = B * B - A * C;
        double T = disc >= 0.0 ? (B + std::sqrt(disc)) / A : std::numeric_limits<double>::quiet_NaN();
        if (!(T >= w.a)) {                    // not causal (or no real root): first order for this m
            double d1 = B1 * B1 - A1 * C1;
            if (d1 < 0.0) break;
            T = (B1 + std::sqrt(d1)) / A1;
        }
        best = T;
        double next = (m + 1 < ndim) ? u[idx[m + 1]].a : kInf;
        if (T <= next) break;
    }
    return best;
}

struct Workspace {
    std::vector<double> T;
    std::vector<uint8_t> frozen;
    Front front;
};

int solve_one(const Domain &D, const double *slow, const uint8_t *in_roi, int64_t roi_count,
              const double *src, double c_unused, int order, Workspace &ws) {
    (void)c_unused;
    const int nd = D.ndim;
    int64_t i0[3] = {0, 0, 0}, inr[3] = {0, 0, 0};
    for (int d = 0; d < nd; ++d) {
        double g = (src[d] - D.org[d]) / D.h;
        if (!(g >= 0.0 && g <= (double)(D.n[d] - 1))) return 1;
        int64_t f = (int64_t)std::floor(g);
        i0[d] = std::min<int64_t>(f, D.n[d] - 2);
        inr[d] = std::min<int64_t>((int64_t)std::floor(g + 0.5), D.n[d] - 1);
    }
    std::fill(ws.T.begin(), ws.T.end(), kInf);
    std::fill(ws.frozen.begin(), ws.frozen.end(), (uint8_t)0);
    std::fill(ws.front.pos.begin(), ws.front.pos.end(), -1);
    ws.front.heap.clear();
    ws.front.key = ws.T.data();
    double *T = ws.T.data();
    uint8_t *fz = ws.frozen.data();

    const double s_near = slow[inr[0] + D.stride[1] * inr[1] + D.stride[2] * inr[2]];
    for (int cn = 0; cn < (1 << nd); ++cn) {
        int64_t q = 0; double d2 = 0;
        for (int d = 0; d < nd; ++d) {
            int64_t id = i0[d] + ((cn >> d) & 1);
            double x = D.org[d] + (double)id * D.h - src[d];
            d2 += x * x; q += id * D.stride[d];
        }
        T[q] = std::sqrt(d2) * s_near;
        ws.front.push_or_decrease((int32_t)q);
    }
    // note: sqrt(d2)*s_near vs the oracle's sqrt(d2)/c_near may differ in the last ulp.

    int64_t left = roi_count;
    while (!ws.front.heap.empty() && left > 0) {
        const int32_t q = ws.front.pop();
        fz[q] = 1;
        if (in_roi[q]) --left;
        int64_t iq[3] = { q % D.n[0], (q / D.n[0]) % D.n[1], q / (D.n[0] * D.n[1]) };
        for (int d = 0; d < nd; ++d) {
            for (int sg = -1; sg <= 1; sg += 2) {
                int64_t jd = iq[d] + sg;
                if (jd < 0 || jd >= D.n[d]) continue;
                const int64_t r = q + sg * D.stride[d];
                if (fz[r]) continue;
                int64_t ir[3] = { iq[0], iq[1], iq[2] };
                ir[d] = jd;
                Upwind u[3] = { {kInf, kInf}, {kInf, kInf}, {kInf, kInf} };
                for (int e = 0; e < nd; ++e) {
                    for (int s2 = -1; s2 <= 1; s2 += 2) {
                        int64_t ke = ir[e] + s2;
                        if (ke < 0 || ke >= D.n[e]) continue;
                        int64_t w = r + s2 * D.stride[e];
                        if (!fz[w] || !(T[w] < u[e].a)) continue;
                        u[e].a = T[w];
                        u[e].a2 = kInf;
                        if (order == 2) {
                            int64_t k2 = ir[e] + 2 * s2;
                            if (k2 >= 0 && k2 < D.n[e]) {
                                int64_t w2 = r + 2 * s2 * D.stride[e];
                                if (fz[w2]) u[e].a2 = T[w2];
                            }
                        }
                    }
                }
                double Tn;
                if (order == 1) {
                    double a[3] = { u[0].a, u[1].a, u[2].a };     // unused axes are +inf
                    if (a[1] < a[0]) std::swap(a[0], a[1]);
                    if (a[2] < a[1]) std::swap(a[1], a[2]);
                    if (a[1] < a[0]) std::swap(a[0], a[1]);
                    Tn = solve_first_order(nd, a[0], nd > 1 ? a[1] : kInf, nd > 2 ? a[2] : kInf,
                                           slow[r] * D.h);
                } else {
                    Tn = solve_mixed_order(nd, u, slow[r], D.h);
                }
                if (Tn < T[r]) { T[r] = Tn; ws.front.push_or_decrease((int32_t)r); }
            }
        }
    }
    return 0;
}

}  // namespace

extern "C" pat_status pat_fmm_travel_times(const pat_grid *grid, const float *c_map,
                                           const float *sensor_xyz, int32_t nsens,
                                           const int64_t *roi_index, int64_t npix,
                                           int32_t sensor_begin, int32_t count, int32_t order,
                                           float *tau_out, int32_t nthreads) {
    if (!grid || !c_map || !sensor_xyz || !tau_out) return PAT_ERR_INVALID_ARG;
    if (grid->ndim != 2 && grid->ndim != 3) return PAT_ERR_INVALID_ARG;
    if (!(grid->h > 0.0f) || (order != 1 && order != 2)) return PAT_ERR_INVALID_ARG;
    if (nsens <= 0 || sensor_begin < 0 || count < 0 || sensor_begin > nsens - count) return PAT_ERR_INVALID_ARG;
    Domain D;
    D.ndim = grid->ndim;
    D.h = (double)grid->h;
    D.N = 1;
    for (int d = 0; d < 3; ++d) {
        D.n[d] = d < D.ndim ? grid->n[d] : 1;
        if (d < D.ndim && D.n[d] < 2) return PAT_ERR_INVALID_ARG;
        D.org[d] = (double)grid->origin[d];
        D.stride[d] = D.N;
        D.N *= D.n[d];
    }
    if (D.N > (int64_t)std::numeric_limits<int32_t>::max()) return PAT_ERR_INVALID_ARG;
    if (npix < 0 || (!roi_index && npix != D.N)) return PAT_ERR_INVALID_ARG;
    if (count == 0 || npix == 0) return PAT_OK;

    std::vector<double> slow;
    std::vector<uint8_t> in_roi;
    try {
        slow.resize((size_t)D.N);
        in_roi.assign((size_t)D.N, roi_index ? 0 : 1);
    } catch (...) { return PAT_ERR_NOMEM; }
    for (int64_t q = 0; q < D.N; ++q) {
        float c = c_map[q];
        if (!(c > 0.0f) || !std::isfinite(c)) return PAT_ERR_INVALID_ARG;
        slow[q] = 1.0 / (double)c;
    }
    if (roi_index)
        for (int64_t j = 0; j < npix; ++j) {
            if (roi_index[j] < 0 || roi_index[j] >= D.N) return PAT_ERR_INVALID_ARG;
            in_roi[roi_index[j]] = 1;
        }
    int64_t roi_count = 0;
    for (int64_t q = 0; q < D.N; ++q) roi_count += in_roi[q];

    int status = 0;
#ifdef _OPENMP
    int nth = nthreads > 0 ? nthreads : omp_get_max_threads();
    nth = std::max(1, std::min(nth, (int)count));
#else
    int nth = 1; (void)nthreads;
#endif
    #pragma omp parallel num_threads(nth)
    {
        Workspace ws;
        bool ok = true;
        try {
            ws.T.resize((size_t)D.N); ws.frozen.resize((size_t)D.N); ws.front.pos.resize((size_t)D.N);
            ws.front.heap.reserve(1 << 16);
        } catch (...) { ok = false; }
        #pragma omp for schedule(dynamic, 1)
        for (int32_t i = 0; i < count; ++i) {
            if (!ok) {
                #pragma omp atomic write
                status = 2;
                continue;
            }
            const float *sf = sensor_xyz + 3 * (int64_t)(sensor_begin + i);
            double src[3] = { (double)sf[0], (double)sf[1], (double)sf[2] };
            int rc = solve_one(D, slow.data(), in_roi.data(), roi_count, src, 0.0, order, ws);
            if (rc) {
                #pragma omp atomic write
                status = rc;
                continue;
            }
            float *row = tau_out + (int64_t)i * npix;
            if (roi_index) for (int64_t j = 0; j < npix; ++j) row[j] = (float)ws.T[roi_index[j]];
            else           for (int64_t j = 0; j < npix; ++j) row[j] = (float)ws.T[j];
        }
    }
    if (status == 1) return PAT_ERR_INVALID_ARG;
    if (status == 2) return PAT_ERR_NOMEM;
    return PAT_OK;
}
