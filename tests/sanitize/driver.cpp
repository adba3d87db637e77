// Sanitizer driver ("race detection / sanitizers"): the CPU oracle (oracle/pat_oracle.c) and the
// production CPU fast marching (csrc/fmm.cpp) built with -fsanitize=address,undefined and run on small problems that
// walk their edge paths: off-node and corner sources, 2-D and 3-D, order 1 and 2, ROI subsets, tables with NaN /
// inf / negative / out-of-record entries, the shortest legal record (nt = 2), zero sensors / pixels / frames.
// Any sanitizer report aborts (halt_on_error); mismatches between the two solvers return a non-zero exit code.
// Test infrastructure only -- built and run by tests/test_sanitizers.py.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <limits>
#include <vector>

#include "../../include/pat.h"

extern "C" {
int oracle_fmm(int32_t ndim, const int32_t *n, double h, const double *origin, const float *c, const double *src,
               int32_t order, double *T, int64_t *frozen_order);
int oracle_fmm_rows(int32_t ndim, const int32_t *n, double h, const double *origin, const float *c, const double *sensors,
                    int32_t nsens, const int64_t *roi_index, int64_t npix, int32_t order, float *tau);
int oracle_tau_conventional(int32_t ndim, const int32_t *n, float h, const float *origin, const float *sensors,
                            int32_t nsens, const int64_t *roi, int64_t npix, float c0, float *tau);
void oracle_weight(const float *p, int32_t nt, double wp, double wd, double t0fs, double *b);
int oracle_backproject(const float *tau, int64_t tau_pitch, const float *traces, int32_t nsens, int64_t npix, int32_t nt,
                       int32_t nframes, float fs, float t0, double wp, double wd, double *image);
int oracle_backproject_exact(const float *tau, int64_t tau_pitch, const float *traces, int32_t nsens, int64_t npix,
                             int32_t nt, int32_t nframes, float fs, float t0, double wp, double wd, double *image);
int oracle_solid_angle_weights(int32_t ndim, const int32_t *n, float h, const float *origin, const float *sensors,
                               const float *normals, int32_t nsens, const int64_t *roi, int64_t npix, float *w, double *omega0);
int oracle_backproject_weighted(const float *tau, const float *wgt, int64_t tau_pitch, const float *traces, int32_t nsens,
                                int64_t npix, int32_t nt, int32_t nframes, float fs, float t0, double wp, double wd, double *image);
}

static uint32_t rng_state = 12345u;
static float urand() { rng_state = rng_state * 1664525u + 1013904223u; return (float)(rng_state >> 8) / 16777216.0f; }

static int fails = 0;
#define CHECK(cond, what) do { if (!(cond)) { std::fprintf(stderr, "FAIL: %s (%s:%d)\n", what, __FILE__, __LINE__); ++fails; } } while (0)

static void fmm_case(int ndim, int n, int order, int nsens) {
    const double h = 0.5e-3;
    int32_t nn[3] = {n, n, ndim == 3 ? n : 1};
    const int64_t N = (int64_t)nn[0] * nn[1] * nn[2];
    double org[3] = {-(n - 1) / 2.0 * h, -(n - 1) / 2.0 * h, ndim == 3 ? -(n - 1) / 2.0 * h : 0.0};
    std::vector<float> c((size_t)N);
    for (auto &v : c) v = 1400.0f + 1700.0f * urand();
    std::vector<double> sens((size_t)nsens * 3, 0.0);
    std::vector<float> sensf((size_t)nsens * 3, 0.0f);
    for (int s = 0; s < nsens; ++s)
        for (int d = 0; d < ndim; ++d) {
            // inside the grid; sensor 0 exactly on the first node, sensor 1 exactly on the last one (corner cells)
            double v = s == 0 ? org[d] : s == 1 ? org[d] + (n - 1) * h : org[d] + urand() * (n - 1) * h;
            sensf[(size_t)s * 3 + d] = (float)v;
            sens[(size_t)s * 3 + d] = (double)sensf[(size_t)s * 3 + d];
        }
    std::vector<int64_t> roi;
    for (int64_t q = 0; q < N; q += 3) roi.push_back(q);
    roi.push_back(N - 1);
    const int64_t P = (int64_t)roi.size();
    std::vector<float> tau_o((size_t)nsens * P), tau_p((size_t)nsens * P);
    // float origins for the production entry point
    pat_grid g{};
    g.ndim = ndim; g.n[0] = nn[0]; g.n[1] = nn[1]; g.n[2] = nn[2]; g.h = (float)h;
    for (int d = 0; d < 3; ++d) g.origin[d] = (float)org[d];
    double orgf[3] = {(double)g.origin[0], (double)g.origin[1], (double)g.origin[2]};
    int rc = oracle_fmm_rows(ndim, nn, (double)g.h, orgf, c.data(), sens.data(), nsens, roi.data(), P, order, tau_o.data());
    CHECK(rc == 0, "oracle_fmm_rows");
    pat_status st = pat_fmm_travel_times(&g, c.data(), sensf.data(), nsens, roi.data(), P, 0, nsens, order, tau_p.data(), 3);
    CHECK(st == PAT_OK, "pat_fmm_travel_times");
    double worst = 0.0, tmax = 0.0;
    for (size_t q = 0; q < tau_o.size(); ++q) {
        worst = std::fmax(worst, std::fabs((double)tau_o[q] - (double)tau_p[q]));
        tmax = std::fmax(tmax, (double)tau_o[q]);
    }
    CHECK(order == 2 || worst <= 1e-6 * tmax, "production FMM vs oracle FMM (first order)");
    // a sensor outside the grid is an error, not a crash
    std::vector<float> bad = sensf;
    bad[0] = (float)(org[0] - 3 * h);
    st = pat_fmm_travel_times(&g, c.data(), bad.data(), nsens, roi.data(), P, 0, 1, order, tau_p.data(), 1);
    CHECK(st == PAT_ERR_INVALID_ARG, "sensor outside the grid");
    std::vector<double> T((size_t)N);
    double outside[3] = {org[0] - 3 * h, org[1], org[2]};
    CHECK(oracle_fmm(ndim, nn, h, org, c.data(), outside, order, T.data(), nullptr) == 1, "oracle: source outside");
    // whole-grid solve with the freeze order recorded
    std::vector<int64_t> fo((size_t)N, -1);
    CHECK(oracle_fmm(ndim, nn, (double)g.h, orgf, c.data(), &sens[3 * (nsens - 1)], order, T.data(), fo.data()) == 0, "oracle_fmm");
    for (int64_t q = 0; q < N; ++q) CHECK(std::isfinite(T[(size_t)q]) && fo[(size_t)q] >= 0, "every node reached");
}

static void bp_case(int S, int P, int nt, int B) {
    const float fs = 20e6f, t0 = 1.5e-7f;
    std::vector<float> tau((size_t)S * P + 1), tr((size_t)B * S * nt + 1), w((size_t)S * P + 1);   // + 1: never a NULL data()
    for (auto &v : tau) v = t0 + urand() * (float)(nt + 2) / fs - 1.0f / fs;        // some below 0, some beyond the record
    for (auto &v : tr) v = urand() - 0.5f;
    for (auto &v : w) v = urand();
    const float specials[] = {std::numeric_limits<float>::quiet_NaN(), std::numeric_limits<float>::infinity(),
                              -std::numeric_limits<float>::infinity(), -1.0f, t0 + (float)(nt - 1) / fs, 1e30f, t0};
    for (size_t q = 0; q < (size_t)S * P && q < 64; ++q) tau[q * 7 % ((size_t)S * P)] = specials[q % 7];
    std::vector<double> img((size_t)B * P + 1, 0.0);
    for (double wd : {0.0, 1.0, 2.0}) {
        int rc = oracle_backproject(tau.data(), P, tr.data(), S, P, nt, B, fs, t0, wd > 0 ? wd : 1.0, wd, img.data());
        CHECK(rc == 0, "oracle_backproject");
        rc = oracle_backproject_exact(tau.data(), P, tr.data(), S, P, nt, B, fs, t0, wd > 0 ? wd : 1.0, wd, img.data());
        CHECK(rc == 0, "oracle_backproject_exact");
        rc = oracle_backproject_weighted(tau.data(), w.data(), P, tr.data(), S, P, nt, B, fs, t0, wd > 0 ? wd : 1.0, wd, img.data());
        CHECK(rc == 0, "oracle_backproject_weighted");
    }
    for (size_t q = 0; q < (size_t)B * P; ++q) CHECK(std::isfinite(img[q]), "finite image");
    std::vector<double> b((size_t)nt);
    if (S > 0 && B > 0) oracle_weight(tr.data(), nt, 1.0, 1.0, 3.0, b.data());
}

static void geometry_case(int ndim) {
    const int n = 9;
    int32_t nn[3] = {n, n, ndim == 3 ? n : 1};
    const float h = 1e-3f, org[3] = {-4e-3f, -4e-3f, ndim == 3 ? -4e-3f : 0.0f};
    const int S = 6;
    std::vector<float> sens((size_t)S * 3, 0.0f), nrm((size_t)S * 3, 0.0f);
    for (int s = 0; s < S; ++s) {
        const float a = 6.2831853f * (float)s / S;
        sens[3 * s] = 20e-3f * std::cos(a); sens[3 * s + 1] = 20e-3f * std::sin(a);
        nrm[3 * s] = std::cos(a); nrm[3 * s + 1] = std::sin(a);
    }
    sens[0] = org[0]; sens[1] = org[1]; sens[2] = org[2];                                 // a detector ON a node
    const int64_t N = (int64_t)nn[0] * nn[1] * nn[2];
    std::vector<float> tau((size_t)S * N), w((size_t)S * N);
    std::vector<double> om((size_t)N);
    CHECK(oracle_tau_conventional(ndim, nn, h, org, sens.data(), S, nullptr, N, 1500.0f, tau.data()) == 0, "tau_conventional");
    CHECK(oracle_solid_angle_weights(ndim, nn, h, org, sens.data(), nrm.data(), S, nullptr, N, w.data(), om.data()) == 0,
          "solid_angle_weights");
    std::vector<int64_t> roi = {0, 5, N - 1};
    CHECK(oracle_tau_conventional(ndim, nn, h, org, sens.data(), S, roi.data(), 3, 1500.0f, tau.data()) == 0, "tau_conventional roi");
    CHECK(oracle_solid_angle_weights(ndim, nn, h, org, sens.data(), nrm.data(), S, roi.data(), 3, w.data(), om.data()) == 0,
          "solid_angle_weights roi");
}

int main() {
    for (int order = 1; order <= 2; ++order) {
        fmm_case(2, 24, order, 4);
        fmm_case(2, 2, order, 2);            // the smallest legal grid: one cell
        fmm_case(3, 10, order, 3);
    }
    bp_case(5, 37, 64, 3);
    bp_case(3, 9, 2, 2);                     // nt = 2: every valid u is in [0, 1)
    bp_case(0, 4, 8, 1);
    bp_case(2, 0, 8, 1);
    bp_case(2, 4, 8, 0);
    geometry_case(2);
    geometry_case(3);
    if (fails) { std::fprintf(stderr, "%d check(s) failed\n", fails); return 1; }
    std::puts("sanitizer driver: ok");
    return 0;
}
