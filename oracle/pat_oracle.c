/*
 * pat_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU restatement of the method of
 * Wang & Jing, "A fast marching method based back projection algorithm for
 * photoacoustic tomography in heterogeneous media" (arxiv 1501.03869):
 *
 *   oracle_fmm          eikonal arrival times, PAPER.md:49-58 (Sec. II.B, Eq. 5)
 *   oracle_weight       the integrand of Eq. 7 at the sample times
 *   oracle_backproject  Eq. 7 as a plain triple loop, PAPER.md:64-69 (Sec. II.C)
 *   oracle_tau_conventional  the conventional BP's analytic delays
 *   oracle_backproject_exact Eq. 7 with the weight taken AT t_ij (its literal form)
 *   oracle_solid_angle_weights, oracle_backproject_weighted  the "exact BP algorithm [5]" that Eq. 7
 *                       approximates: every term weighted by dOmega_ij / Omega0_j
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this file.  It shares no code, header, table or
 * helper with the CUDA path under paper_1501_03869_b200/ and imports nothing
 * from it.  Double precision everywhere except the one place the reading
 * DESIGN.md R8 fixes in fp32 (the time -> sample-index map u = fl32(tau*fs)).
 *
 * Pins (tests/test_oracle_*.py): every function here is pinned by closed forms,
 * invariants or brute force; what is NOT pinned is agreement
 * with the paper's figures 2-5 (no numeric values printed, data not available):
 * "parity unpinned" for the paper's images.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 * -ffp-contract=off matters: u = tau*fs must be ONE IEEE fp32 multiply.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------- */
/* Fast marching method ("starting with an initial condition, the
 * neighboring point with the shortest arrival time is calculated.  This
 * repeats recursively until all the points in the region are visited").
 * First-order upwind (BASELINE north_star) or the paper's second-order
 * one-sided stencil Eq. 6 with first-order fallback.           */
/* ------------------------------------------------------------------------- */

typedef struct { double t; int64_t idx; } heap_ent;
typedef struct { heap_ent *e; int64_t n, cap; } heap_t;

static int ent_less(const heap_ent *a, const heap_ent *b)
{
    if (a->t != b->t) return a->t < b->t;
    return a->idx < b->idx;            /* tie: smaller linear index first */
}

static int heap_push(heap_t *hp, double t, int64_t idx)
{
    if (hp->n == hp->cap) {
        int64_t nc = hp->cap ? 2 * hp->cap : 1024;
        heap_ent *ne = (heap_ent *)realloc(hp->e, (size_t)nc * sizeof(heap_ent));
        if (!ne) return -1;
        hp->e = ne; hp->cap = nc;
    }
    int64_t i = hp->n++;
    hp->e[i].t = t; hp->e[i].idx = idx;
    while (i > 0) {
        int64_t p = (i - 1) / 2;
        if (!ent_less(&hp->e[i], &hp->e[p])) break;
        heap_ent tmp = hp->e[i]; hp->e[i] = hp->e[p]; hp->e[p] = tmp;
        i = p;
    }
    return 0;
}

static heap_ent heap_pop(heap_t *hp)
{
    heap_ent top = hp->e[0];
    hp->e[0] = hp->e[--hp->n];
    int64_t i = 0;
    for (;;) {
        int64_t l = 2 * i + 1, r = l + 1, m = i;
        if (l < hp->n && ent_less(&hp->e[l], &hp->e[m])) m = l;
        if (r < hp->n && ent_less(&hp->e[r], &hp->e[m])) m = r;
        if (m == i) break;
        heap_ent tmp = hp->e[i]; hp->e[i] = hp->e[m]; hp->e[m] = tmp;
        i = m;
    }
    return top;
}

enum { FAR = 0, TRIAL = 1, FROZEN = 2 };

/* Solve  sum_{d<m} (alpha_d*T - beta_d)^2 = s^2  for the larger root, where
 * each used axis contributes the one-sided difference
 *   first order : (T - a)/h                 -> alpha = 1/h,   beta = a/h
 *   second order: (3T - 4a + a2)/(2h) Eq. 6 -> alpha = 3/(2h), beta = (4a - a2)/(2h)
 * Returns NaN if the discriminant is negative. */
static double quad_root(int m, const double *alpha, const double *beta, double s)
{
    double A = 0.0, Bq = 0.0, C = -s * s;
    for (int d = 0; d < m; ++d) {
        A  += alpha[d] * alpha[d];
        Bq += alpha[d] * beta[d];
        C  += beta[d] * beta[d];
    }
    double disc = Bq * Bq - A * C;
    if (disc < 0.0) return NAN;
    return (Bq + sqrt(disc)) / A;
}

/* Local upwind solve at one node (Godunov / Rouy-Tourin form).
 * a[d]  = smaller frozen neighbour value along axis d (INFINITY if none),
 * a2[d] = value one node further upwind along the same side, usable for the
 *         second-order stencil only if frozen and a2[d] <= a[d] (else INFINITY).
 * Axes are taken in ascending order of a[d]; the first m with T_m <= a_{m+1}
 * (or m = number of finite a's) is accepted. */
static double local_solve(int ndim, const double *a_in, const double *a2_in,
                          double s /* slowness */, double h, int order)
{
    int perm[3] = {0, 1, 2};
    for (int i = 0; i < ndim; ++i)            /* tiny insertion sort by a */
        for (int j = i; j > 0 && a_in[perm[j]] < a_in[perm[j - 1]]; --j) {
            int t = perm[j]; perm[j] = perm[j - 1]; perm[j - 1] = t;
        }
    double a[4], alpha[3], beta[3];
    int nfin = 0;
    for (int d = 0; d < ndim; ++d) {
        int p = perm[d];
        a[d] = a_in[p];
        if (isfinite(a[d])) nfin = d + 1;
        if (order == 2 && isfinite(a2_in[p]) && a2_in[p] <= a_in[p]) {
            alpha[d] = 3.0 / (2.0 * h);
            beta[d]  = (4.0 * a_in[p] - a2_in[p]) / (2.0 * h);
        } else {
            alpha[d] = 1.0 / h;
            beta[d]  = a_in[p] / h;
        }
    }
    a[ndim] = INFINITY;
    if (nfin == 0) return INFINITY;
    double T = INFINITY;
    for (int m = 1; m <= nfin; ++m) {
        double Tm = quad_root(m, alpha, beta, s);
        if (isnan(Tm) || Tm < a[m - 1]) {
            /* second-order stencil not causal here: redo this m in first order */
            double al1[3], be1[3];
            for (int d = 0; d < m; ++d) { al1[d] = 1.0 / h; be1[d] = a[d] / h; }
            Tm = quad_root(m, al1, be1, s);
            if (isnan(Tm)) break;               /* keep the previous m's value */
        }
        T = Tm;
        if (m == nfin || Tm <= a[m]) break;
    }
    return T;
}

/* oracle_fmm: arrival time T (seconds, double) at every node of a regular grid
 * from a point source at src (metres).
 *   ndim        2 or 3;  n[3] nodes per axis, x fastest (n[2] = 1 in 2-D)
 *   h           isotropic spacing [m];  origin[3] = coordinates of node (0,0,0)
 *   c           speed of sound [m/s] at the nodes, fp32, n0*n1*n2 entries
 *   order       1 = first-order upwind; 2 = Eq. 6 with first-order fallback
 *   T           out, n0*n1*n2 doubles
 *   frozen_order out, may be NULL: linear index of the q-th frozen node
 * Returns 0, or 1 bad argument / source outside the grid, 2 out of memory. */
int oracle_fmm(int32_t ndim, const int32_t *n, double h, const double *origin,
               const float *c, const double *src, int32_t order,
               double *T, int64_t *frozen_order)
{
    if (ndim != 2 && ndim != 3) return 1;
    if (!(h > 0.0) || (order != 1 && order != 2)) return 1;
    int64_t nn[3] = { n[0], n[1], ndim == 3 ? n[2] : 1 };
    for (int d = 0; d < ndim; ++d) if (nn[d] < 2) return 1;
    const int64_t N = nn[0] * nn[1] * nn[2];
    const int64_t stride[3] = { 1, nn[0], nn[0] * nn[1] };

    /* cell enclosing the source and the node nearest to it (reading R12) */
    int64_t i0[3] = {0, 0, 0}, inear[3] = {0, 0, 0};
    for (int d = 0; d < ndim; ++d) {
        double g = (src[d] - origin[d]) / h;
        if (!(g >= 0.0 && g <= (double)(nn[d] - 1))) return 1;
        int64_t f = (int64_t)floor(g);
        if (f > nn[d] - 2) f = nn[d] - 2;
        i0[d] = f;
        int64_t r = (int64_t)floor(g + 0.5);
        if (r > nn[d] - 1) r = nn[d] - 1;
        inear[d] = r;
    }
    const double c_near = (double)c[inear[0] + stride[1] * inear[1] + stride[2] * inear[2]];

    unsigned char *state = (unsigned char *)calloc((size_t)N, 1);
    heap_t hp = {0, 0, 0};
    if (!state) return 2;
    for (int64_t q = 0; q < N; ++q) T[q] = INFINITY;

    const int ncorner = 1 << ndim;
    for (int cn = 0; cn < ncorner; ++cn) {
        int64_t id[3] = {0, 0, 0};
        double d2 = 0.0;
        for (int d = 0; d < ndim; ++d) {
            id[d] = i0[d] + ((cn >> d) & 1);
            double x = origin[d] + (double)id[d] * h;
            d2 += (x - src[d]) * (x - src[d]);
        }
        int64_t q = id[0] + stride[1] * id[1] + stride[2] * id[2];
        T[q] = sqrt(d2) / c_near;
        state[q] = TRIAL;
        if (heap_push(&hp, T[q], q)) { free(state); free(hp.e); return 2; }
    }

    int64_t nfrozen = 0;
    while (hp.n > 0) {
        heap_ent top = heap_pop(&hp);
        int64_t q = top.idx;
        if (state[q] == FROZEN || top.t != T[q]) continue;       /* stale entry */
        state[q] = FROZEN;
        if (frozen_order) frozen_order[nfrozen] = q;
        ++nfrozen;

        int64_t iq[3] = { q % nn[0], (q / nn[0]) % nn[1], q / (nn[0] * nn[1]) };
        for (int d = 0; d < ndim; ++d) {
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                int64_t jd = iq[d] + sgn;
                if (jd < 0 || jd >= nn[d]) continue;
                int64_t r = q + sgn * stride[d];
                if (state[r] == FROZEN) continue;
                /* gather the upwind data of node r from FROZEN neighbours only */
                int64_t ir[3] = { iq[0], iq[1], iq[2] };
                ir[d] = jd;
                double a[3]  = { INFINITY, INFINITY, INFINITY };
                double a2[3] = { INFINITY, INFINITY, INFINITY };
                for (int e = 0; e < ndim; ++e) {
                    for (int s2 = -1; s2 <= 1; s2 += 2) {
                        int64_t ke = ir[e] + s2;
                        if (ke < 0 || ke >= nn[e]) continue;      /* outside = +inf */
                        int64_t w = r + s2 * stride[e];
                        if (state[w] != FROZEN) continue;
                        if (T[w] < a[e]) {
                            a[e] = T[w];
                            a2[e] = INFINITY;
                            int64_t ke2 = ir[e] + 2 * s2;
                            if (ke2 >= 0 && ke2 < nn[e]) {
                                int64_t w2 = r + 2 * s2 * stride[e];
                                if (state[w2] == FROZEN) a2[e] = T[w2];
                            }
                        }
                    }
                }
                double sl = 1.0 / (double)c[r];    /* slowness at the node being updated */
                double Tn = local_solve(ndim, a, a2, sl, h, order);
                if (Tn < T[r]) {
                    T[r] = Tn;
                    state[r] = TRIAL;
                    if (heap_push(&hp, Tn, r)) { free(state); free(hp.e); return 2; }
                }
            }
        }
    }
    free(state);
    free(hp.e);
    return 0;
}

/* oracle_fmm_rows: reciprocity: one FMM per SENSOR, the row
 * tau[i][j] = (float) T_i(node roi_index[j]), computed in double, rounded once.
 *   sensors  nsens*3 doubles [m];  roi_index npix linear node indices
 *   tau      out, fp32 [nsens][npix]
 * Sensors are independent, so the loop is an OpenMP parallel for. */
int oracle_fmm_rows(int32_t ndim, const int32_t *n, double h, const double *origin,
                    const float *c, const double *sensors, int32_t nsens,
                    const int64_t *roi_index, int64_t npix, int32_t order,
                    float *tau)
{
    int64_t N = (int64_t)n[0] * n[1] * (ndim == 3 ? n[2] : 1);
    int rc = 0;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int32_t i = 0; i < nsens; ++i) {
        double *T = (double *)malloc((size_t)N * sizeof(double));
        int r = T ? oracle_fmm(ndim, n, h, origin, c, sensors + 3 * (int64_t)i, order, T, NULL) : 2;
        if (r == 0)
            for (int64_t j = 0; j < npix; ++j)
                tau[(int64_t)i * npix + j] = (float)T[roi_index[j]];
        else {
            #pragma omp critical
            rc = r;
        }
        free(T);
    }
    return rc;
}

/* ------------------------------------------------------------------------- */
/* Eq. 7:  P(r_j) = sum_i [ p_i(t_ij) - t_ij * dp_i/dt (t_ij) ] */
/* ------------------------------------------------------------------------- */

/* oracle_tau_conventional: the conventional back projection's delays
 * ("In the conventional BP algorithm, t_ij is calculated
 * analytically by assuming a constant speed"): tau_ij = |r_j - s_i| / c0, with
 * r_j the position of ROI node j and s_i the sensor position.  The delay goes
 * through floor() in Eq. 7's time -> sample map, so its arithmetic type is part
 * of the definition (R26): fp32, one IEEE operation per step, in the
 * order
 *     x_d  = fl(origin_d + fl((float)i_d * h))          node coordinate, axis d
 *     e_d  = fl(x_d - s_d)
 *     d2   = fl(fl(fl(e_0*e_0) + fl(e_1*e_1)) + fl(e_2*e_2))   (no e_2 term in 2-D)
 *     tau  = fl(fl(sqrt(d2)) * fl(1/c0))
 * (-ffp-contract=off: no fused multiply-add).  sensors: fp32 [nsens][3];
 * roi: linear node indices (x fastest) or NULL for all nodes; tau: fp32
 * [nsens][npix].  Returns 0, or 1 for a bad argument. */
int oracle_tau_conventional(int32_t ndim, const int32_t *n, float h, const float *origin,
                            const float *sensors, int32_t nsens, const int64_t *roi,
                            int64_t npix, float c0, float *tau)
{
    if ((ndim != 2 && ndim != 3) || !n || !origin || !sensors || !tau || !(c0 > 0.0f)) return 1;
    const int64_t n0 = n[0], n1 = n[1];
    const float inv_c0 = 1.0f / c0;
    for (int32_t i = 0; i < nsens; ++i) {
        const float *s = sensors + 3 * (int64_t)i;
        for (int64_t j = 0; j < npix; ++j) {
            const int64_t q = roi ? roi[j] : j;
            const int64_t id[3] = { q % n0, (q / n0) % n1, q / (n0 * n1) };
            float d2 = 0.0f;
            for (int d = 0; d < ndim; ++d) {
                const float step = (float)id[d] * h;
                const float x = origin[d] + step;
                const float e = x - s[d];
                const float sq = e * e;
                d2 = d == 0 ? sq : d2 + sq;
            }
            const float dist = sqrtf(d2);
            tau[(int64_t)i * npix + j] = dist * inv_c0;
        }
    }
    return 0;
}

/* oracle_weight: b[n] = wp*p[n] - wd*t_n*(dp/dt)[n] at the sample times
 * t_n = t0 + n/fs.  With the finite difference D[n] (central, one-sided at the
 * two ends; reading R3) dp/dt = D[n]*fs, so t_n*dp/dt = (n + t0*fs)*D[n].
 * (wp, wd) = (1,1) is Eq. 7 as printed, (1,0) plain delay-and-sum, (2,2) the
 * universal-BP form of ref. [5].  p is fp32 (the data), b is double. */
void oracle_weight(const float *p, int32_t nt, double wp, double wd, double t0fs, double *b)
{
    for (int32_t k = 0; k < nt; ++k) {
        double D;
        if (k == 0)            D = (double)p[1] - (double)p[0];
        else if (k == nt - 1)  D = (double)p[nt - 1] - (double)p[nt - 2];
        else                   D = ((double)p[k + 1] - (double)p[k - 1]) / 2.0;
        b[k] = wp * (double)p[k] - wd * ((double)k + t0fs) * D;
    }
}

/* oracle_backproject: for every frame f and pixel j
 *     image[f][j] = sum_{i<nsens} (1-a)*b_fi[k] + a*b_fi[k+1],
 *     u = fl32( fl32(tau[i][j] - t0) * fs ),  k = floor(u),  a = u - k,
 * terms with !(0 <= u < nt-1) contribute 0 (readings R6-R8).
 *   tau     fp32 seconds, [nsens][tau_pitch] (tau_pitch >= npix)
 *   traces  fp32 [nframes][nsens][nt]
 *   image   out, double [nframes][npix]
 * Returns 0, or 1 bad argument, 2 out of memory. */
int oracle_backproject(const float *tau, int64_t tau_pitch, const float *traces,
                       int32_t nsens, int64_t npix, int32_t nt, int32_t nframes,
                       float fs, float t0, double wp, double wd, double *image)
{
    if (nsens < 0 || npix < 0 || nt < 2 || nframes < 0 || tau_pitch < npix) return 1;
    double *b = (double *)malloc((size_t)(nsens > 0 ? nsens : 1) * (size_t)nt * sizeof(double));
    if (!b) return 2;
    const double t0fs = (double)t0 * (double)fs;
    const float ulim = (float)(nt - 1);
    for (int32_t f = 0; f < nframes; ++f) {
        for (int32_t i = 0; i < nsens; ++i)
            oracle_weight(traces + ((int64_t)f * nsens + i) * nt, nt, wp, wd, t0fs,
                          b + (int64_t)i * nt);
        #pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < npix; ++j) {
            double acc = 0.0;
            for (int32_t i = 0; i < nsens; ++i) {
                float ts = tau[(int64_t)i * tau_pitch + j] - t0;   /* fp32 subtract */
                float u = ts * fs;                                 /* ONE fp32 multiply */
                if (!(u >= 0.0f && u < ulim)) continue;
                float kf = floorf(u);
                int32_t k = (int32_t)kf;
                float a = u - kf;                                  /* exact in fp32 */
                const double *bi = b + (int64_t)i * nt;
                acc += (1.0 - (double)a) * bi[k] + (double)a * bi[k + 1];
            }
            image[(int64_t)f * npix + j] = acc;
        }
    }
    free(b);
    return 0;
}

/* oracle_backproject_exact: Eq. 7 read literally ("p_i(t_ij) - t_ij * dp_i(t_ij)/dt"): the
 * pressure AND its derivative are each sampled at the arrival time t_ij by linear interpolation, and the
 * factor t is t_ij itself, not the sample times (reading R4b):
 *     image[f][j] = sum_i  wp * [(1-a)*p[k] + a*p[k+1]]  -  wd * (u + t0*fs) * [(1-a)*D[k] + a*D[k+1]]
 * with u, k, a exactly as in oracle_backproject (t_ij*fs = u + t0*fs in sample units; dp/dt = D*fs, so
 * fs cancels) and D the finite difference of oracle_weight (central, one-sided at the two ends).
 * Same arguments and return codes as oracle_backproject. */
int oracle_backproject_exact(const float *tau, int64_t tau_pitch, const float *traces,
                             int32_t nsens, int64_t npix, int32_t nt, int32_t nframes,
                             float fs, float t0, double wp, double wd, double *image)
{
    if (nsens < 0 || npix < 0 || nt < 2 || nframes < 0 || tau_pitch < npix) return 1;
    double *D = (double *)malloc((size_t)(nsens > 0 ? nsens : 1) * (size_t)nt * sizeof(double));
    if (!D) return 2;
    const double t0fs = (double)t0 * (double)fs;
    const float ulim = (float)(nt - 1);
    for (int32_t f = 0; f < nframes; ++f) {
        const float *pf = traces + (int64_t)f * nsens * nt;
        for (int32_t i = 0; i < nsens; ++i) {
            const float *p = pf + (int64_t)i * nt;
            double *Di = D + (int64_t)i * nt;
            for (int32_t k = 0; k < nt; ++k) {
                if (k == 0)            Di[k] = (double)p[1] - (double)p[0];
                else if (k == nt - 1)  Di[k] = (double)p[nt - 1] - (double)p[nt - 2];
                else                   Di[k] = ((double)p[k + 1] - (double)p[k - 1]) / 2.0;
            }
        }
        #pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < npix; ++j) {
            double acc = 0.0;
            for (int32_t i = 0; i < nsens; ++i) {
                float ts = tau[(int64_t)i * tau_pitch + j] - t0;   /* fp32 subtract */
                float u = ts * fs;                                 /* ONE fp32 multiply */
                if (!(u >= 0.0f && u < ulim)) continue;
                float kf = floorf(u);
                int32_t k = (int32_t)kf;
                double a = (double)(u - kf);                       /* exact in fp32 */
                const float *p = pf + (int64_t)i * nt;
                const double *Di = D + (int64_t)i * nt;
                double pv = (1.0 - a) * (double)p[k] + a * (double)p[k + 1];
                double dv = (1.0 - a) * Di[k] + a * Di[k + 1];
                acc += wp * pv - wd * ((double)u + t0fs) * dv;
            }
            image[(int64_t)f * npix + j] = acc;
        }
    }
    free(D);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* "Eq. 7 can be viewed as an approximation to the exact BP algorithm [5].  It assumes a
 * circular scanning geometry and that the scanning radius is considerably larger than the region of
 * interest."  Ref. [5] (universal back projection) weights the term of detector i at point r_j by the solid
 * angle dOmega_ij the detector element subtends at r_j, normalised by the total Omega0_j:
 *     P(r_j) = sum_i (dOmega_ij / Omega0_j) * b_i(t_ij),   b = 2p - 2t dp/dt  (weighting mode 2),
 *     dOmega_ij = dS_i * n_i . (s_i - r_j) / |s_i - r_j|^3 ,   Omega0_j = sum_i dOmega_ij ,
 * n_i = the unit normal of the detection surface at s_i pointing AWAY from the imaged region.  Equal element
 * areas dS_i cancel.  Under the paper's assumption (large circle) dOmega_ij / Omega0_j -> 1/S and the sum
 * becomes Eq. 7 up to the constant 1/S.  Readings (R27): in 2-D (ring of detectors in the image
 * plane) the subtended ANGLE n.e/|e|^2 takes the place of the solid angle; a detector facing away from the
 * point (n.e <= 0) or sitting on it (|e| = 0) gets weight 0; a point that no detector faces gets all-zero
 * weights.  SURVEY.md 8(f) NEXT-4.
 *
 * oracle_solid_angle_weights: node coordinates x_d = origin_d + i_d*h and everything after in double from the
 * fp32 inputs.  w: fp32 out [nsens][npix] (the normalised weights); omega0: double out [npix] or NULL (the
 * un-normalised sum, for the closed-curve / closed-surface pins).  Returns 0, or 1 bad argument. */
int oracle_solid_angle_weights(int32_t ndim, const int32_t *n, float h, const float *origin,
                               const float *sensors, const float *normals, int32_t nsens,
                               const int64_t *roi, int64_t npix, float *w, double *omega0)
{
    if ((ndim != 2 && ndim != 3) || !n || !origin || !sensors || !normals || !w || nsens < 0) return 1;
    const int64_t n0 = n[0], n1 = n[1];
    for (int64_t j = 0; j < npix; ++j) {
        const int64_t q = roi ? roi[j] : j;
        const int64_t id[3] = { q % n0, (q / n0) % n1, q / (n0 * n1) };
        double r[3] = { 0.0, 0.0, 0.0 };
        for (int d = 0; d < ndim; ++d) r[d] = (double)origin[d] + (double)id[d] * (double)h;
        double total = 0.0;
        for (int pass = 0; pass < 2; ++pass) {
            for (int32_t i = 0; i < nsens; ++i) {
                double dot = 0.0, d2 = 0.0;
                for (int d = 0; d < ndim; ++d) {
                    const double e = (double)sensors[3 * (int64_t)i + d] - r[d];
                    dot += (double)normals[3 * (int64_t)i + d] * e;
                    d2 += e * e;
                }
                double om = 0.0;
                if (dot > 0.0 && d2 > 0.0) om = ndim == 3 ? dot / (d2 * sqrt(d2)) : dot / d2;
                if (pass == 0) total += om;
                else w[(int64_t)i * npix + j] = total > 0.0 ? (float)(om / total) : 0.0f;
            }
        }
        if (omega0) omega0[j] = total;
    }
    return 0;
}

/* oracle_backproject_weighted: oracle_backproject with every term multiplied by wgt[i][j] (fp32, same pitch
 * as tau):  image[f][j] = sum_i wgt_ij * [ (1-a)*b_fi[k] + a*b_fi[k+1] ].  Same arguments otherwise. */
int oracle_backproject_weighted(const float *tau, const float *wgt, int64_t tau_pitch, const float *traces,
                                int32_t nsens, int64_t npix, int32_t nt, int32_t nframes,
                                float fs, float t0, double wp, double wd, double *image)
{
    if (nsens < 0 || npix < 0 || nt < 2 || nframes < 0 || tau_pitch < npix || !wgt) return 1;
    double *b = (double *)malloc((size_t)(nsens > 0 ? nsens : 1) * (size_t)nt * sizeof(double));
    if (!b) return 2;
    const double t0fs = (double)t0 * (double)fs;
    const float ulim = (float)(nt - 1);
    for (int32_t f = 0; f < nframes; ++f) {
        for (int32_t i = 0; i < nsens; ++i)
            oracle_weight(traces + ((int64_t)f * nsens + i) * nt, nt, wp, wd, t0fs, b + (int64_t)i * nt);
        #pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < npix; ++j) {
            double acc = 0.0;
            for (int32_t i = 0; i < nsens; ++i) {
                float ts = tau[(int64_t)i * tau_pitch + j] - t0;   /* fp32 subtract */
                float u = ts * fs;                                 /* ONE fp32 multiply */
                if (!(u >= 0.0f && u < ulim)) continue;
                float kf = floorf(u);
                int32_t k = (int32_t)kf;
                float a = u - kf;                                  /* exact in fp32 */
                const double *bi = b + (int64_t)i * nt;
                acc += (double)wgt[(int64_t)i * tau_pitch + j] * ((1.0 - (double)a) * bi[k] + (double)a * bi[k + 1]);
            }
            image[(int64_t)f * npix + j] = acc;
        }
    }
    free(b);
    return 0;
}
