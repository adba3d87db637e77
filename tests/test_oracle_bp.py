"""Pins P6-P14 for oracle_weight / oracle_backproject (Eq. 7)."""
import numpy as np
import pytest

import oracle
import workloads as W

FS = 20e6


def _rand_case(rng, S=6, P=50, Nt=64, B=2, umax=None):
    umax = umax or (Nt - 2)
    tau = (rng.uniform(0.5, umax, size=(S, P)) / FS).astype(np.float32)
    tr = rng.standard_normal((B, S, Nt)).astype(np.float32)
    return tau, tr


def _u(tau, fs=FS):
    return (tau.astype(np.float32) * np.float32(fs)).astype(np.float32)


# ---- P14: brute force, independent pure-Python float64 loops of Eq. 7 + weighting ----------
def _brute(tau, tr, fs, mode):
    wp, wd = {0: (1, 0), 1: (1, 1), 2: (2, 2)}[mode]
    B, S, Nt = tr.shape
    P = tau.shape[1]
    img = np.zeros((B, P))
    for f in range(B):
        for j in range(P):
            acc = 0.0
            for i in range(S):
                u = np.float32(tau[i, j]) * np.float32(fs)          # fp32 product
                if not (u >= 0 and u < Nt - 1):
                    continue
                k = int(np.floor(u))
                a = float(u) - k
                vals = []
                for n in (k, k + 1):
                    p = tr[f, i].astype(np.float64)
                    if n == 0:
                        D = p[1] - p[0]
                    elif n == Nt - 1:
                        D = p[Nt - 1] - p[Nt - 2]
                    else:
                        D = (p[n + 1] - p[n - 1]) / 2
                    vals.append(wp * p[n] - wd * n * D)
                acc += (1 - a) * vals[0] + a * vals[1]
            img[f, j] = acc
    return img


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_p14_brute_force_tiny_grid(mode):
    rng = np.random.default_rng(1)
    tau, tr = _rand_case(rng, S=4, P=64, Nt=32, B=2, umax=33)   # some u beyond the record
    tau[0, :5] = (np.array([0.0, 30.0, 30.999, 31.0, 0.25]) / FS).astype(np.float32)
    got = oracle.backproject(tau, tr, FS, mode=mode)
    np.testing.assert_allclose(got, _brute(tau, tr, FS, mode), rtol=1e-12, atol=1e-12)


# ---- P7: conventional BP (analytic tau) + mode 0 = library np.interp ----------
def test_p7_delay_and_sum_equals_np_interp():
    g = W.make_geometry(0)
    xy = g.roi_coords()
    s = g.sensors.astype(np.float64)
    dist = np.hypot(xy[None, :, 0] - s[:, None, 0], xy[None, :, 1] - s[:, None, 1])
    tau = (dist / 1560.0).astype(np.float32)
    rng = np.random.default_rng(3)
    tr = rng.standard_normal((1, g.nsens, g.nt)).astype(np.float32)
    got = oracle.backproject(tau, tr, g.fs, mode=0)[0]
    u = _u(tau, g.fs).astype(np.float64)
    assert not np.any(u == g.nt - 1)
    ref = sum(np.interp(u[i], np.arange(g.nt), tr[0, i].astype(np.float64), left=0.0, right=0.0)
              for i in range(g.nsens))
    np.testing.assert_allclose(got, ref, rtol=1e-12, atol=1e-12)


# ---- P8: linearity in the traces (north_star check 3) ----------------------------------------
@pytest.mark.parametrize("mode", [0, 1])
def test_p8_linearity(mode):
    rng = np.random.default_rng(4)
    tau, x = _rand_case(rng, S=8, P=100, Nt=128, B=1)
    y = rng.standard_normal(x.shape).astype(np.float32)
    al, be = 2.0, -0.5
    # make the fp32 combination exact: x, y on a coarse dyadic grid
    x = np.round(x * 256) / 256
    y = np.round(y * 256) / 256
    z = (al * x + be * y).astype(np.float32)
    assert np.array_equal(z.astype(np.float64), al * x.astype(np.float64) + be * y.astype(np.float64))
    bx = oracle.backproject(tau, x.astype(np.float32), FS, mode=mode)
    by = oracle.backproject(tau, y.astype(np.float32), FS, mode=mode)
    bz = oracle.backproject(tau, z, FS, mode=mode)
    scale = np.max(np.abs(bz))
    assert np.max(np.abs(bz - (al * bx + be * by))) <= 1e-12 * scale


# ---- P9: closed forms -------------------------------------------------------------------------
def test_p9_constant_signal_counts_valid_sensors():
    rng = np.random.default_rng(5)
    S, P, Nt = 7, 200, 64
    tau = (rng.uniform(-10, Nt + 10, size=(S, P)) / FS).astype(np.float32)
    tr = np.ones((1, S, Nt), np.float32)
    u = _u(tau)
    count = np.sum((u >= 0) & (u < Nt - 1), axis=0)
    for mode in (0, 1):
        got = oracle.backproject(tau, tr, FS, mode=mode)[0]
        np.testing.assert_allclose(got, count, rtol=0, atol=1e-12)


def test_p9_ramp_signal():
    """p[n] = n: mode 0 image = sum_i u_ij; Eq. 7 annihilates signals linear in t."""
    rng = np.random.default_rng(6)
    S, P, Nt = 5, 120, 64
    tau, _ = _rand_case(rng, S=S, P=P, Nt=Nt)
    tr = np.tile(np.arange(Nt, dtype=np.float32), (1, S, 1))
    u = _u(tau).astype(np.float64)
    got0 = oracle.backproject(tau, tr, FS, mode=0)[0]
    np.testing.assert_allclose(got0, u.sum(axis=0), rtol=1e-13)
    got1 = oracle.backproject(tau, tr, FS, mode=1)[0]
    np.testing.assert_allclose(got1, 0.0, atol=1e-10)


def test_p9_quadratic_signal():
    """p[n] = n^2: central differences exact => b[n] = -n^2, image = -sum(k^2 + a(2k+1))."""
    rng = np.random.default_rng(7)
    S, P, Nt = 5, 120, 64
    tau, _ = _rand_case(rng, S=S, P=P, Nt=Nt, umax=Nt - 2.5)
    tr = np.tile((np.arange(Nt, dtype=np.float64) ** 2).astype(np.float32), (1, S, 1))
    u = _u(tau).astype(np.float64)
    k = np.floor(u)
    a = u - k
    expect = -np.sum(k * k + a * (2 * k + 1), axis=0)
    got = oracle.backproject(tau, tr, FS, mode=1)[0]
    np.testing.assert_allclose(got, expect, rtol=1e-13)


def test_weight_closed_forms_and_ends():
    Nt = 16
    n = np.arange(Nt, dtype=np.float64)
    p = (3 * n * n - 2 * n + 5).astype(np.float32)
    b = oracle.weight(p, mode=1)
    D = 6 * n - 2
    D[0] = p[1] - p[0]
    D[-1] = p[-1] - p[-2]
    np.testing.assert_allclose(b, p - n * D, rtol=1e-14)
    np.testing.assert_array_equal(oracle.weight(p, mode=0), p.astype(np.float64))
    np.testing.assert_array_equal(oracle.weight(p, mode=2), 2 * b)
    # t0 shifts the time axis of the weight: t_n * fs = n + t0*fs
    np.testing.assert_allclose(oracle.weight(p, mode=1, t0fs=2.5), p - (n + 2.5) * D, rtol=1e-14)


# ---- P10: one sensor, delta trace => the linear-interpolation hat kernel --------------------
def test_p10_hat_kernel():
    Nt, n0 = 64, 20
    uu = np.linspace(15, 25, 401)
    tau = (uu / FS).astype(np.float32)[None, :]
    tr = np.zeros((1, 1, Nt), np.float32)
    tr[0, 0, n0] = 1.0
    got = oracle.backproject(tau, tr, FS, mode=0)[0]
    u = _u(tau)[0].astype(np.float64)
    np.testing.assert_allclose(got, np.maximum(0, 1 - np.abs(u - n0)), atol=1e-14)


# ---- P11 / P12: mode scaling, sensor permutation, batch = single frames ---------------------
def test_p11_p12_modes_permutation_batch():
    rng = np.random.default_rng(8)
    tau, tr = _rand_case(rng, S=9, P=80, Nt=96, B=3)
    i1 = oracle.backproject(tau, tr, FS, mode=1)
    i2 = oracle.backproject(tau, tr, FS, mode=2)
    np.testing.assert_array_equal(i2, 2 * i1)
    perm = rng.permutation(9)
    ip = oracle.backproject(np.ascontiguousarray(tau[perm]), np.ascontiguousarray(tr[:, perm]), FS, mode=1)
    assert np.max(np.abs(ip - i1)) <= 1e-13 * np.max(np.abs(i1))
    for f in range(3):
        np.testing.assert_array_equal(oracle.backproject(tau, tr[f:f + 1], FS, mode=1)[0], i1[f])


# ---- P13: tau outside the record / non-finite contributes 0 ---------------------------------
def test_p13_out_of_record_and_nonfinite_tau():
    rng = np.random.default_rng(9)
    S, P, Nt = 4, 40, 32
    tau, tr = _rand_case(rng, S=S, P=P, Nt=Nt, B=1)
    base = oracle.backproject(tau[1:], tr[:, 1:], FS, mode=1)[0]
    bad = np.array([np.inf, -np.inf, np.nan, -1e-9, (Nt - 1) / FS, 1.0, -3.0, 1e30], np.float32)
    for v in bad:
        t2 = tau.copy()
        t2[0, :] = v
        got = oracle.backproject(t2, tr, FS, mode=1)[0]
        np.testing.assert_array_equal(got, base)
    # u == 0 exactly is inside the record
    t2 = tau.copy()
    t2[0, :] = 0.0
    got = oracle.backproject(t2, tr, FS, mode=0)[0]
    np.testing.assert_allclose(got - oracle.backproject(tau[1:], tr[:, 1:], FS, mode=0)[0], tr[0, 0, 0], atol=1e-13)


def test_t0_shifts_the_record():
    rng = np.random.default_rng(10)
    tau, tr = _rand_case(rng, S=3, P=30, Nt=64, B=1, umax=40)
    t0 = np.float32(8) / np.float32(FS)
    tau_shift = (tau + t0).astype(np.float32)
    a = oracle.backproject(tau_shift, tr, FS, t0=float(t0), mode=0)
    u = ((tau_shift - t0).astype(np.float32) * np.float32(FS)).astype(np.float64)
    ref = sum(np.interp(u[i], np.arange(64), tr[0, i].astype(np.float64), left=0, right=0) for i in range(3))
    np.testing.assert_allclose(a[0], ref, rtol=1e-12, atol=1e-12)


# ---- P6: a single point absorber peaks at its own pixel (north_star check 2) ---------------
@pytest.mark.parametrize("mode,pulse", [(0, "gaussian"), (1, "bipolar")])
def test_p6_point_source_peaks_at_its_pixel(mode, pulse):
    g = W.make_geometry(0)
    tau = oracle.fmm_rows(g.n, g.h, g.origin, g.c_map, g.sensors.astype(np.float64), g.roi_index)
    xy = g.roi_coords()
    for node in (32 * 64 + 32, 25 * 64 + 40, 38 * 64 + 22, 20 * 64 + 30):
        assert np.hypot(*xy[node]) < 10e-3
        tr = W.make_traces(g, tau, frames=[0], noise_sigma=0.0, pulse=pulse,
                           absorbers=[(np.array([node]), np.array([1.0]))])
        img = oracle.backproject(tau, tr, g.fs, mode=mode)[0]
        assert int(np.argmax(img)) == node


def test_pitch_and_empty_inputs():
    rng = np.random.default_rng(11)
    tau, tr = _rand_case(rng, S=3, P=20, Nt=32, B=1)
    wide = np.zeros((3, 32), np.float32)
    wide[:, :20] = tau
    np.testing.assert_array_equal(oracle.backproject(wide[:, :20], tr, FS), oracle.backproject(tau, tr, FS))
    assert oracle.backproject(tau[:, :0], tr, FS).shape == (1, 0)


# ---- P15: the conventional BP's analytic delays -------------------------------------
def test_tau_conventional_matches_the_closed_form_and_its_invariants():
    """oracle.tau_conventional against |r - s| / c0 written out in fp64 from the SAME fp32-rounded node
    coordinates (what is pinned is the formula and the index -> coordinate map, x fastest); a transposed
    axis, a missing square root, c0 instead of 1/c0 or a dropped axis all fail here."""
    rng = np.random.default_rng(2)
    for n, origin in [((13, 9), (-6.0e-4, 2.0e-4)), ((7, 5, 6), (1.0e-4, -3.0e-4, 0.0))]:
        h, c0 = np.float32(1.0e-4), np.float32(1560.0)
        N = int(np.prod(n))
        roi = np.sort(rng.choice(N, size=N // 2, replace=False)).astype(np.int64)
        sens = np.zeros((4, 3), dtype=np.float32)
        for d in range(len(n)):
            sens[:, d] = np.float32(origin[d]) + rng.uniform(-3, n[d] + 3, size=4).astype(np.float32) * h
        tau = oracle.tau_conventional(n, h, origin, sens, roi, c0)
        assert tau.shape == (4, roi.size) and tau.dtype == np.float32
        idx = np.stack(np.unravel_index(roi, n[::-1]), axis=1)[:, ::-1]          # (i0, i1[, i2]), x fastest
        x32 = (np.asarray(origin, np.float32)[None, :] + (idx.astype(np.float32) * h)).astype(np.float32)
        for i in range(4):
            e = x32.astype(np.float64) - sens[i, :len(n)].astype(np.float64)[None, :]
            want = np.sqrt((e * e).sum(axis=1)) / float(c0)
            np.testing.assert_allclose(tau[i].astype(np.float64), want, rtol=6 * 2.0 ** -24, atol=0.0)
    # a sensor sitting on a node: that node's delay is exactly 0, its axis neighbours' exactly h/c0 (to rounding)
    n, h, c0 = (9, 9), np.float32(0.5), np.float32(2.0)
    sens = np.array([[2.0, 1.5, 0.0]], dtype=np.float32)                         # node (4, 3) with origin 0
    tau = oracle.tau_conventional(n, h, (0.0, 0.0), sens, None, c0).reshape(9, 9)
    assert tau[3, 4] == 0.0
    assert tau[3, 5] == tau[3, 3] == tau[4, 4] == tau[2, 4] == np.float32(0.25)
    assert tau[0, 0] == np.float32(np.sqrt(np.float32(2.0 * 2.0 + 1.5 * 1.5))) * np.float32(0.5)


def test_conventional_bp_point_source_focuses_at_the_source():
    """End to end (Eq. 7 with analytic delays): traces that carry one pulse at |r* - s_i|/c0
    back-project to an image whose maximum sits on the node r*."""
    n, h, c0, fs, nt = (31, 31), np.float32(1.0e-4), np.float32(1500.0), 40.0e6, 256
    ang = np.linspace(0, 2 * np.pi, 24, endpoint=False)
    sens = np.zeros((24, 3), dtype=np.float32)
    sens[:, 0] = 1.5e-3 + 4.0e-3 * np.cos(ang)
    sens[:, 1] = 1.5e-3 + 4.0e-3 * np.sin(ang)
    src = (19, 11)
    rs = np.array([src[0] * float(h), src[1] * float(h)])
    tr = np.zeros((1, 24, nt), dtype=np.float32)
    for i in range(24):
        k = int(round(np.hypot(*(rs - sens[i, :2].astype(np.float64))) / float(c0) * fs))
        tr[0, i, k] = 1.0
    tau = oracle.tau_conventional(n, h, (0.0, 0.0), sens, None, c0)
    img = oracle.backproject(tau, tr, fs, 0.0, 0)                               # plain delay and sum
    j = int(np.argmax(img[0]))
    assert (j % 31, j // 31) == src


# ---- P16: Eq. 7 with the weight taken AT t_ij (modes 3, 4; oracle_backproject_exact) ----
def _brute_exact(tau, tr, fs, t0, wp, wd):
    """Independent pure-Python float64 loops: p and dp/dt each interpolated at t_ij, multiplied by t_ij*fs."""
    B, S, Nt = tr.shape
    P = tau.shape[1]
    img = np.zeros((B, P))
    for f in range(B):
        for j in range(P):
            acc = 0.0
            for i in range(S):
                u = (np.float32(tau[i, j]) - np.float32(t0)) * np.float32(fs)   # two fp32 roundings (R8)
                if not (u >= 0 and u < Nt - 1):
                    continue
                k = int(np.floor(u))
                a = float(u) - k
                p = tr[f, i].astype(np.float64)

                def D(n):
                    if n == 0:
                        return p[1] - p[0]
                    if n == Nt - 1:
                        return p[Nt - 1] - p[Nt - 2]
                    return (p[n + 1] - p[n - 1]) / 2

                t_samples = float(u) + float(np.float32(t0)) * float(np.float32(fs))
                acc += wp * ((1 - a) * p[k] + a * p[k + 1]) - wd * t_samples * ((1 - a) * D(k) + a * D(k + 1))
            img[f, j] = acc
    return img


@pytest.mark.parametrize("mode,t0", [(3, 0.0), (4, 0.0), (3, 3.25 / FS)])
def test_p16_exact_time_brute_force(mode, t0):
    rng = np.random.default_rng(16)
    tau, tr = _rand_case(rng, S=4, P=64, Nt=32, B=2, umax=33)
    tau[0, :5] = (np.array([0.0, 30.0, 30.999, 31.0, 0.25]) / FS).astype(np.float32)
    tau = (tau + np.float32(t0)).astype(np.float32)
    wp, wd = oracle.WEIGHTS[mode]
    got = oracle.backproject(tau, tr, FS, t0=t0, mode=mode)
    np.testing.assert_allclose(got, _brute_exact(tau, tr, FS, t0, wp, wd), rtol=1e-12, atol=1e-12)


def test_p16_exact_time_closed_forms():
    """p = c0 + c1*n: p(t) - t*p'(t) = c0 for every t.  p = n^2: lerp(p) = k^2 + a(2k+1), lerp(D) = 2u away from
    the ends, so the term is k^2 + a(2k+1) - 2u^2.  A dropped term, a wrong sign or t_n instead of t_ij fails."""
    rng = np.random.default_rng(17)
    S, P, Nt = 5, 40, 128
    tau = (rng.uniform(1.0, Nt - 3.0, size=(S, P)) / FS).astype(np.float32)
    n = np.arange(Nt, dtype=np.float64)
    ramp = (3.0 + 0.5 * n).astype(np.float32)
    img = oracle.backproject(tau, np.broadcast_to(ramp, (1, S, Nt)).copy(), FS, mode=3)
    np.testing.assert_allclose(img[0], 3.0 * S, rtol=0, atol=1e-9)
    quad = (n * n).astype(np.float32)                     # exact in fp32
    img = oracle.backproject(tau, np.broadcast_to(quad, (1, S, Nt)).copy(), FS, mode=3)
    u = _u(tau).astype(np.float64)
    k = np.floor(u)
    a = u - k
    np.testing.assert_allclose(img[0], (k * k + a * (2 * k + 1) - 2 * u * u).sum(axis=0), rtol=1e-12)


def test_p16_exact_time_differs_from_sample_time_by_the_second_order_term():
    """exact - sample-time = wd * a(1-a) * (D[k+1] - D[k]) per term (t0 = 0); mode 4 = 2 x mode 3."""
    rng = np.random.default_rng(18)
    tau, tr = _rand_case(rng, S=7, P=90, Nt=96, B=3)
    u = _u(tau).astype(np.float64)
    k = np.floor(u).astype(np.int64)
    a = u - k
    for mode_s, mode_e, wd in ((1, 3, 1.0), (2, 4, 2.0)):
        base = oracle.backproject(tau, tr, FS, mode=mode_s)
        corr = np.zeros_like(base)
        for f in range(tr.shape[0]):
            p = tr[f].astype(np.float64)
            D = np.empty_like(p)
            D[:, 1:-1] = (p[:, 2:] - p[:, :-2]) / 2
            D[:, 0] = p[:, 1] - p[:, 0]
            D[:, -1] = p[:, -1] - p[:, -2]
            rows = np.arange(p.shape[0])[:, None]
            corr[f] = (wd * a * (1 - a) * (D[rows, k + 1] - D[rows, k])).sum(axis=0)
        np.testing.assert_allclose(oracle.backproject(tau, tr, FS, mode=mode_e), base + corr, rtol=1e-11, atol=1e-11)
    np.testing.assert_array_equal(oracle.backproject(tau, tr, FS, mode=4), 2 * oracle.backproject(tau, tr, FS, mode=3))


def test_p16_exact_time_out_of_record_terms_vanish():
    tau = (np.array([[-1.0, 0.0, 5.5, 62.999, 63.0, np.nan, np.inf]]) / FS).astype(np.float32)
    tr = np.ones((1, 1, 64), dtype=np.float32)
    img = oracle.backproject(tau, tr, FS, mode=3)
    np.testing.assert_array_equal(img[0], [0, 1, 1, 1, 0, 0, 0])


# ---- P17: solid-angle weights of the universal BP [5] and the weighted sum (R27) ----
def _ring(S, R):
    th = 2 * np.pi * np.arange(S) / S
    s = np.stack([R * np.cos(th), R * np.sin(th), np.zeros(S)], axis=1)
    nrm = np.stack([np.cos(th), np.sin(th), np.zeros(S)], axis=1)
    return s.astype(np.float32), nrm.astype(np.float32)


def test_p17_ring_subtends_two_pi_and_weights_sum_to_one():
    """A closed curve subtends 2*pi at every interior point: sum_i (n.e/|e|^2) * (2*pi*R/S) -> 2*pi (trapezoid rule
    on a periodic integrand: spectrally accurate).  Wrong exponent, sign or normal fails.  Centre: w = 1/S."""
    n, h = (33, 33), 0.5e-3
    origin = (-16 * h, -16 * h)
    S, R = 256, 20e-3
    sens, nrm = _ring(S, R)
    w, om = oracle.solid_angle_weights(n, h, origin, sens, nrm, None, return_omega0=True)
    np.testing.assert_allclose(om * (2 * np.pi * R / S), 2 * np.pi, rtol=1e-6)
    np.testing.assert_allclose(w.astype(np.float64).sum(axis=0), 1.0, rtol=0, atol=2e-6)
    centre = 16 * 33 + 16
    np.testing.assert_allclose(w[:, centre], 1.0 / S, rtol=1e-6)
    # off centre the nearer detectors weigh more (that is the whole point of the weighting)
    j = 16 * 33 + 30                                                  # x = +7 mm
    assert w[0, j] > 1.5 / S and w[S // 2, j] < 0.8 / S


def test_p17_sphere_subtends_four_pi():
    S, R = 4000, 20e-3
    i = np.arange(S)
    z = 1 - 2 * (i + 0.5) / S                                         # Fibonacci sphere: equal-area elements
    ph = i * np.pi * (3 - np.sqrt(5))
    rho = np.sqrt(1 - z * z)
    nrm = np.stack([rho * np.cos(ph), rho * np.sin(ph), z], axis=1)
    sens = (R * nrm).astype(np.float32)
    n, h = (5, 5, 5), 2e-3
    w, om = oracle.solid_angle_weights(n, h, (-2 * h,) * 3, sens, nrm.astype(np.float32), None, return_omega0=True)
    np.testing.assert_allclose(om * (4 * np.pi * R * R / S), 4 * np.pi, rtol=2e-3)
    np.testing.assert_allclose(w.astype(np.float64).sum(axis=0), 1.0, atol=1e-5)


def test_p17_weights_brute_force_and_degenerate_cases():
    rng = np.random.default_rng(21)
    h = 2.0 ** -10                                                    # exactly representable coordinates
    n, origin = (7, 6), (-3 * h, -2 * h)
    S = 9
    sens = np.zeros((S, 3), np.float32)
    sens[:, :2] = rng.uniform(-8e-3, 8e-3, size=(S, 2))
    nrm = np.zeros((S, 3), np.float32)
    nrm[:, :2] = rng.standard_normal((S, 2))
    sens[0, :2] = (origin[0] + 2 * h, origin[1] + 3 * h)              # a detector ON node (2, 3): weight 0 there
    roi = np.sort(rng.choice(42, size=30, replace=False)).astype(np.int64)
    roi[0] = 3 * 7 + 2
    roi = np.unique(roi)
    w = oracle.solid_angle_weights(n, h, origin, sens, nrm, roi)
    ref = np.zeros((S, roi.size))
    for jj, q in enumerate(roi):
        r = np.array([np.float32(origin[0]) + np.float64(q % 7) * np.float32(h),
                      np.float32(origin[1]) + np.float64(q // 7) * np.float32(h)], dtype=np.float64)
        raw = np.zeros(S)
        for i in range(S):
            e = sens[i, :2].astype(np.float64) - r
            dot = float(nrm[i, :2].astype(np.float64) @ e)
            d2 = float(e @ e)
            raw[i] = dot / d2 if (dot > 0 and d2 > 0) else 0.0
        ref[:, jj] = raw / raw.sum() if raw.sum() > 0 else 0.0
    np.testing.assert_allclose(w, ref, rtol=2e-7, atol=1e-12)
    assert w[0, list(roi).index(3 * 7 + 2)] == 0.0
    # all detectors facing away: all-zero weights, no NaN
    w0 = oracle.solid_angle_weights(n, h, origin, np.array([[1.0, 0, 0]], np.float32), np.array([[-1.0, 0, 0]], np.float32), None)
    assert np.all(w0 == 0.0)


def test_p17_weighted_sum():
    """w = 1: the plain sum; one-hot w: that sensor alone; linear in w; brute force."""
    rng = np.random.default_rng(22)
    tau, tr = _rand_case(rng, S=5, P=40, Nt=48, B=2, umax=49)
    for mode in (0, 1, 2):
        plain = oracle.backproject(tau, tr, FS, mode=mode)
        np.testing.assert_allclose(oracle.backproject(tau, tr, FS, mode=mode, weights=np.ones_like(tau)), plain,
                                   rtol=1e-13, atol=1e-13)
    hot = np.zeros_like(tau)
    hot[3] = 1.0
    np.testing.assert_allclose(oracle.backproject(tau, tr, FS, weights=hot),
                               oracle.backproject(tau[3:4], tr[:, 3:4], FS), rtol=1e-13, atol=1e-13)
    w1 = rng.uniform(0, 1, tau.shape).astype(np.float32)
    w2 = rng.uniform(0, 1, tau.shape).astype(np.float32)
    w12 = (w1.astype(np.float64) + w2).astype(np.float32)
    ok = w12.astype(np.float64) == w1.astype(np.float64) + w2                # keep the exactly representable sums
    w1[~ok] = 0; w2[~ok] = 0; w12[~ok] = 0
    np.testing.assert_allclose(oracle.backproject(tau, tr, FS, weights=w12),
                               oracle.backproject(tau, tr, FS, weights=w1) + oracle.backproject(tau, tr, FS, weights=w2),
                               rtol=1e-11, atol=1e-11)
    # brute force: per-sensor images times the weights
    acc = np.zeros((2, tau.shape[1]))
    for i in range(tau.shape[0]):
        acc += w1[i].astype(np.float64)[None, :] * _brute(tau[i:i + 1], tr[:, i:i + 1], FS, 1)
    np.testing.assert_allclose(oracle.backproject(tau, tr, FS, weights=w1), acc, rtol=1e-11, atol=1e-11)


def test_p17_large_ring_recovers_eq7():
    """for a scanning radius much larger than the region, dOmega/Omega0 -> 1/S and the universal BP
    becomes Eq. 7 / S."""
    n, h = (9, 9), 0.25e-3
    origin = (-4 * h, -4 * h)
    S, R = 64, 1.0                                                     # 1 m ring around a 2 mm region
    sens, nrm = _ring(S, R)
    w = oracle.solid_angle_weights(n, h, origin, sens, nrm, None)
    np.testing.assert_allclose(w * S, 1.0, rtol=3e-3)
    rng = np.random.default_rng(23)
    tau = (rng.uniform(2.0, 60.0, size=(S, 81)) / FS).astype(np.float32)
    tr = rng.standard_normal((1, S, 64)).astype(np.float32)
    a = oracle.backproject(tau, tr, FS, mode=2, weights=w) * S
    b = oracle.backproject(tau, tr, FS, mode=2)
    assert np.linalg.norm(a - b) <= 3e-3 * np.linalg.norm(b)
