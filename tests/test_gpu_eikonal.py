"""the GPU fast-sweeping eikonal solver (csrc/eikonal.cu) against the oracle's
fast marching (oracle/pat_oracle.c, fp64) -- the same first-order upwind system, two
different orders of solving it.  Bar: the fp32 rows agree to 1 ulp (both sides round an fp64 field once;
the source-cell seeds differ in the last fp64 bit, sqrt(d2)*s vs sqrt(d2)/c)."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity

pytestmark = pytest.mark.gpu


def _f32(x):
    """The C-ABI grid carries h and the origin as fp32: give the oracle exactly the same numbers."""
    return float(np.float32(x))


def _solve_gpu(n, h, origin, c_map, sensors, roi, lo=0, cnt=None, max_rounds=0):
    import torch
    import paper_1501_03869_b200 as pat
    sensors = np.ascontiguousarray(sensors, dtype=np.float32).reshape(-1, 3)
    S = sensors.shape[0]
    cnt = S - lo if cnt is None else cnt
    grid = pat.PatGrid.make(n, h, origin)
    N = int(np.prod(n))
    npix = N if roi is None else int(roi.size)
    out = torch.full((cnt, npix), float("nan"), dtype=torch.float32, device="cuda")
    rounds = pat.pat_eikonal_travel_times_device(grid, np.ascontiguousarray(c_map, dtype=np.float32).ravel(),
                                                 sensors, S, roi, npix, lo, cnt, out, max_rounds)
    return out.cpu().numpy(), rounds


def _ulp_diff(a, b):
    a = np.asarray(a, dtype=np.float32)
    b = np.asarray(b, dtype=np.float32)
    return np.abs(a.view(np.int32).astype(np.int64) - b.view(np.int32).astype(np.int64))


def _cmap_2d(n0, n1, seed, kind):
    rng = np.random.default_rng(seed)
    c = np.full((n1, n0), 1500.0, dtype=np.float32)
    if kind == "layers":
        c[n1 // 3: n1 // 2, :] = 2900.0                     # a fast slab (bone-like), sharp jumps
        c[(2 * n1) // 3:, :] = 1450.0
    elif kind == "ring":                                    # skull-like ring around the centre
        y, x = np.mgrid[0:n1, 0:n0]
        r = np.hypot(x - n0 / 2, y - n1 / 2)
        c[(r > 0.30 * n0) & (r < 0.36 * n0)] = 3000.0
        c[r <= 0.30 * n0] = 1540.0
    elif kind == "random":
        c = (1500.0 * (1.0 + 0.3 * rng.uniform(-1, 1, size=(n1, n0)))).astype(np.float32)
    return c


@pytest.mark.parametrize("kind", ["homogeneous", "layers", "ring", "random"])
def test_eikonal_2d_matches_oracle_fmm(kind):
    n, h, origin = (96, 80), _f32(1.0e-4), (_f32(-4.8e-3), _f32(-4.0e-3))
    c = _cmap_2d(n[0], n[1], 3, kind)
    rng = np.random.default_rng(11)
    sens = np.zeros((7, 3), dtype=np.float32)
    sens[:, 0] = origin[0] + rng.uniform(0.01, n[0] - 1.01, size=7) * h
    sens[:, 1] = origin[1] + rng.uniform(0.01, n[1] - 1.01, size=7) * h
    sens[0, :2] = (origin[0], origin[1])                    # the corner node
    sens[1, :2] = (origin[0] + (n[0] - 2) * h, origin[1] + 17 * h)   # next to the far edge, (nearly) on a node
    roi = np.arange(n[0] * n[1], dtype=np.int64)
    ref = oracle.fmm_rows(n, h, origin, c, sens, roi, order=1)
    got, rounds = _solve_gpu(n, h, origin, c, sens, roi)
    assert 1 <= rounds <= 40
    assert np.isfinite(got).all()
    d = _ulp_diff(got, ref)
    assert d.max() <= 1, "max ulp difference %d (rounds %d)" % (d.max(), rounds)
    assert (d == 0).mean() > 0.9


def test_eikonal_3d_matches_oracle_fmm_with_roi_and_sensor_range():
    n, h, origin = (28, 24, 20), _f32(2.0e-4), (0.0, _f32(-1.0e-3), _f32(0.5e-3))
    rng = np.random.default_rng(5)
    c = (1500.0 * (1.0 + 0.25 * rng.uniform(-1, 1, size=(n[2], n[1], n[0])))).astype(np.float32)
    c[8:11] = 2800.0
    sens = np.zeros((6, 3), dtype=np.float32)
    for d in range(3):
        sens[:, d] = origin[d] + rng.uniform(0.01, n[d] - 1.01, size=6) * h
    roi = np.sort(rng.choice(n[0] * n[1] * n[2], size=3000, replace=False)).astype(np.int64)
    ref = oracle.fmm_rows(n, h, origin, c, sens, roi, order=1)
    got, rounds = _solve_gpu(n, h, origin, c, sens, roi, lo=2, cnt=3)
    assert got.shape == (3, 3000)
    d = _ulp_diff(got, ref[2:5])
    assert d.max() <= 1, "max ulp difference %d (rounds %d)" % (d.max(), rounds)


def test_eikonal_homogeneous_first_order_error_and_axis_exactness():
    """Closed form: along the grid axes through a source ON a node the first-order scheme is exact;
    elsewhere it over-estimates the distance (never under)."""
    n, h, origin, c0 = (65, 65), _f32(1.0e-4), (0.0, 0.0), 1500.0
    c = np.full((n[1], n[0]), c0, dtype=np.float32)
    sens = np.array([[32 * h, 32 * h, 0.0]], dtype=np.float32)
    got, _ = _solve_gpu(n, h, origin, c, sens, None)
    T = got.reshape(n[1], n[0]).astype(np.float64)
    xs = (np.arange(65) - 32) * h
    exact = np.hypot(xs[None, :], xs[:, None]) / c0
    np.testing.assert_allclose(T[32, :], np.abs(xs) / c0, rtol=2e-6, atol=1e-12)
    np.testing.assert_allclose(T[:, 32], np.abs(xs) / c0, rtol=2e-6, atol=1e-12)
    assert (T >= exact * (1 - 1e-6)).all()
    assert np.max(T - exact) < 2.5 * h / c0


def test_eikonal_errors_and_round_cap():
    import paper_1501_03869_b200 as pat
    n, h, origin = (40, 40), _f32(1.0e-4), (0.0, 0.0)
    c = _cmap_2d(40, 40, 1, "ring")
    outside = np.array([[-1.0e-3, 1.0e-3, 0.0]], dtype=np.float32)
    with pytest.raises(pat.PatError) as ei:
        _solve_gpu(n, h, origin, c, outside, None)
    assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    bad = c.copy()
    bad[3, 3] = 0.0
    inside = np.array([[1.0e-3, 1.0e-3, 0.0]], dtype=np.float32)
    with pytest.raises(pat.PatError) as ei:
        _solve_gpu(n, h, origin, bad, inside, None)
    assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    with pytest.raises(pat.PatError) as ei:               # one round cannot certify convergence
        _solve_gpu(n, h, origin, c, inside, None, max_rounds=1)
    assert ei.value.status == pat.PAT_ERR_BAD_STATE


def test_plan_compute_travel_times_gpu_end_to_end():
    """configs[0]: tau solved on the GPU, fed to the hot path on the device; the image matches the oracle's
    image made with the ORACLE's own tau (tau differences of an ulp move no sample index here)."""
    import torch
    import paper_1501_03869_b200 as pat
    geom = W.make_geometry(0)
    rng = np.random.default_rng(9)
    traces = rng.standard_normal((2, geom.nsens, geom.nt)).astype(np.float32)
    tau_ref = oracle.fmm_rows(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, 1)
    ref = oracle.backproject(tau_ref, traces, geom.fs, geom.t0, 1)
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0, max_batch=2)
    try:
        rounds = plan.compute_travel_times_gpu()
        assert rounds >= 1
        img = torch.empty((2, geom.npix), dtype=torch.float32, device="cuda")
        plan.backproject(torch.from_numpy(traces).cuda(), img, 2)
        torch.cuda.synchronize()
        got = img.cpu().numpy()
    finally:
        plan.close()
    # a tau that differs by an ulp can move a pixel across a sample boundary: linear interpolation is
    # continuous there, so the image moves by O(ulp) too
    assert_parity(got, ref, "gpu tau -> image")


def test_block_ordered_solver_and_fast_sweeping_agree(monkeypatch):
    """The default block-ordered solver and round 1's level-by-level fast sweeping (PAT_EIK_ALGO=sweep) solve the
    same discrete system: rows within 1 ulp of each other in 2-D (ragged blocks: 70 x 45 is no multiple of 16) and 3-D,
    and the work counters say which one ran."""
    import paper_1501_03869_b200 as pat
    for n, origin in [((70, 45), (0.0, 0.0)), ((21, 19, 26), (0.0, 0.0, 0.0))]:
        h = _f32(1.0e-4)
        rng = np.random.default_rng(11)
        shape = tuple(reversed(n))
        c = (1500.0 * (1.0 + 0.3 * rng.uniform(-1, 1, size=shape))).astype(np.float32)
        hi = [(v - 1) * float(h) for v in n]
        sens = np.zeros((3, 3), dtype=np.float32)
        sens[:, :len(n)] = rng.uniform(0.05, 0.95, size=(3, len(n))) * np.asarray(hi)
        monkeypatch.delenv("PAT_EIK_ALGO", raising=False)
        a, _ = _solve_gpu(n, h, origin, c, sens, None)
        assert pat.pat_eikonal_last_stats()[0] > 0
        monkeypatch.setenv("PAT_EIK_ALGO", "sweep")
        b, _ = _solve_gpu(n, h, origin, c, sens, None)
        assert pat.pat_eikonal_last_stats() == (0, 0, 0)
        monkeypatch.delenv("PAT_EIK_ALGO", raising=False)
        assert np.isfinite(a).all() and _ulp_diff(a, b).max() <= 1
