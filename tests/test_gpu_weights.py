"""per-(sensor, pixel) weights (pat_set_pixel_weights) and the universal BP's solid-angle
factors computed on the device (pat_compute_solid_angle_weights, ref. [5]) against
oracle.backproject(weights=...) / oracle.solid_angle_weights.  Same table, same bar as the plain sum."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity, case

pytestmark = pytest.mark.gpu
FS = 20e6


def _geom(npix, nsens, nt, nx=64, ny=64):
    g = W.make_geometry(0)
    g.n = (nx, ny)
    g.c_map = np.full((ny, nx), 1540.0, np.float32)
    rng = np.random.default_rng(npix + nsens)
    g.roi_index = np.sort(rng.choice(nx * ny, size=npix, replace=False)).astype(np.int64)
    g.sensors = np.zeros((nsens, 3), np.float32)
    g.nt = nt
    return g


def _plan(geom, B, mode=1, t0=None):
    import paper_1501_03869_b200 as pat
    return pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0 if t0 is None else t0, weighting=mode, max_batch=B)


def _bp(plan, traces, npix, c0=None):
    import torch
    B = traces.shape[0]
    img = torch.full((B, npix), float("nan"), dtype=torch.float32, device="cuda")
    tr = torch.from_numpy(np.ascontiguousarray(traces)).cuda()
    if c0 is None:
        plan.backproject(tr, img, B)
    else:
        plan.backproject_conventional(tr, img, c0, B)
    torch.cuda.synchronize()
    return img.cpu().numpy()


def _radial_normals(sensors):
    s = sensors.astype(np.float64)
    return (s / np.linalg.norm(s, axis=1, keepdims=True)).astype(np.float32)


@pytest.mark.parametrize("B", [1, 2, 3, 5, 9, 17, 33])
def test_random_weights_every_frame_count_class(B):
    """Whole rows (fast path), segmented rows, out-of-record entries; host and device weight rows, set in pieces."""
    import torch
    g = _geom(700, 9, 160)
    rng = np.random.default_rng(500 + B)
    base = rng.uniform(20.0, 120.0, size=(9, 1))
    tau = ((base + rng.uniform(0.0, 30.0, size=(9, 700))) / FS).astype(np.float32)
    tau[2, ::50] = np.float32(3.0 / FS)
    tau[4, 7::90] = np.float32(400.0 / FS)
    w = rng.uniform(-0.5, 1.5, size=(9, 700)).astype(np.float32)
    tr = rng.standard_normal((B, 9, 160)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, 0.0, 1, weights=w)
    plan = _plan(g, B)
    try:
        plan.set_travel_times(tau)
        plan.set_pixel_weights(w[:4])                                  # host rows
        plan.set_pixel_weights(torch.from_numpy(w[4:]).cuda(), 4)      # device rows
        assert_parity(_bp(plan, tr, g.npix), ref, "weighted B=%d" % B)
        # rows that were never set are 1: weights for sensor 0 only
        plan.set_pixel_weights(None)
        plan.set_pixel_weights(w[:1])
        w1 = np.ones_like(w)
        w1[0] = w[0]
        assert_parity(_bp(plan, tr, g.npix), oracle.backproject(tau, tr, FS, 0.0, 1, weights=w1), "one weighted row")
        # weights removed: the plain sum again
        plan.set_pixel_weights(None)
        assert_parity(_bp(plan, tr, g.npix), oracle.backproject(tau, tr, FS, 0.0, 1), "weights removed")
    finally:
        plan.close()


@pytest.mark.parametrize("npix,nsens,nt,B", [(1, 1, 2, 1), (257, 17, 33, 2), (1000, 33, 101, 3)])
def test_weights_ragged_sizes_random_tau(npix, nsens, nt, B):
    g = _geom(npix, nsens, nt)
    rng = np.random.default_rng(6)
    tau = (rng.uniform(-2.0, nt + 1.0, size=(nsens, npix)) / FS).astype(np.float32)
    w = rng.uniform(0.0, 2.0, size=(nsens, npix)).astype(np.float32)
    tr = rng.standard_normal((B, nsens, nt)).astype(np.float32)
    plan = _plan(g, B, mode=2)
    try:
        plan.set_travel_times(tau)
        plan.set_pixel_weights(w)
        got = _bp(plan, tr, npix)
    finally:
        plan.close()
    assert np.all(np.isfinite(got))
    assert_parity(got, oracle.backproject(tau, tr, FS, 0.0, 2, weights=w), "weighted ragged")


def test_config1_universal_bp_solid_angle_weights_from_the_device():
    """configs[1]: the device-computed solid-angle table (ring, radial normals) with the FMM delays, weighting 2 =
    the universal BP's 2p - 2t dp/dt; the oracle computes its own weights.  Also B = 4 frames on the same plan."""
    geom, tau = case(1)
    nrm = _radial_normals(geom.sensors)
    w = oracle.solid_angle_weights(geom.n, geom.h, geom.origin, geom.sensors, nrm, geom.roi_index)
    assert abs(float(w.astype(np.float64).sum(axis=0).mean()) - 1.0) < 1e-5
    tr = W.make_traces(geom, tau, frames=range(4))
    plan = _plan(geom, 4, mode=2)
    try:
        plan.set_travel_times(tau)
        plan.compute_solid_angle_weights(nrm)
        ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 2, weights=w)
        assert_parity(_bp(plan, tr[:1], geom.npix), ref[:1], "config1 UBP B=1")
        assert_parity(_bp(plan, tr, geom.npix), ref, "config1 UBP B=4")
        # the weighting matters on this geometry (ring radius 30 mm, region radius ~20 mm): not just Eq. 7 / S
        plain = oracle.backproject(tau, tr[:1], geom.fs, geom.t0, 2) / geom.nsens
        assert np.linalg.norm(ref[:1] - plain) > 0.02 * np.linalg.norm(plain)
    finally:
        plan.close()


def test_3d_solid_angle_weights_with_the_conventional_bp():
    """Hemisphere, 3-D: device-computed dOmega/Omega0 + delays computed in the gather = the universal BP of [5]
    for a constant speed of sound."""
    geom, _ = case(4, True)
    nrm = _radial_normals(geom.sensors)
    c0 = 1540.0
    tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
    w = oracle.solid_angle_weights(geom.n, geom.h, geom.origin, geom.sensors, nrm, geom.roi_index)
    rng = np.random.default_rng(8)
    tr = rng.standard_normal((2, geom.nsens, geom.nt)).astype(np.float32)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 2, weights=w)
    plan = _plan(geom, 2, mode=2)
    try:
        plan.compute_solid_angle_weights(nrm)
        assert_parity(_bp(plan, tr, geom.npix, c0=c0), ref, "3-D UBP, conventional delays")
    finally:
        plan.close()


def test_weights_errors():
    import paper_1501_03869_b200 as pat
    geom, tau = case(0)
    plan = _plan(geom, 2, mode=pat.PAT_W_PAPER_EXACT)
    try:
        with pytest.raises(pat.PatError) as ei:
            plan.set_pixel_weights(np.ones((geom.nsens, geom.npix), np.float32))
        assert ei.value.status == pat.PAT_ERR_UNSUPPORTED
    finally:
        plan.close()
    plan = _plan(geom, 1)
    try:
        with pytest.raises(pat.PatError) as ei:
            plan.set_pixel_weights(np.ones((2, geom.npix), np.float32), geom.nsens - 1, 2)
        assert ei.value.status == pat.PAT_ERR_INVALID_ARG
        bad = np.zeros((geom.nsens, 3), np.float32)
        bad[3, 1] = np.nan
        with pytest.raises(pat.PatError) as ei:
            plan.compute_solid_angle_weights(bad)
        assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    finally:
        plan.close()
