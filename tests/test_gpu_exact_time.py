"""Eq. 7 with the weight taken AT t_ij (PAT_W_PAPER_EXACT, PAT_W_UBP_EXACT;
PAPER.md:66 read literally) against oracle.backproject(mode = 3, 4) -- same table, same bar as the other
weightings.  The CUDA path carries two channels per frame through the pre-pass and the gather."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity, case, gpu_backproject

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


@pytest.mark.parametrize("mode", [3, 4])
def test_config0_exact_time(mode):
    geom, tau = case(0)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, mode)
    assert_parity(gpu_backproject(geom, tau, tr, mode=mode), ref, "config0 mode %d" % mode)
    # the variant really is a different image than the sample-time weighting (second-order term)
    other = oracle.backproject(tau, tr, geom.fs, geom.t0, mode - 2)
    assert np.linalg.norm(ref - other) > 1e-4 * np.linalg.norm(ref)


def test_config1_paper_scale_exact_time():
    geom, tau = case(1)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 3)
    assert_parity(gpu_backproject(geom, tau, tr, mode=3), ref, "config1 exact")
    assert_parity(gpu_backproject(geom, tau, tr, mode=3, host=True), ref, "config1 exact, host buffers")


@pytest.mark.parametrize("B", [1, 2, 3, 4, 5, 8, 9, 16, 17, 33])
def test_exact_time_every_channel_count_class(B):
    """2B channels: classes 2, 4, 8, 16 (blocked trace layout), 32 and multi-group launches; whole rows on the
    fast path plus segmented rows with out-of-record entries."""
    g = _geom(700, 9, 160)
    rng = np.random.default_rng(300 + B)
    base = rng.uniform(20.0, 120.0, size=(9, 1))
    tau = ((base + rng.uniform(0.0, 30.0, size=(9, 700))) / FS).astype(np.float32)
    tau[2, ::50] = np.float32(3.0 / FS)
    tau[4, 7::90] = np.float32(400.0 / FS)
    tr = rng.standard_normal((B, 9, 160)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, 0.0, 3)
    assert_parity(gpu_backproject(g, tau, tr, mode=3), ref, "exact B=%d" % B)


@pytest.mark.parametrize("npix,nsens,nt,B", [(1, 1, 2, 1), (257, 17, 33, 2), (1000, 33, 101, 3), (777, 50, 512, 7)])
def test_exact_time_ragged_sizes_random_tau_and_t0(npix, nsens, nt, B):
    g = _geom(npix, nsens, nt)
    rng = np.random.default_rng(5)
    t0 = float(np.float32(1.7e-6))
    tau = (t0 + rng.uniform(-2.0, nt + 1.0, size=(nsens, npix)) / FS).astype(np.float32)
    tau[0, 0] = np.nan
    tr = rng.standard_normal((B, nsens, nt)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, t0, 4)
    got = gpu_backproject(g, tau, tr, mode=4, t0=t0)
    assert np.all(np.isfinite(got))
    assert_parity(got, ref, "exact ragged")


def test_exact_time_3d_reduced_and_batch_equals_single_frames():
    geom, tau = case(4, True)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 3)
    assert_parity(gpu_backproject(geom, tau, tr, mode=3), ref, "config4 reduced exact")
    geom, tau = case(2)
    tr = W.make_traces(geom, tau, frames=range(5))
    got = gpu_backproject(geom, tau, tr, mode=3)
    assert_parity(got, oracle.backproject(tau, tr, geom.fs, geom.t0, 3), "config2 x 5 frames exact")
    one = gpu_backproject(geom, tau, tr[4:5], mode=3)
    assert_parity(got[4], one[0].astype(np.float64), "batch vs single frame")


@pytest.mark.parametrize("B", [1, 6])
def test_exact_time_conventional_bp(B):
    """The same weighting through pat_backproject_conventional (delays computed in the gather)."""
    import torch
    import paper_1501_03869_b200 as pat
    geom = W.make_geometry(0)
    c0 = 1560.0
    rng = np.random.default_rng(11 + B)
    traces = rng.standard_normal((B, geom.nsens, geom.nt)).astype(np.float32)
    tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
    ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 3)
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0, weighting=pat.PAT_W_PAPER_EXACT, max_batch=2 * B)
    try:
        img = torch.full((B, geom.npix), float("nan"), dtype=torch.float32, device="cuda")
        plan.backproject_conventional(torch.from_numpy(traces).cuda(), img, c0, B)
        torch.cuda.synchronize()
        assert_parity(img.cpu().numpy(), ref, "conventional exact B=%d" % B)
    finally:
        plan.close()


def test_exact_time_needs_two_frame_slots_per_frame():
    import torch
    import paper_1501_03869_b200 as pat
    geom, tau = case(0)
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0, weighting=pat.PAT_W_UBP_EXACT, max_batch=3)
    try:
        plan.set_travel_times(tau)
        tr = torch.zeros((2, geom.nsens, geom.nt), dtype=torch.float32, device="cuda")
        img = torch.zeros((2, geom.npix), dtype=torch.float32, device="cuda")
        with pytest.raises(pat.PatError) as ei:
            plan.backproject(tr, img, 2)                              # 4 channels > max_batch = 3
        assert ei.value.status == pat.PAT_ERR_INVALID_ARG
        plan.backproject(tr, img, 1)
        torch.cuda.synchronize()
    finally:
        plan.close()
