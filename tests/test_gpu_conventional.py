"""the conventional back projection with the delays computed inside the gather
(pat_backproject_conventional) against the oracle: oracle.tau_conventional (the analytic delays
in the fixed fp32 order) fed to oracle.backproject (Eq. 7).  Same bar as the table path."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity

pytestmark = pytest.mark.gpu


def _plan(geom, max_batch, mode=1):
    import paper_1501_03869_b200 as pat
    return pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                    geom.t0, weighting=mode, max_batch=max_batch)


def _run(plan, traces, c0, npix):
    import torch
    B = traces.shape[0]
    img = torch.full((B, npix), float("nan"), dtype=torch.float32, device="cuda")
    plan.backproject_conventional(torch.from_numpy(np.ascontiguousarray(traces)).cuda(), img, c0, B)
    torch.cuda.synchronize()
    return img.cpu().numpy()


@pytest.mark.parametrize("B,mode", [(1, 1), (2, 1), (5, 0), (16, 1), (33, 2)])
def test_conventional_2d_every_frame_class(B, mode):
    geom = W.make_geometry(0)
    c0 = 1560.0
    rng = np.random.default_rng(100 + B)
    traces = rng.standard_normal((B, geom.nsens, geom.nt)).astype(np.float32)
    tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
    ref = oracle.backproject(tau, traces, geom.fs, geom.t0, mode)
    plan = _plan(geom, B, mode)
    try:
        got = _run(plan, traces, c0, geom.npix)
    finally:
        plan.close()
    assert_parity(got, ref, "conventional B=%d mode=%d" % (B, mode))


def test_conventional_3d_and_c0_change_and_mixing_with_the_table():
    """3-D geometry; a second c0 on the same plan (work lists rebuilt); table calls in between are untouched."""
    import torch
    geom = W.make_geometry(3, True)
    rng = np.random.default_rng(7)
    traces = rng.standard_normal((3, geom.nsens, geom.nt)).astype(np.float32)
    plan = _plan(geom, 3)
    try:
        for c0 in (1560.0, 1480.0):
            tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
            ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
            assert_parity(_run(plan, traces, c0, geom.npix), ref, "3-D conventional c0=%g" % c0)
        # the table path on the same plan, fed with the oracle's analytic table: the same image again
        plan.set_travel_times(tau)
        img = torch.empty((3, geom.npix), dtype=torch.float32, device="cuda")
        plan.backproject(torch.from_numpy(traces).cuda(), img, 3)
        torch.cuda.synchronize()
        assert_parity(img.cpu().numpy(), ref, "table path with the analytic table")
        assert_parity(_run(plan, traces, 1480.0, geom.npix), ref, "conventional after a table call")
    finally:
        plan.close()


def test_conventional_windows_clipped_by_the_trace_ends():
    """A short trace: many pixels fall before sample 0 or after nt-2 for some sensors (rows that are partly or
    wholly invalid, long k-ranges) -- the index rule is the table path's."""
    geom = W.make_geometry(0)
    geom.nt = 96
    rng = np.random.default_rng(3)
    traces = rng.standard_normal((2, geom.nsens, geom.nt)).astype(np.float32)
    c0 = 1500.0
    tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
    u = (tau.astype(np.float32) - np.float32(geom.t0)) * np.float32(geom.fs)
    valid = (u >= 0) & (u < geom.nt - 1)
    assert 0.02 < valid.mean() < 0.98                                # the case really is mixed
    ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
    plan = _plan(geom, 2)
    try:
        got = _run(plan, traces, c0, geom.npix)
    finally:
        plan.close()
    assert_parity(got, ref, "clipped windows")


def test_conventional_errors():
    import torch
    import paper_1501_03869_b200 as pat
    geom = W.make_geometry(0)
    plan = _plan(geom, 1)
    tr = torch.zeros((1, geom.nsens, geom.nt), dtype=torch.float32, device="cuda")
    img = torch.zeros((1, geom.npix), dtype=torch.float32, device="cuda")
    try:
        for bad in (0.0, -1.0, float("nan"), float("inf")):
            with pytest.raises(pat.PatError) as ei:
                plan.backproject_conventional(tr, img, bad, 1)
            assert ei.value.status == pat.PAT_ERR_INVALID_ARG
        with pytest.raises(pat.PatError) as ei:
            plan.backproject_conventional(tr, img, 1500.0, 2)        # nframes > max_batch
        assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    finally:
        plan.close()
    bare = pat.Plan(geom.n, geom.h, geom.origin, None, None, geom.roi_index, geom.nt, geom.fs, geom.t0, max_batch=1,
                    nsens=geom.nsens)
    try:
        with pytest.raises(pat.PatError) as ei:
            bare.backproject_conventional(tr, img, 1500.0, 1)
        assert ei.value.status == pat.PAT_ERR_BAD_STATE
    finally:
        bare.close()


def test_conventional_host_buffers_transfer_only_the_reachable_samples():
    """Pinned host traces with the conventional BP: the strided H2D copy covers the k-ranges computed from the
    geometry for this c0 (a changed c0 moves the window); three calls, both staging buffers."""
    import torch
    geom = W.make_geometry(0)
    rng = np.random.default_rng(17)
    plan = _plan(geom, 2)
    try:
        for c0 in (1560.0, 2400.0, 1560.0):
            traces = rng.standard_normal((2, geom.nsens, geom.nt)).astype(np.float32)
            tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
            ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
            tr = torch.from_numpy(traces).pin_memory()
            img = torch.empty((2, geom.npix), dtype=torch.float32).pin_memory()
            plan.backproject_conventional(tr, img, c0, 2)
            torch.cuda.synchronize()
            assert_parity(img.numpy(), ref, "conventional, host buffers, c0=%g" % c0)
    finally:
        plan.close()


# ---- the c0 sweep ("+ a c0 sweep (autofocus-style)") ---------------------
def _sweep(plan, traces1, c0s, npix):
    import torch
    img = torch.full((len(c0s), npix), float("nan"), dtype=torch.float32, device="cuda")
    plan.backproject_conventional_sweep(torch.from_numpy(np.ascontiguousarray(traces1)).cuda(), img, c0s)
    torch.cuda.synchronize()
    return img.cpu().numpy()


@pytest.mark.parametrize("k,reduced,c0s,mode", [
    (0, False, [1480.0, 1520.0, 1560.0, 1600.0, 1640.0], 1),
    (1, False, [1560.0], 1),
    (1, False, list(np.linspace(1450.0, 1650.0, 16)), 2),
    (4, True, [1500.0, 1540.0, 1580.0], 0),
])
def test_c0_sweep_equals_one_oracle_run_per_speed(k, reduced, c0s, mode):
    """images[q] of ONE sweep call = the oracle's conventional BP with c0[q] (K oracle runs), same tolerance; speeds in
    any order, the extremes define the staged windows."""
    geom = W.make_geometry(k, reduced)
    rng = np.random.default_rng(300 + k)
    traces = rng.standard_normal((1, geom.nsens, geom.nt)).astype(np.float32)
    c0s = list(c0s)
    rng.shuffle(c0s)
    plan = _plan(geom, 1, mode)
    try:
        got = _sweep(plan, traces[0], c0s, geom.npix)
        for q, c0 in enumerate(c0s):
            tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
            ref = oracle.backproject(tau, traces, geom.fs, geom.t0, mode)
            assert_parity(got[q:q + 1], ref, "sweep k=%d c0=%g" % (k, c0))
        # a single-speed call on the same plan afterwards (row ranges and work lists are rebuilt for it)
        c0 = c0s[0]
        tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
        assert_parity(_run(plan, traces, c0, geom.npix), oracle.backproject(tau, traces, geom.fs, geom.t0, mode), "after the sweep")
    finally:
        plan.close()


def test_c0_sweep_with_speeds_that_push_delays_out_of_the_record_and_argument_errors():
    """A very low speed moves most delays past the end of the record (those terms are 0, R7); bad arguments."""
    import torch
    import paper_1501_03869_b200 as pat
    geom = W.make_geometry(0)
    rng = np.random.default_rng(31)
    traces = rng.standard_normal((1, geom.nsens, geom.nt)).astype(np.float32)
    c0s = [600.0, 1540.0, 9000.0]
    plan = _plan(geom, 1)
    try:
        got = _sweep(plan, traces[0], c0s, geom.npix)
        for q, c0 in enumerate(c0s):
            tau = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0)
            assert_parity(got[q:q + 1], oracle.backproject(tau, traces, geom.fs, geom.t0, 1), "sweep c0=%g" % c0)
        tr = torch.from_numpy(traces[0]).cuda()
        img = torch.empty((17, geom.npix), dtype=torch.float32, device="cuda")
        for bad in ([], [1500.0] * 17, [1500.0, -1.0], [float("nan")]):
            with pytest.raises(pat.PatError) as ei:
                plan.backproject_conventional_sweep(tr, img, bad)
            assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    finally:
        plan.close()


def test_fast_delays_are_the_generic_delays_and_a_detector_on_a_node_switches_them_off(monkeypatch):
    """The one-frame conventional BP computes 2-D, t0 = 0 delays with the square root written out (gather.cu,
    onfly_u_fast2d): valid only while every |r - s|^2 is a normal number, which the set-up kernel checks per plan.
    (a) default (fast) and PAT_NO_FAST_DELAYS=1 (generic) both match the oracle on configs[0] -- the image moves
    by rel-L2 ~1e-5 if a single rounding of the delay differs (gather.cu, note on packed multiplies); (b) with one
    detector moved ONTO a node |r - s| = 0 occurs (rsqrt(0) = inf: the fast path would produce NaN -> a dropped term;
    the oracle's sqrt gives 0 -> u = 0, a valid term), the plan must fall back and still match; (c) the c0 sweep too."""
    import torch
    geom = W.make_geometry(0)
    c0 = 1560.0
    rng = np.random.default_rng(41)
    traces = rng.standard_normal((1, geom.nsens, geom.nt)).astype(np.float32)
    traces[:, :, :3] += 5.0                                        # make the u = 0 term of (b) count
    c0s = np.array([1500.0, 1560.0, 1610.0], dtype=np.float32)

    def check(sensors, tag):
        g = W.make_geometry(0)
        g.sensors = sensors
        tau = oracle.tau_conventional(g.n, g.h, g.origin, sensors, g.roi_index, c0)
        ref = oracle.backproject(tau, traces, g.fs, g.t0, 1)
        plan = _plan(g, 1)
        try:
            assert_parity(_run(plan, traces, c0, g.npix), ref, tag)
            img = torch.full((len(c0s), g.npix), float("nan"), dtype=torch.float32, device="cuda")
            plan.backproject_conventional_sweep(torch.from_numpy(traces[0]).cuda(), img, c0s)
            torch.cuda.synchronize()
            for q, c in enumerate(c0s):
                tq = oracle.tau_conventional(g.n, g.h, g.origin, sensors, g.roi_index, float(c))
                assert_parity(img[q:q + 1].cpu().numpy(), oracle.backproject(tq, traces, g.fs, g.t0, 1), tag + " sweep c0=%g" % c)
        finally:
            plan.close()
        return tau

    check(geom.sensors.copy(), "fast delays")
    monkeypatch.setenv("PAT_NO_FAST_DELAYS", "1")
    check(geom.sensors.copy(), "generic delays")
    monkeypatch.delenv("PAT_NO_FAST_DELAYS")
    on_node = geom.sensors.copy()
    j = geom.npix // 2 + 5                                        # node (i, j) of the 64 x 64 grid: its fp32 coordinates
    q = int(geom.roi_index[j])
    ix, iy = q % geom.n[0], q // geom.n[0]
    on_node[3, 0] = np.float32(geom.origin[0]) + np.float32(ix) * np.float32(geom.h)
    on_node[3, 1] = np.float32(geom.origin[1]) + np.float32(iy) * np.float32(geom.h)
    tau = check(on_node, "a detector on a node")
    assert tau[3, j] == 0.0
